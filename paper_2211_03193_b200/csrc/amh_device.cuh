// amh_device.cuh - device-side building blocks of the AMH hot path (sm_100a).
//
//   Philox4x32-10 keyed by (seed, chain, step, purpose)          DESIGN.md R6 (replaces the LFSRs of PAPER.md:145)
//   3x4 rigid transforms in fp64 and the NeRF prefix product      PAPER.md:39, 77; R1-R3
//   the pair term e_ij(d) of Eq. 3a                               PAPER.md:75; R8
//
// Nothing here is shared with oracle/: the geometry is the closed-form bond-frame recursion of
// DESIGN.md "Geometry" (no cross products or normalisations, unlike the oracle's sequential place()).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace amh {

// ------------------------------------------------------------------------------------------------
// Model constants, passed to every kernel by value.
// ------------------------------------------------------------------------------------------------
struct Xf {            // x -> R x + t, R row-major
    double r[9];
    double t[3];
};

struct DevModel {
    int L, nb, min_sep, n;           // residues, bins, minimum sequence separation, variables (2L)
    // Energy table, upper triangle only (R9: only p[i][j], i < j, is read).  Row r = tri(i, j) of pair i < j.
    // With E = -log(p + eps) and Elast = E[nb-1] (the value R8's clamp gives to every d >= the last bin centre), the
    // tables hold the EXCESS E'[b] = fp32(E[b] - Elast) (E'[nb-1] = 0: a far pair's term is exactly 0):
    //   Epk[r][b]   = { E'[b], E'[min(b+1, nb-1)] - E'[b] }   (the two operands of R8's lerp)
    //   Elast[r]    = fp32(Elast)
    //   Ebd[j][q][b] = E'[b] of the pair (j - min_sep - q, j), q = 0 .. band_rows - 1 (the band j - i <= band_dmax), rows
    //                 padded to row_stride floats (16-byte multiples whose bank offset differs from row to row), zero
    //                 where i < 0: a COLUMN of the local phase is one contiguous block, staged into shared memory by one
    //                 TMA bulk copy
    //   v_far       = sum over the pairs j - i >= min_sep of Elast (fp64): V = v_far + sum of the excess terms
    //   P[r][b]     = p_ij(b) as given (fp32): the fp64 path of the exact-decision guard takes -log(p + eps) itself
    const float2 *Epk;
    const float *Elast;
    const float *Ebd;
    int band_rows;                   // rows per column of Ebd: band_dmax - min_sep + 1 (0 = no band)
    const float *P;
    int row_stride;
    double c0_d, delta_d, eps_d;     // first bin centre, bin width, eps in fp64 (fp64 path)
    double far2_d;                   // squared distance from which the fp64 path is surely clamped (last centre + margin)
    float c0, inv_delta, tmax;       // first bin centre, 1/bin width, nb-1
    float t0;                        // -c0 / bin width
    float thmax;                     // nb - 1.75 (bin_frac)
    double v_far;
    float dfar;                      // >= sqrt(far2)
    float far2;                      // d^2 >= far2  =>  the clamp of R8 applies: e_ij(d) = Elast
    // bond-frame recursion H_{i+1} = H_i * A * Mplus(theta2, psi_i) * W * Rx(phi_{i+1})
    Xf A;                            // place C_i from the N->CA bond frame: Mplus(ang_n_ca_c, 0, len_ca_c)
    Xf W;                            // Mplus(ang_c_n_ca, omega, len_n_ca)
    double c2, s2, l3;               // cos/sin of ang_ca_c_n, len_c_n
    double loc[4][3];                // N, CA, C, CB in the residue's bond frame (origin CA, x along N->CA)
    double h0x;                      // H_0 = [I | (len_n_ca, 0, 0)]
    double inv_len_n_ca, inv_len_ca_c;   // 1 / length of the bonds the torsions turn about
    double cbA, cbB, cbC;            // CB = CA + cbA ex + cbB (C - CA) + cbC ex x (C - CA), ex = (CA - N) / |CA - N|   (R3)
};

// ------------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11), from the algorithm description.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              uint32_t k0, uint32_t k1, uint32_t out[4])
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        const uint32_t n0 = hi1 ^ c1 ^ k0;
        const uint32_t n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

enum { PURPOSE_PROPOSAL = 0, PURPOSE_ACCEPT = 1 };

// word 0 of Philox(key = seed; counter = (step_lo, step_hi, chain, purpose))   R6
__device__ __forceinline__ uint32_t draw0(unsigned long long seed, unsigned long long chain,
                                          unsigned long long step, uint32_t purpose)
{
    uint32_t x[4];
    philox4x32_10((uint32_t)step, (uint32_t)(step >> 32), (uint32_t)chain, purpose,
                  (uint32_t)seed, (uint32_t)(seed >> 32), x);
    return x[0];
}

// words 0 (returned) and 1 of the same block
__device__ __forceinline__ uint32_t draw01(unsigned long long seed, unsigned long long chain,
                                           unsigned long long step, uint32_t purpose, uint32_t &x1)
{
    uint32_t x[4];
    philox4x32_10((uint32_t)step, (uint32_t)(step >> 32), (uint32_t)chain, purpose,
                  (uint32_t)seed, (uint32_t)(seed >> 32), x);
    x1 = x[1];
    return x[0];
}

// ------------------------------------------------------------------------------------------------
// Rigid transforms (fp64)
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ Xf xf_identity()
{
    Xf a;
#pragma unroll
    for (int q = 0; q < 9; ++q) a.r[q] = (q % 4 == 0) ? 1.0 : 0.0;
    a.t[0] = a.t[1] = a.t[2] = 0.0;
    return a;
}

// c = a * b  (apply b first, then a)
__device__ __forceinline__ Xf xf_mul(const Xf &a, const Xf &b)
{
    Xf c;
#pragma unroll
    for (int i = 0; i < 3; ++i) {
#pragma unroll
        for (int j = 0; j < 3; ++j)
            c.r[3 * i + j] = fma(a.r[3 * i], b.r[j], fma(a.r[3 * i + 1], b.r[3 + j], a.r[3 * i + 2] * b.r[6 + j]));
        c.t[i] = fma(a.r[3 * i], b.t[0], fma(a.r[3 * i + 1], b.t[1], fma(a.r[3 * i + 2], b.t[2], a.t[i])));
    }
    return c;
}

__device__ __forceinline__ void xf_apply(const Xf &a, double x, double y, double z, double &ox, double &oy, double &oz)
{
    ox = fma(a.r[0], x, fma(a.r[1], y, fma(a.r[2], z, a.t[0])));
    oy = fma(a.r[3], x, fma(a.r[4], y, fma(a.r[5], z, a.t[1])));
    oz = fma(a.r[6], x, fma(a.r[7], y, fma(a.r[8], z, a.t[2])));
}

__device__ __forceinline__ Xf xf_shfl_up(const Xf &a, int d)
{
    Xf o;
#pragma unroll
    for (int q = 0; q < 9; ++q) o.r[q] = __shfl_up_sync(0xffffffffu, a.r[q], d);
#pragma unroll
    for (int q = 0; q < 3; ++q) o.t[q] = __shfl_up_sync(0xffffffffu, a.t[q], d);
    return o;
}

// Transition of the residue bond frame, T_i = A * Mplus(theta2, psi_i) * W * Rx(phi_{i+1}).
// Mplus(ang, tor, len) = [M | len * M[:,0]],  M = [[-ca, -sa, 0], [sa ct, -ca ct, -st], [sa st, -ca st, ct]]
// (the frame reached by one NeRF placement, written in the previous bond frame).
__device__ __forceinline__ Xf transition(const DevModel &m, float psi_i, float phi_next)
{
    double sp, cp, sf, cf;
    sincos((double)psi_i, &sp, &cp);
    sincos((double)phi_next, &sf, &cf);
    Xf M;
    M.r[0] = -m.c2;      M.r[1] = -m.s2;      M.r[2] = 0.0;
    M.r[3] = m.s2 * cp;  M.r[4] = -m.c2 * cp; M.r[5] = -sp;
    M.r[6] = m.s2 * sp;  M.r[7] = -m.c2 * sp; M.r[8] = cp;
    M.t[0] = m.l3 * M.r[0]; M.t[1] = m.l3 * M.r[3]; M.t[2] = m.l3 * M.r[6];
    Xf P = xf_mul(xf_mul(m.A, M), m.W);
    // * Rx(phi): columns 1, 2 of R mix; translation unchanged
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        const double a = P.r[3 * i + 1], b = P.r[3 * i + 2];
        P.r[3 * i + 1] = fma(cf, a, sf * b);
        P.r[3 * i + 2] = fma(cf, b, -sf * a);
    }
    return P;
}

// x = G(s) by ONE WARP: per-lane chunk products, a shuffle scan of 3x4 transforms across the lanes,
// then a second pass that emits the atoms.  s: L*2 torsions (shared or global).  emit(res, atom, x, y, z)
// is called once for every atom (atom 0..3 = N, CA, C, CB) by exactly one lane.
template <class Emit>
__device__ __forceinline__ void nerf_build_warp(const DevModel &m, const float *s, int lane, Emit emit)
{
    const int L = m.L;
    const int nt = L - 1;                                   // transitions i -> i+1
    const int chunk = (nt + 31) / 32;
    const int lo = lane * chunk;
    const int hi = min(nt, lo + chunk);
    Xf q = xf_identity();
    for (int i = lo; i < hi; ++i) q = xf_mul(q, transition(m, s[2 * i + 1], s[2 * i + 2]));
    // inclusive scan: q_lane <- q_0 * q_1 * ... * q_lane
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const Xf o = xf_shfl_up(q, d);
        if (lane >= d) q = xf_mul(o, q);
    }
    Xf h = xf_shfl_up(q, 1);                                // exclusive prefix
    if (lane == 0) h = xf_identity();
    h.t[0] += m.h0x;                                        // H_0 * prefix (H_0 is a pure translation)
    auto put = [&](int res, const Xf &f) {
#pragma unroll
        for (int a = 0; a < 4; ++a) {
            double x, y, z;
            xf_apply(f, m.loc[a][0], m.loc[a][1], m.loc[a][2], x, y, z);
            emit(res, a, x, y, z);
        }
    };
    if (lane == 0 && L > 0) put(0, h);
    for (int i = lo; i < hi; ++i) {
        h = xf_mul(h, transition(m, s[2 * i + 1], s[2 * i + 2]));
        put(i + 1, h);
    }
}

// ------------------------------------------------------------------------------------------------
// Excess pair term e'(d) = e(d) - Elast (Eq. 3a, R8): linear interpolation between bin centres, clamped at the end
// centres.  d2 = 0 is safe (IEEE sqrt), so coincident atoms score E'[0].
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ float pair_energy(const float2 *__restrict__ row, float d2, float c0, float inv_delta, float tmax, int nb)
{
    const float d = sqrtf(d2);
    float t = (d - c0) * inv_delta;
    t = fminf(fmaxf(t, 0.0f), tmax);
    int b = (int)t;
    b = min(b, nb - 2);
    const float f = t - (float)b;
    const float2 v = __ldg(row + b);              // { E[b], E[b+1] - E[b] }: one 8-byte gather per evaluation
    return fmaf(f, v.y, v.x);
}

// The same term in fp64 from the probabilities themselves (exact-decision guard, R24): E_b = -log((double)p_b + eps),
// interpolation without fma contraction, as the plain definition reads.
__device__ __forceinline__ double pair_energy_exact(const float *__restrict__ prow, double d, double c0, double delta, double eps, int nb)
{
    double t = (d - c0) / delta;
    t = fmin(fmax(t, 0.0), (double)(nb - 1));
    int b = (int)floor(t);
    b = min(b, nb - 2);
    const double f = t - (double)b;
    const double e0 = -log((double)__ldg(prow + b) + eps), e1 = -log((double)__ldg(prow + b + 1) + eps);
    return __dadd_rn(e0, __dmul_rn(f, __dadd_rn(e1, -e0)));
}

// row index of the pair i < j in the upper-triangle tables: tri(i, j) = tri_base(i) + j
__device__ __forceinline__ long long tri_base(int i, int L)
{
    return (long long)i * (2 * L - i - 1) / 2 - i - 1;
}

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
    return v;
}

}  // namespace amh
