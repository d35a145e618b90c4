// amh_tr5.cuh - config 3 (NEXT-2): the trRosetta2-style energy on the 5-slot state (BASELINE.json:11; PAPER.md:25, 125;
// DESIGN.md R25), sm_100a.
//
//   state   n = 5L: s[5i+0] = phi_i, s[5i+1] = psi_i, s[5i+2] = omega_i (torsion of the peptide bond C_i - N_{i+1}),
//           s[5i+3], s[5i+4] = two slots that move no backbone atom and no C-beta (dE = 0: always accepted)
//   energy  V = sum over i < j, j - i >= min_sep of  e_d(|CB_i CB_j|) + e_o(dihedral CA_i CB_i CB_j CA_j)
//             + e_t[i][j](dihedral N_i CA_i CB_i CB_j) + e_t[j][i](dihedral N_j CA_j CB_j CB_i)
//             + e_p[i][j](angle CA_i CB_i CB_j) + e_p[j][i](angle CA_j CB_j CB_i)
//           e = -log(p + eps), interpolated linearly between bin centres: R8's clamp for the distance (37 bins over 2-20 A)
//           and the angle (12 bins over [0, pi]), circularly for the two dihedrals (24 bins over [-pi, pi))
//
// Everything here is fp64 - coordinates, dihedrals (atan2), tables - so the dE of a proposal is the oracle's to rounding
// and no decision guard is needed; the orientation terms do not vanish with distance, so nothing is culled either.
// One CTA per chain, one proposal at a time by the whole CTA (Alg. 1 literally): a proposal turns the atoms right of the
// flipped bond into a scratch copy, the pairs that straddle the bond (all of them, or those inside the window) are dealt
// to the threads (new state only: the old state's sum is carried from step to step as in amh_sweep.cuh), block reduction,
// Metropolis test, commit.  This row is built for parity and a first number, not yet for speed.
#pragma once
#include "amh_device.cuh"
#include "amh_sweep.cuh"

#ifndef AMH_TR5_CTAS
#define AMH_TR5_CTAS 3      // resident CTAs per SM the sweep kernel is compiled for (3: 168 registers)
#endif

namespace amh {

struct Tr5Model {
    int L, n;                        // residues, variables (5 L)
    int nb_d, nb_o, nb_t, nb_p, min_sep;
    const double *Ed, *Eo, *Et, *Ep; // [L][L][nb]: -log(p + eps) in fp64; Ed, Eo read for i < j, Et, Ep per ordered pair
    double c0, delta;                // distance bins: first centre, width
    // NeRF constants: as DevModel, with the C-N-CA placement depending on omega_i
    Xf A;
    double c2, s2, l3;               // cos/sin of ang_ca_c_n, len_c_n
    double c3, s3, l1;               // cos/sin of ang_c_n_ca, len_n_ca
    double loc[4][3];
    double h0x;
    double inv_len_n_ca, inv_len_ca_c, inv_len_c_n;
};

// T_i = A * Mplus(ang_ca_c_n, psi_i, len_c_n) * Mplus(ang_c_n_ca, omega_i, len_n_ca) * Rx(phi_{i+1})
__device__ __forceinline__ Xf tr5_transition(const Tr5Model &m, float psi_i, float omega_i, float phi_next)
{
    double sp, cp, so, co, sf, cf;
    sincos((double)psi_i, &sp, &cp);
    sincos((double)omega_i, &so, &co);
    sincos((double)phi_next, &sf, &cf);
    Xf M, W;
    M.r[0] = -m.c2;      M.r[1] = -m.s2;      M.r[2] = 0.0;
    M.r[3] = m.s2 * cp;  M.r[4] = -m.c2 * cp; M.r[5] = -sp;
    M.r[6] = m.s2 * sp;  M.r[7] = -m.c2 * sp; M.r[8] = cp;
    M.t[0] = m.l3 * M.r[0]; M.t[1] = m.l3 * M.r[3]; M.t[2] = m.l3 * M.r[6];
    W.r[0] = -m.c3;      W.r[1] = -m.s3;      W.r[2] = 0.0;
    W.r[3] = m.s3 * co;  W.r[4] = -m.c3 * co; W.r[5] = -so;
    W.r[6] = m.s3 * so;  W.r[7] = -m.c3 * so; W.r[8] = co;
    W.t[0] = m.l1 * W.r[0]; W.t[1] = m.l1 * W.r[3]; W.t[2] = m.l1 * W.r[6];
    Xf P = xf_mul(xf_mul(m.A, M), W);
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        const double a = P.r[3 * i + 1], b = P.r[3 * i + 2];
        P.r[3 * i + 1] = fma(cf, a, sf * b);
        P.r[3 * i + 2] = fma(cf, b, -sf * a);
    }
    return P;
}

// x = G(s) by one warp (the scan of nerf_build_warp on the 5-slot state); emit(res, atom, x, y, z), atom = N, CA, C, CB
template <class Emit>
__device__ __forceinline__ void tr5_build_warp(const Tr5Model &m, const float *s, int lane, Emit emit)
{
    const int L = m.L;
    const int nt = L - 1;
    const int chunk = (nt + 31) / 32;
    const int lo = lane * chunk;
    const int hi = min(nt, lo + chunk);
    Xf q = xf_identity();
    for (int i = lo; i < hi; ++i) q = xf_mul(q, tr5_transition(m, s[5 * i + 1], s[5 * i + 2], s[5 * i + 5]));
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const Xf o = xf_shfl_up(q, d);
        if (lane >= d) q = xf_mul(o, q);
    }
    Xf h = xf_shfl_up(q, 1);
    if (lane == 0) h = xf_identity();
    h.t[0] += m.h0x;
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
        h = xf_mul(h, tr5_transition(m, s[5 * i + 1], s[5 * i + 2], s[5 * i + 5]));
        put(i + 1, h);
    }
}

struct V3 { double x, y, z; };
__device__ __forceinline__ V3 v3sub(const V3 a, const V3 b) { return V3{a.x - b.x, a.y - b.y, a.z - b.z}; }
__device__ __forceinline__ V3 v3cross(const V3 a, const V3 b) { return V3{a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x}; }
__device__ __forceinline__ double v3dot(const V3 a, const V3 b) { return a.x * b.x + a.y * b.y + a.z * b.z; }

// atan2 in fp64 without a branch or a call, so that the five angles of a pair overlap in the pipeline: the octant by
// selects, a = min/max in [0, 1] split at tan(pi/16) and tan(3 pi/16) around c = 0, tan(pi/8), 1, one division
// t = (min - c max) / (max + c min), |t| <= tan(pi/16), and the Taylor series of atan to t^21 (next term < 2e-17 relative).
// Within 1 ulp of pi of the exact value (checked against a 40-digit reference on 2e6 random points and the axes).
// Zeros as libm's atan2: (+-0, +0) -> +-0, (+-0, -0) -> +-pi (a zero vector takes the first octant and the sign BIT of
// x decides the half plane) - coincident or collinear atoms score the bin the oracle's atan2 scores.
__device__ __forceinline__ double tr5_atan2(double y, double x)
{
    const double ax = fabs(x), ay = fabs(y);
    const double mx = fmax(ax, ay), mn = fmin(ax, ay);
    const bool lo = mn < 0.198912367379658 * mx || mx == 0.0, hi = mn >= 0.6681786379192989 * mx && !lo;
    const double c = lo ? 0.0 : (hi ? 1.0 : 0.41421356237309503);
    const double off = lo ? 0.0 : (hi ? 0.7853981633974483 : 0.39269908169872414);
    const double num = fma(-c, mx, mn), den = fma(c, mn, mx);
    const double t = den > 0.0 ? num / den : 0.0;
    const double s = t * t;
    double q = 1.0 / 21.0;
    q = fma(q, s, -1.0 / 19.0);
    q = fma(q, s, 1.0 / 17.0);
    q = fma(q, s, -1.0 / 15.0);
    q = fma(q, s, 1.0 / 13.0);
    q = fma(q, s, -1.0 / 11.0);
    q = fma(q, s, 1.0 / 9.0);
    q = fma(q, s, -1.0 / 7.0);
    q = fma(q, s, 1.0 / 5.0);
    q = fma(q, s, -1.0 / 3.0);
    double r = off + fma(t * s, q, t);
    r = ay > ax ? 1.5707963267948966 - r : r;
    r = signbit(x) ? 3.141592653589793 - r : r;
    return copysign(r, y);
}

#ifndef AMH_TR5_ATAN2
#define AMH_TR5_ATAN2 tr5_atan2
#endif

// IUPAC dihedral a-b-c-d: atan2(|b2| b1 . (b2 x b3), (b1 x b2) . (b2 x b3))
__device__ __forceinline__ double tr5_dihedral(const V3 a, const V3 b, const V3 c, const V3 d)
{
    const V3 b1 = v3sub(b, a), b2 = v3sub(c, b), b3 = v3sub(d, c);
    const V3 n2 = v3cross(b2, b3);
    return AMH_TR5_ATAN2(sqrt(v3dot(b2, b2)) * v3dot(b1, n2), v3dot(v3cross(b1, b2), n2));
}
// angle a-b-c at b: atan2(|u x v|, u . v)
__device__ __forceinline__ double tr5_angle(const V3 a, const V3 b, const V3 c)
{
    const V3 u = v3sub(a, b), v = v3sub(c, b);
    const V3 w = v3cross(u, v);
    return AMH_TR5_ATAN2(sqrt(v3dot(w, w)), v3dot(u, v));
}
__device__ __forceinline__ double tr5_periodic(const double *__restrict__ E, int nb, double x)
{
    const double delta = 6.283185307179586 / (double)nb;
    const double t = (x + 3.141592653589793) / delta - 0.5;
    const double fl = floor(t);
    const double f = t - fl;
    int b = (int)fl;
    b = b < 0 ? b + nb : (b >= nb ? b - nb : b);
    const int b1 = (b + 1 == nb) ? 0 : b + 1;
    const double e0 = __ldg(E + b), e1 = __ldg(E + b1);
    return e0 + f * (e1 - e0);
}
__device__ __forceinline__ double tr5_clamped(const double *__restrict__ E, int nb, double c0, double delta, double x)
{
    double t = (x - c0) / delta;
    t = fmin(fmax(t, 0.0), (double)(nb - 1));
    int b = (int)floor(t);
    b = min(b, nb - 2);
    const double f = t - (double)b;
    const double e0 = __ldg(E + b), e1 = __ldg(E + b + 1);
    return e0 + f * (e1 - e0);
}

// the six terms of the unordered pair i < j from the two residues' N, CA, CB
__device__ __forceinline__ double tr5_pair(const Tr5Model &m, int i, int j, const V3 Ni, const V3 CAi, const V3 CBi,
                                           const V3 Nj, const V3 CAj, const V3 CBj)
{
    const size_t ij = (size_t)i * m.L + j, ji = (size_t)j * m.L + i;
    const V3 dv = v3sub(CBi, CBj);
    const double d = sqrt(v3dot(dv, dv));
    const double dp = 3.141592653589793 / (double)m.nb_p;
    double e = tr5_clamped(m.Ed + ij * m.nb_d, m.nb_d, m.c0, m.delta, d);
    e += tr5_periodic(m.Eo + ij * m.nb_o, m.nb_o, tr5_dihedral(CAi, CBi, CBj, CAj));
    e += tr5_periodic(m.Et + ij * m.nb_t, m.nb_t, tr5_dihedral(Ni, CAi, CBi, CBj));
    e += tr5_periodic(m.Et + ji * m.nb_t, m.nb_t, tr5_dihedral(Nj, CAj, CBj, CBi));
    e += tr5_clamped(m.Ep + ij * m.nb_p, m.nb_p, 0.5 * dp, dp, tr5_angle(CAi, CBi, CBj));
    e += tr5_clamped(m.Ep + ji * m.nb_p, m.nb_p, 0.5 * dp, dp, tr5_angle(CAj, CBj, CBi));
    return e;
}

// E = -log(p + eps) in fp64 for one map; every entry is validated
__global__ void tr5_table_kernel(const float *__restrict__ p, double *__restrict__ E, long long count, double eps, int *__restrict__ bad)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    int local_bad = 0;
    for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < count; q += stride) {
        const float v = p[q];
        if (!(v >= 0.0f) || isinf(v)) local_bad = 1;
        E[q] = -log((double)v + eps);
    }
    if (local_bad) atomicOr(bad, 1);
}

// shared memory of one chain: double A[4][3][L] (N, CA, C, CB; x, y, z planes), double Rn[3][3][L] (N, CA, CB turned),
// double red[32], float s[5L]
__host__ __device__ inline size_t tr5_smem_bytes(int L, bool with_scratch)
{
    return sizeof(double) * ((size_t)(with_scratch ? 21 : 12) * L + 32) + sizeof(float) * 5 * (size_t)L;
}

__device__ __forceinline__ V3 tr5_atom(const double *A, int L, int at, int res)
{
    const double *p = A + (size_t)at * 3 * L + res;
    return V3{p[0], p[L], p[2 * L]};
}

__device__ __forceinline__ double tr5_block_sum(double v, double *red)
{
    v = warp_sum(v);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
    if (lane == 0) red[warp] = v;
    __syncthreads();
    double tot = 0.0;
    for (int w = 0; w < nw; ++w) tot += red[w];
    __syncthreads();
    return tot;
}

// two sums at once
__device__ __forceinline__ void tr5_block_sum2(double &a, double &b, double *red)
{
    a = warp_sum(a); b = warp_sum(b);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
    if (lane == 0) { red[warp] = a; red[16 + warp] = b; }
    __syncthreads();
    a = 0.0; b = 0.0;
    for (int w = 0; w < nw; ++w) { a += red[w]; b += red[16 + w]; }
    __syncthreads();
}

// V restricted to residues lo..hi of the atoms in shared memory (every thread returns the total)
__device__ __forceinline__ double tr5_energy_range(const Tr5Model &m, const double *A, double *red, int lo, int hi)
{
    const int L = m.L;
    double e = 0.0;
    const int nr = hi - lo + 1;
    for (int idx = threadIdx.x; idx < nr * nr; idx += blockDim.x) {
        const int i = lo + idx / nr, j = lo + idx % nr;
        if (j - i < m.min_sep) continue;
        e += tr5_pair(m, i, j, tr5_atom(A, L, 0, i), tr5_atom(A, L, 1, i), tr5_atom(A, L, 3, i),
                      tr5_atom(A, L, 0, j), tr5_atom(A, L, 1, j), tr5_atom(A, L, 3, j));
    }
    return tr5_block_sum(e, red);
}

__device__ __forceinline__ void tr5_load_state(const Tr5Model &m, const float *src, float *s, double *A)
{
    const int L = m.L;
    for (int q = threadIdx.x; q < m.n; q += blockDim.x) s[q] = src[q];
    __syncthreads();
    if (threadIdx.x < 32)
        tr5_build_warp(m, s, threadIdx.x, [&](int res, int at, double x, double y, double z) {
            double *p = A + (size_t)at * 3 * L + res;
            p[0] = x; p[L] = y; p[2 * L] = z;
        });
    __syncthreads();
}

// amh_energy / amh_energy_local on a TR5 context: one CTA per state
__global__ void __launch_bounds__(128) tr5_energy_kernel(Tr5Model m, const float *__restrict__ states, long long B, int k, int window,
                                                         float *__restrict__ out)
{
    extern __shared__ double tr5_sm[];
    double *A = tr5_sm, *red = A + 12 * (size_t)m.L;
    float *s = reinterpret_cast<float *>(red + 32);
    for (long long row = blockIdx.x; row < B; row += gridDim.x) {
        tr5_load_state(m, states + row * m.n, s, A);
        int lo = 0, hi = m.L - 1;
        if (k >= 0) { const int c = k / 5; lo = max(0, c - window); hi = min(m.L - 1, c + window); }
        const double e = tr5_energy_range(m, A, red, lo, hi);
        if (threadIdx.x == 0) out[row] = (float)e;
        __syncthreads();
    }
}

// amh_coords on a TR5 context
__global__ void __launch_bounds__(128) tr5_coords_kernel(Tr5Model m, const float *__restrict__ states, long long B,
                                                         float *__restrict__ cb_out, double *__restrict__ atoms_out)
{
    const int lane = threadIdx.x & 31;
    const long long row = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (row >= B) return;
    const float *s = states + row * m.n;
    float *cb = cb_out ? cb_out + row * m.L * 3 : nullptr;
    double *at = atoms_out ? atoms_out + row * m.L * 12 : nullptr;
    tr5_build_warp(m, s, lane, [&](int res, int a, double x, double y, double z) {
        if (at) { double *q = at + (res * 4 + a) * 3; q[0] = x; q[1] = y; q[2] = z; }
        if (cb && a == 3) { float *q = cb + res * 3; q[0] = (float)x; q[1] = (float)y; q[2] = (float)z; }
    });
}

// d, omega, theta, phi of every ordered pair of one state (input synthesis for config 3: the reference structure's values)
__global__ void __launch_bounds__(128) tr5_geometry_kernel(Tr5Model m, const float *__restrict__ states, long long B,
                                                           double *__restrict__ d_out, double *__restrict__ om_out,
                                                           double *__restrict__ th_out, double *__restrict__ ph_out)
{
    extern __shared__ double tr5_sm[];
    double *A = tr5_sm, *red = A + 12 * (size_t)m.L;
    float *s = reinterpret_cast<float *>(red + 32);
    const int L = m.L;
    for (long long row = blockIdx.x; row < B; row += gridDim.x) {
        tr5_load_state(m, states + row * m.n, s, A);
        for (int idx = threadIdx.x; idx < L * L; idx += blockDim.x) {
            const int i = idx / L, j = idx % L;
            double d = 0.0, om = 0.0, th = 0.0, ph = 0.0;
            if (i != j) {
                const V3 Ni = tr5_atom(A, L, 0, i), CAi = tr5_atom(A, L, 1, i), CBi = tr5_atom(A, L, 3, i);
                const V3 CAj = tr5_atom(A, L, 1, j), CBj = tr5_atom(A, L, 3, j);
                const V3 dv = v3sub(CBi, CBj);
                d = sqrt(v3dot(dv, dv));
                om = tr5_dihedral(CAi, CBi, CBj, CAj);
                th = tr5_dihedral(Ni, CAi, CBi, CBj);
                ph = tr5_angle(CAi, CBi, CBj);
            }
            const size_t z = (size_t)row * L * L + idx;
            if (d_out) d_out[z] = d;
            if (om_out) om_out[z] = om;
            if (th_out) th_out[z] = th;
            if (ph_out) ph_out[z] = ph;
        }
        __syncthreads();
    }
}

// Alg. 1 on the 5-slot state: one CTA per chain, one proposal at a time
__global__ void __launch_bounds__(128, AMH_TR5_CTAS) tr5_sweep_kernel(Tr5Model m, RunArgs a)
{
    extern __shared__ double tr5_sm[];
    const int L = m.L, n = m.n;
    double *A = tr5_sm, *Rn = A + 12 * (size_t)L, *red = Rn + 9 * (size_t)L;
    float *s = reinterpret_cast<float *>(red + 32);
    __shared__ double sh_cd, sh_sd, sh_lu;
    __shared__ float sh_sp;
    const int tid = threadIdx.x, nthr = blockDim.x;
    const long long cyc = (long long)a.n_global + a.n_local;

    for (long long row = blockIdx.x; row < a.B; row += gridDim.x) {
        const unsigned long long chain = (unsigned long long)(a.chain_offset + row);
        tr5_load_state(m, a.states + row * n, s, A);
        double best = INFINITY, e_end = 0.0;
        unsigned long long acc_l = 0, acc_g = 0;
        for (long long t = a.sweep_offset; t < a.sweep_offset + a.n_sweeps; ++t) {
            const long long rr = t % cyc;
            const bool gp = a.global_first ? (rr < a.n_global) : (rr >= a.n_local);
            double T;
            if (a.per_chain_T) T = (double)a.per_chain_T[row];
            else if (a.t_start == a.t_end || a.ramp_sweeps <= 1 || t <= 0) T = a.t_start;
            else if (t >= a.ramp_sweeps - 1) T = a.t_end;
            else T = a.t_start * pow(a.t_end / a.t_start, (double)t / (double)(a.ramp_sweeps - 1));
            double sigma_t = a.sigma_start;
            if (!(a.sigma_start == a.sigma_end || a.ramp_sigma <= 1 || t <= 0))
                sigma_t = (t >= a.ramp_sigma - 1) ? a.sigma_end
                                                  : a.sigma_start + (a.sigma_end - a.sigma_start) * ((double)t / (double)(a.ramp_sigma - 1));
            // dE = S_new - S_old over the straddling pairs; only S_new is summed pair by pair: S_old is carried from step to step
            // by the row and the column that enter and leave the straddling set (transition_lines of amh_sweep.cuh on the
            // equivalent (phi, psi) index k2: phi_c <-> 2c, psi_c and omega_c <-> 2c + 1, the same set for both) and becomes
            // the accepted proposal's S_new
            double S_prev = 0.0;
            int k2_prev = 0;
            for (int k = 0; k < n; ++k) {
                const int c = k / 5, slot = k - 5 * c;
                const int split = c + (slot > 0 ? 1 : 0);
                const bool inert = slot >= 3 || split <= 0 || split >= L;
                // ---- a1/a2: draws (R5-R7) ------------------------------------------------------------------
                if (tid == 0) {
                    const unsigned long long step = (unsigned long long)t * (unsigned long long)n + (unsigned long long)k;
                    uint32_t x1;
                    const uint32_t x0 = draw01(a.seed, chain, step, PURPOSE_PROPOSAL, x1);
                    float sp;
                    if (a.prop_mode == 2) {
                        const double u1 = ((double)(x0 >> 8) + 1.0) * 5.9604644775390625e-08;
                        const double u2 = (double)(x1 >> 8) * 5.9604644775390625e-08;
                        const double z = sqrt(-2.0 * log(u1)) * cos(6.283185307179586 * u2);
                        double v = (double)s[k] + sigma_t * z;
                        v -= 6.283185307179586 * floor((v + 3.141592653589793) / 6.283185307179586);
                        sp = (float)v;
                        if (sp >= 3.14159274101257324f) sp -= 2.0f * 3.14159274101257324f;
                    } else if (a.prop_mode == 1) {
                        const int mm = (int)(x0 % (uint32_t)a.grid);
                        sp = __fmul_rn(__fdiv_rn((float)(2 * mm - a.grid), (float)a.grid), 3.14159274101257324f);
                    } else {
                        const int h = (int)(x0 >> 8) - (1 << 23);
                        sp = __fmul_rn((float)h * 1.1920928955078125e-07f, 3.14159274101257324f);
                    }
                    double sd, cd;
                    sincos((double)sp - (double)s[k], &sd, &cd);
                    sh_sp = sp; sh_cd = cd; sh_sd = sd;
                }
                if (tid == 32 % nthr) {
                    const unsigned long long step = (unsigned long long)t * (unsigned long long)n + (unsigned long long)k;
                    const uint32_t x0 = draw0(a.seed, chain, step, PURPOSE_ACCEPT);
                    sh_lu = log((double)((x0 >> 8) + 1u) * 5.9604644775390625e-08);
                }
                __syncthreads();
                double dE = 0.0, s_new_sum = 0.0;
                Rot R;
                if (!inert) {
                    // ---- a3: the bond the slot turns about: phi_c N_c -> CA_c, psi_c CA_c -> C_c, omega_c C_c -> N_{c+1} -------
                    const int ra = c, rb = slot == 2 ? c + 1 : c;
                    const int aa = slot, ab = slot == 2 ? 0 : slot + 1;
                    const V3 pa = tr5_atom(A, L, aa, ra), pb = tr5_atom(A, L, ab, rb);
                    R = rot_about(pa.x, pa.y, pa.z, pb.x, pb.y, pb.z, sh_cd, sh_sd,
                                  slot == 0 ? m.inv_len_n_ca : (slot == 1 ? m.inv_len_ca_c : m.inv_len_c_n));
                    const int ilo = gp ? 0 : max(0, c - min(a.window, L - 1)), jhi = gp ? L - 1 : min(L - 1, c + min(a.window, L - 1));
                    // the N, CA, CB of the residues right of the bond, turned (atoms on the axis turn into themselves)
                    for (int q = tid; q < 3 * (jhi - split + 1); q += nthr) {
                        const int j = split + q / 3, w = q % 3, at = w == 2 ? 3 : w;
                        const V3 p = tr5_atom(A, L, at, j);
                        double x, y, z;
                        rot_apply(R, p.x, p.y, p.z, x, y, z);
                        double *o = Rn + (size_t)w * 3 * L + j;
                        o[0] = x; o[L] = y; o[2 * L] = z;
                    }
                    __syncthreads();
                    // ---- a4/a5: straddling pairs of the new state; the lines that enter / leave the set at the old one ------------
                    const int nI = split - ilo, nJ = jhi - split + 1;
                    double part = 0.0, part_T = 0.0;
                    for (int idx = tid; idx < nI * nJ; idx += nthr) {
                        const int i = ilo + idx / nJ, j = split + idx % nJ;
                        if (j - i < m.min_sep) continue;
                        part += tr5_pair(m, i, j, tr5_atom(A, L, 0, i), tr5_atom(A, L, 1, i), tr5_atom(A, L, 3, i),
                                         tr5_atom(Rn, L, 0, j), tr5_atom(Rn, L, 1, j), tr5_atom(Rn, L, 2, j));
                    }
                    const int k2 = 2 * c + (slot > 0 ? 1 : 0);
                    if (k2 != k2_prev) {                          // k2 = k2_prev + 1: one row and one column change hands
                        Line lv, en;
                        transition_lines(k2, L, gp ? L : min(a.window, L - 1), m.min_sep, lv, en);
                        for (int q = tid; q < lv.cnt + en.cnt; q += nthr) {
                            const bool isl = q < lv.cnt;
                            const int tq = isl ? q : q - lv.cnt;
                            const int i = isl ? lv.i0 + tq * lv.di : en.i0 + tq * en.di;
                            const int j = isl ? lv.j0 + tq * lv.dj : en.j0 + tq * en.dj;
                            const double e = tr5_pair(m, i, j, tr5_atom(A, L, 0, i), tr5_atom(A, L, 1, i), tr5_atom(A, L, 3, i),
                                                      tr5_atom(A, L, 0, j), tr5_atom(A, L, 1, j), tr5_atom(A, L, 3, j));
                            part_T += isl ? -e : e;
                        }
                    }
                    tr5_block_sum2(part, part_T, red);
                    S_prev += part_T;                             // S_old of this step's set for the current state
                    k2_prev = k2;
                    dE = part - S_prev;
                    s_new_sum = part;
                }
                // ---- a7: Metropolis test (Eq. 1a/2a, R14), in fp64 like everything else here ------------------
                const bool accept = sh_lu <= -dE / T;
                if (tid == 0) {
                    const long long q = (t - a.sweep_offset) * n + k;
                    if (q < a.trace_steps) {
                        const size_t z = (size_t)row * a.trace_steps + q;
                        if (a.trace_prop) a.trace_prop[z] = sh_sp;
                        if (a.trace_dE) a.trace_dE[z] = dE;
                        if (a.trace_acc) a.trace_acc[z] = accept ? 3 : 2;       // bit 1: an fp64 decision (every one is)
                    }
                }
                if (accept) {
                    if (gp) ++acc_g; else ++acc_l;
                    if (!inert) S_prev = s_new_sum;               // the accepted proposal's S_new is its set's S_old from now on
                    if (tid == 0) s[k] = sh_sp;
                    if (!inert) {
                        // every atom bonded after the turned bond moves: phi_c: C_c, CB_c and the residues after c;
                        // psi_c: the residues after c; omega_c: CA, C, CB of c + 1 and the residues after it
                        for (int q = tid; q < 4 * (L - split); q += nthr) {
                            const int res = split + q / 4, at = q % 4;
                            if (res == split && ((slot == 0 && at < 2) || (slot == 2 && at == 0))) continue;   // on the axis
                            const V3 p = tr5_atom(A, L, at, res);
                            double x, y, z;
                            rot_apply(R, p.x, p.y, p.z, x, y, z);
                            double *o = A + (size_t)at * 3 * L + res;
                            o[0] = x; o[L] = y; o[2 * L] = z;
                        }
                    }
                }
                __syncthreads();
            }
            // ---- a9: book-keeping at the sweep end ------------------------------------------------------------
            e_end = tr5_energy_range(m, A, red, 0, L - 1);
            if (e_end < best) {
                best = e_end;
                if (a.best_state)
                    for (int q = tid; q < n; q += nthr) a.best_state[row * n + q] = s[q];
            }
            if (tid == 0 && a.first_hit && (float)e_end <= a.energy_threshold) atomicMin(a.first_hit, (unsigned long long)t);
        }
        if (a.n_sweeps == 0) e_end = tr5_energy_range(m, A, red, 0, L - 1);
        for (int q = tid; q < n; q += nthr) a.states[row * n + q] = s[q];
        if (tid == 0) {
            if (a.energy) a.energy[row] = (float)e_end;
            if (a.best_energy) a.best_energy[row] = (float)best;
            if (a.n_accept_local) a.n_accept_local[row] = acc_l;
            if (a.n_accept_global) a.n_accept_global[row] = acc_g;
        }
        __syncthreads();
    }
}

}  // namespace amh
