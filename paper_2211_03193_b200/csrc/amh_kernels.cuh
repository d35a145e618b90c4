// amh_kernels.cuh - the kernels of the AMH hot path (sm_100a): table build, x = G(s), V / V_local of
// a batch, and the per-chain alternating MH sweep kernel.  See DESIGN.md "Kernels" for the layout
// and the roofline of each.
#pragma once
#include "amh_device.cuh"

namespace amh {

// ------------------------------------------------------------------------------------------------
// a0  E = -log(p + eps)   (Eq. 3a; BASELINE.json:7's 1e-8)
// ------------------------------------------------------------------------------------------------
__global__ void table_kernel(const float *__restrict__ p, float2 *__restrict__ Epk, float *__restrict__ Elast,
                             float *__restrict__ Ebd, int band_rows, int min_sep, float *__restrict__ P, int row_stride, int L, int nb, double eps,
                             int *__restrict__ bad)
{
    // bad[0] = 1 if an entry is invalid; bad[1], bad[2] = bit patterns of max |E'| and max |E'[b+1] - E'[b]| over the
    // pairs the energy reads (j - i >= min_sep): the exact-decision guard is scaled by them (amh_run, R24)
    const long long count = (long long)L * L * nb;
    const long long stride = (long long)gridDim.x * blockDim.x;
    int local_bad = 0;
    float max_e = 0.0f, max_step = 0.0f;
    for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < count; q += stride) {
        const float v = p[q];
        if (!(v >= 0.0f) || isinf(v)) local_bad = 1;                 // every entry is validated, i >= j too
        const int b = (int)(q % nb);
        const long long ij = q / nb;
        const int i = (int)(ij / L), j = (int)(ij % L);
        if (j <= i) continue;                                        // R9: only i < j is read
        // excess over the clamped value of the row (DevModel): E'[nb-1] = 0 exactly
        const double elast = -log((double)p[q - b + nb - 1] + eps);
        const float e0 = (float)(-log((double)v + eps) - elast);
        const float e1 = (b + 1 < nb) ? (float)(-log((double)p[q + 1] + eps) - elast) : e0;
        const float de = e1 - e0;
        const long long r = tri_base(i, L) + j;
        Epk[r * nb + b] = make_float2(e0, de);
        const int q_ = j - i - min_sep;
        if (q_ >= 0 && q_ < band_rows) Ebd[((long long)j * band_rows + q_) * row_stride + b] = e0;
        P[r * nb + b] = v;
        if (b == nb - 1) Elast[r] = (float)elast;
        if (j - i >= min_sep) { max_e = fmaxf(max_e, fabsf(e0)); max_step = fmaxf(max_step, fabsf(de)); }
    }
    if (local_bad) atomicOr(bad, 1);
    // non-negative floats order like their bit patterns
    const unsigned be = __reduce_max_sync(0xffffffffu, __float_as_uint(max_e));
    const unsigned bs = __reduce_max_sync(0xffffffffu, __float_as_uint(max_step));
    if ((threadIdx.x & 31) == 0) {
        if (be) atomicMax(reinterpret_cast<unsigned *>(bad) + 1, be);
        if (bs) atomicMax(reinterpret_cast<unsigned *>(bad) + 2, bs);
    }
}

// v_far = sum over the pairs j - i >= min_sep of -log(p[nb-1] + eps) in fp64 (one block, fixed order: deterministic)
__global__ void __launch_bounds__(1024) vfar_kernel(const float *__restrict__ P, int L, int nb, int min_sep, double eps, double *__restrict__ out)
{
    __shared__ double sh[1024];
    double acc = 0.0;
    for (int i = 0; i < L; ++i) {
        const long long rb = tri_base(i, L);
        for (int j = i + min_sep + (int)threadIdx.x; j < L; j += (int)blockDim.x)
            acc += -log((double)P[(rb + j) * nb + nb - 1] + eps);
    }
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int d = 512; d > 0; d >>= 1) {
        if ((int)threadIdx.x < d) sh[threadIdx.x] += sh[threadIdx.x + d];
        __syncthreads();
    }
    if (threadIdx.x == 0) *out = sh[0];
}

__global__ void philox_test_kernel(const uint32_t *ctr, const uint32_t *key, uint32_t *out, long long count)
{
    const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= count) return;
    uint32_t x[4];
    philox4x32_10(ctr[4 * q], ctr[4 * q + 1], ctr[4 * q + 2], ctr[4 * q + 3], key[2 * q], key[2 * q + 1], x);
    for (int w = 0; w < 4; ++w) out[4 * q + w] = x[w];
}

// ------------------------------------------------------------------------------------------------
// a3  x = G(s) for a batch: one warp per state
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) coords_kernel(DevModel m, const float *__restrict__ states, long long B,
                                                     float *__restrict__ cb_out, double *__restrict__ atoms_out)
{
    const int lane = threadIdx.x & 31;
    const long long row = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (row >= B) return;
    const float *s = states + row * m.n;
    float *cb = cb_out ? cb_out + row * m.L * 3 : nullptr;
    double *at = atoms_out ? atoms_out + row * m.L * 12 : nullptr;
    nerf_build_warp(m, s, lane, [&](int res, int a, double x, double y, double z) {
        if (at) { double *q = at + (res * 4 + a) * 3; q[0] = x; q[1] = y; q[2] = z; }
        if (cb && a == 3) { float *q = cb + res * 3; q[0] = (float)x; q[1] = (float)y; q[2] = (float)z; }
    });
}

// ------------------------------------------------------------------------------------------------
// a5/a9  V (Eq. 3a) or V_local (Eq. 3b) of a batch: one CTA per state.
// shared: float cb[3][L], double red[32]
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ double energy_range_cta(const DevModel &m, const float *cbx, const float *cby,
                                                   const float *cbz, int lo, int hi, bool whole, int warp, int nwarps, int lane)
{
    double e = 0.0;
    for (int i = lo + warp; i <= hi; i += nwarps) {
        const float xi = cbx[i], yi = cby[i], zi = cbz[i];
        const long long rb = tri_base(i, m.L);
        for (int j = i + m.min_sep + lane; j <= hi; j += 32) {
            const float dx = xi - cbx[j], dy = yi - cby[j], dz = zi - cbz[j];
            const float d2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
            // a window's pairs take their clamped value from the compact array (coalesced in j; the whole chain's are
            // v_far), near pairs add their excess
            if (!whole) e += (double)__ldg(m.Elast + rb + j);
            if (d2 < m.far2) e += (double)pair_energy(m.Epk + (rb + j) * m.nb, d2, m.c0, m.inv_delta, m.tmax, m.nb);
        }
    }
    return e;
}

__global__ void __launch_bounds__(128) energy_kernel(DevModel m, const float *__restrict__ states, long long B,
                                                     int k, int window, float *__restrict__ out)
{
    extern __shared__ double smem_d[];
    double *red = smem_d;                                  // [32]
    float *cbx = reinterpret_cast<float *>(smem_d + 32);
    float *cby = cbx + m.L, *cbz = cby + m.L;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    for (long long row = blockIdx.x; row < B; row += gridDim.x) {
        const float *s = states + row * m.n;
        if (warp == 0)
            nerf_build_warp(m, s, lane, [&](int res, int a, double x, double y, double z) {
                if (a == 3) { cbx[res] = (float)x; cby[res] = (float)y; cbz[res] = (float)z; }
            });
        __syncthreads();
        int lo = 0, hi = m.L - 1;
        if (k >= 0) { const int c = k >> 1; lo = max(0, c - window); hi = min(m.L - 1, c + window); }
        double e = warp_sum(energy_range_cta(m, cbx, cby, cbz, lo, hi, k < 0, warp, nwarps, lane));
        if (lane == 0) red[warp] = e;
        __syncthreads();
        if (threadIdx.x == 0) {
            double tot = 0.0;
            for (int w = 0; w < nwarps; ++w) tot += red[w];
            out[row] = (float)(k < 0 ? m.v_far + tot : tot);
        }
        __syncthreads();
    }
}


// ------------------------------------------------------------------------------------------------
// NEXT-3  replica exchange (R23): one thread per tested pair (r, r+1) of a group of `replicas`
// consecutive chains, r = cycle (mod 2).  accept iff log u <= (1/T_a - 1/T_b)(V_a - V_b), evaluated in fp64 on
// the fp32 energies and temperatures; an accepted pair swaps its temperatures.  Pairs are disjoint: no races.
// ------------------------------------------------------------------------------------------------
__global__ void exchange_kernel(const float *__restrict__ V, float *__restrict__ T, long long B, int replicas,
                                long long cycle, unsigned long long seed, long long chain_offset,
                                unsigned long long *__restrict__ n_tried, unsigned long long *__restrict__ n_accepted)
{
    const int per_group = (replicas - 1 - (int)(cycle & 1) + 1) / 2;      // pairs tested in one group this cycle
    const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (per_group <= 0 || q >= (B / replicas) * per_group) return;
    const long long g = q / per_group;
    const int r = (int)(cycle & 1) + 2 * (int)(q - g * per_group);
    const long long a = g * replicas + r, b = a + 1;
    const uint32_t x0 = draw0(seed, (unsigned long long)(chain_offset + a), (unsigned long long)cycle, 3u /* SWAP */);
    const double lu = log((double)((x0 >> 8) + 1u) * 5.9604644775390625e-08);
    const float ta = T[a], tb = T[b];
    const double d = (1.0 / (double)ta - 1.0 / (double)tb) * ((double)V[a] - (double)V[b]);
    const bool ok = lu <= d;
    if (ok) { T[a] = tb; T[b] = ta; }
    if (n_tried) atomicAdd(n_tried, 1ull);
    if (n_accepted && ok) atomicAdd(n_accepted, 1ull);
}

// ------------------------------------------------------------------------------------------------
// Measurement hooks: the two memory ceilings of the pair loops, measured on the device the
// library runs on.  Neither is on the hot path.
//   l2_read_kernel    read-only sweep of a buffer with 16-byte loads that bypass L1 (ld.global.cg): every SM reads the
//                     WHOLE buffer, so a buffer that fits in L2 is served by L2 after the first touch
//   gather_kernel     8-byte gathers at pseudo-random entries of a table (the access pattern of a near pair's lerp
//                     operands): bounded by one L1 wavefront per lane and clock, not by L2 bandwidth
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(512) l2_read_kernel(const uint4 *__restrict__ p, size_t n16, int reps, unsigned *__restrict__ out)
{
    unsigned acc = 0;
    // CTA b starts at its own offset so that the SMs do not walk the buffer in lockstep
    const size_t start = ((size_t)blockIdx.x * 7919u * blockDim.x) % n16;
    for (int r = 0; r < reps; ++r) {
        for (size_t q0 = 0; q0 < n16; q0 += (size_t)blockDim.x * 4) {
            uint4 v[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                size_t q = start + q0 + (size_t)u * blockDim.x + threadIdx.x;
                if (q >= n16) q -= n16;
                if (q >= n16) q %= n16;
                v[u] = __ldcg(p + q);
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) acc += v[u].x ^ v[u].y ^ v[u].z ^ v[u].w;
        }
    }
    if (acc == 0x9e3779b9u) out[0] = acc;                  // keeps the loads alive
}

__global__ void __launch_bounds__(256) gather_kernel(const float2 *__restrict__ p, unsigned mask, int iters, float *__restrict__ out)
{
    float acc = 0.0f;
    unsigned idx = (blockIdx.x * blockDim.x + threadIdx.x) * 2654435761u + 12345u;
    for (int it = 0; it < iters; ++it) {
        float2 v[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) { idx = idx * 1664525u + 1013904223u; v[q] = __ldg(p + ((idx >> 4) & mask)); }
#pragma unroll
        for (int q = 0; q < 8; ++q) acc += v[q].x + v[q].y;
    }
    if (acc == 1234.5f) out[0] = acc;
}

// the running minimum of the sweep-end energies over the cycles of amh_run_pt
__global__ void min_into_kernel(float *__restrict__ dst, const float *__restrict__ src, long long count, int first)
{
    const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (q < count) dst[q] = first ? src[q] : fminf(dst[q], src[q]);
}

}  // namespace amh
