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
                             int L, int nb, double eps, int *__restrict__ bad)
{
    const long long count = (long long)L * L * nb;
    const long long stride = (long long)gridDim.x * blockDim.x;
    int local_bad = 0;
    for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < count; q += stride) {
        const float v = p[q];
        if (!(v >= 0.0f) || isinf(v)) local_bad = 1;                 // every entry is validated, i >= j too
        const int b = (int)(q % nb);
        const long long ij = q / nb;
        const int i = (int)(ij / L), j = (int)(ij % L);
        if (j <= i) continue;                                        // R9: only i < j is read
        const float e0 = (float)(-log((double)v + eps));
        const float e1 = (b + 1 < nb) ? (float)(-log((double)p[q + 1] + eps)) : e0;
        const float de = e1 - e0;
        const long long r = tri_base(i, L) + j;
        Epk[r * nb + b] = make_float2(e0, de);
        if (b == nb - 2) Elast[r] = fmaf(1.0f, de, e0);              // the value pair_energy() returns at t = tmax
    }
    if (local_bad) atomicOr(bad, 1);
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
                                                   const float *cbz, int lo, int hi, int warp, int nwarps, int lane)
{
    double e = 0.0;
    for (int i = lo + warp; i <= hi; i += nwarps) {
        const float xi = cbx[i], yi = cby[i], zi = cbz[i];
        const long long rb = tri_base(i, m.L);
        for (int j = i + m.min_sep + lane; j <= hi; j += 32) {
            const float dx = xi - cbx[j], dy = yi - cby[j], dz = zi - cbz[j];
            const float d2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
            // far pairs take the clamped value from the compact array (coalesced in j), near pairs gather their row
            e += (double)((d2 >= m.far2) ? __ldg(m.Elast + rb + j)
                                         : pair_energy(m.Epk + (rb + j) * m.nb, d2, m.c0, m.inv_delta, m.tmax, m.nb));
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
        double e = warp_sum(energy_range_cta(m, cbx, cby, cbz, lo, hi, warp, nwarps, lane));
        if (lane == 0) red[warp] = e;
        __syncthreads();
        if (threadIdx.x == 0) {
            double tot = 0.0;
            for (int w = 0; w < nwarps; ++w) tot += red[w];
            out[row] = (float)tot;
        }
        __syncthreads();
    }
}


// ------------------------------------------------------------------------------------------------
// a1-a9  Alternating MH: one CTA per chain, W warps per CTA.
//
// Global sweeps: the whole CTA evaluates one proposal at a time (O(L^2/6) straddling pairs).
// Local sweeps: a proposal has only ~65-150 pairs, one warp's worth, and Alg. 1 orders the proposals
// of a chain strictly.  The draws are counter-based (R6), so the proposals of
// steps k, k+1, ... are known in advance: warp r evaluates step k+r AGAINST THE CURRENT STATE, and the
// results are consumed in order up to and including the first accepted step; later results were
// computed against a state that no longer exists and are thrown away (their steps are evaluated again
// in the next pass).  The trajectory is exactly the sequential one - only rejected steps are skipped
// over in parallel.
//
// shared (per chain):  double X[4L], Y[4L], Z[4L]   N, CA, C, CB of every residue, flat index 4*res + atom
//                      double red[16], b_cd[32], b_sd[32], b_lu[32], rot[16][12], sp_dE[16]
//                      float  cb[3][L]   fp32 copy of the C-betas (what the pair loop reads)
//                      float  nw[3][L]   candidate C-betas of a global proposal
//                      float  s[n], b_sp[32], lnw[W][3][wcap]  candidate C-betas of warp r's local proposal
//                      int    sp_acc[16]
// ------------------------------------------------------------------------------------------------
struct RunArgs {
    float *states;
    long long B, n_sweeps, sweep_offset, chain_offset;
    int n_global, n_local, window, global_first;
    double t_start, t_end;
    long long ramp_sweeps;
    const float *per_chain_T;
    int prop_mode, grid;
    int spec_local;                      // local proposals evaluated per pass (<= warps per chain)
    unsigned long long seed;
    float *energy, *best_energy, *best_state;
    unsigned long long *n_accept_local, *n_accept_global;
    unsigned long long *first_hit;       // min over chains of the absolute sweep index; ~0ull = none
    float energy_threshold;
    int trace_steps;
    float *trace_prop;
    double *trace_dE;
    unsigned char *trace_acc;
};

constexpr int kDrawBatch = 32;           // steps whose draws are generated together, one lane per step
constexpr int kMaxWarps = 16;

__host__ __device__ inline int sweep_wcap(int L, int window) { return (window + 1 < L) ? window + 1 : L; }

__host__ __device__ inline size_t sweep_smem_bytes(int L, int window, int nwarps)
{
    const size_t doubles = 12 * (size_t)L + kMaxWarps + 3 * kDrawBatch + 12 * kMaxWarps + kMaxWarps;
    const size_t floats = 6 * (size_t)L + 2 * (size_t)L + kDrawBatch + (size_t)nwarps * 3 * sweep_wcap(L, window) + kMaxWarps;
    return sizeof(double) * doubles + sizeof(float) * floats;
}

struct Rot { double r[9], t[3]; };

__device__ __forceinline__ void rot_apply(const Rot &R, double x, double y, double z, double &ox, double &oy, double &oz)
{
    ox = fma(R.r[0], x, fma(R.r[1], y, fma(R.r[2], z, R.t[0])));
    oy = fma(R.r[3], x, fma(R.r[4], y, fma(R.r[5], z, R.t[1])));
    oz = fma(R.r[6], x, fma(R.r[7], y, fma(R.r[8], z, R.t[2])));
}

// rotation by (cd, sd) = (cos, sin) of the torsion change about the axis a -> b (right-handed about b - a,
// which raises the IUPAC dihedral of everything bonded after b).  inv0 = 1 / ideal bond length:
// |b - a| equals it to rounding, so one Newton step from inv0 gives 1/|b - a| to full fp64 precision.
__device__ __forceinline__ Rot rot_about(double ax, double ay, double az, double bx, double by, double bz,
                                         double cd, double sd, double inv0)
{
    double ux = bx - ax, uy = by - ay, uz = bz - az;
    const double r2 = fma(ux, ux, fma(uy, uy, uz * uz));
    const double inv = inv0 * fma(-0.5 * r2, inv0 * inv0, 1.5);
    ux *= inv; uy *= inv; uz *= inv;
    const double v = 1.0 - cd;
    Rot R;
    R.r[0] = fma(v * ux, ux, cd);       R.r[1] = fma(v * ux, uy, -sd * uz); R.r[2] = fma(v * ux, uz, sd * uy);
    R.r[3] = fma(v * uy, ux, sd * uz);  R.r[4] = fma(v * uy, uy, cd);       R.r[5] = fma(v * uy, uz, -sd * ux);
    R.r[6] = fma(v * uz, ux, -sd * uy); R.r[7] = fma(v * uz, uy, sd * ux);  R.r[8] = fma(v * uz, uz, cd);
    R.t[0] = ax - fma(R.r[0], ax, fma(R.r[1], ay, R.r[2] * az));
    R.t[1] = ay - fma(R.r[3], ax, fma(R.r[4], ay, R.r[5] * az));
    R.t[2] = az - fma(R.r[6], ax, fma(R.r[7], ay, R.r[8] * az));
    return R;
}

// sum over the pairs (i, j), ilo <= i < split <= j <= jhi, j - i >= min_sep, of e(new) - e(old); the candidate
// C-beta of residue j is (nx, ny, nz)[j - joff].  Work is dealt to `nthr` threads, this one being `tid`.
__device__ __forceinline__ double cross_pairs_dE(const DevModel &m, const float *cbx, const float *cby, const float *cbz,
                                                 const float *nx, const float *ny, const float *nz, int joff,
                                                 int ilo, int split, int jhi, int tid, int nthr)
{
    const int nI = split - ilo, nJ = jhi - split + 1;
    double acc = 0.0;
    if (nI <= 0 || nJ <= 0) return acc;
    const int total = nI * nJ;
    const int stepI = nthr / nJ, stepJ = nthr - stepI * nJ;
    int ii = tid / nJ, jj = tid - ii * nJ;
    for (int q = tid; q < total; q += nthr) {
        const int i = ilo + ii, j = split + jj;
        if (j - i >= m.min_sep) {
            const float xi = cbx[i], yi = cby[i], zi = cbz[i];
            float dx = xi - nx[j - joff], dy = yi - ny[j - joff], dz = zi - nz[j - joff];
            const float d2n = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
            dx = xi - cbx[j]; dy = yi - cby[j]; dz = zi - cbz[j];
            const float d2o = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
            // a pair beyond the last bin centre before and after scores the same clamped value twice:
            // its term is exactly 0 and its row is never touched
            if (d2n < m.far2 || d2o < m.far2) {
                const float2 *rowp = m.Epk + (tri_base(i, m.L) + j) * m.nb;
                const float en = pair_energy(rowp, d2n, m.c0, m.inv_delta, m.tmax, m.nb);
                const float eo = pair_energy(rowp, d2o, m.c0, m.inv_delta, m.tmax, m.nb);
                acc += (double)(en - eo);
            }
        }
        ii += stepI; jj += stepJ;
        if (jj >= nJ) { jj -= nJ; ++ii; }
    }
    return acc;
}

__global__ void __launch_bounds__(512) sweep_kernel(DevModel m, RunArgs a)
{
    extern __shared__ double smem_d[];
    const int L = m.L, n = m.n;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nthreads = blockDim.x, nwarps = nthreads >> 5;
    const int wcap = sweep_wcap(L, a.window);

    double *X = smem_d, *Y = X + 4 * L, *Z = Y + 4 * L;
    double *red = Z + 4 * L, *b_cd = red + kMaxWarps, *b_sd = b_cd + kDrawBatch, *b_lu = b_sd + kDrawBatch;
    double *rot_s = b_lu + kDrawBatch, *sp_dE = rot_s + 12 * kMaxWarps;
    float *cbx = reinterpret_cast<float *>(sp_dE + kMaxWarps), *cby = cbx + L, *cbz = cby + L;
    float *nwx = cbz + L, *nwy = nwx + L, *nwz = nwy + L;
    float *s = nwz + L;
    float *b_sp = s + n;
    float *lnw = b_sp + kDrawBatch;
    int *sp_acc = reinterpret_cast<int *>(lnw + (size_t)nwarps * 3 * wcap);

    const long long row = blockIdx.x;
    const unsigned long long chain = (unsigned long long)(a.chain_offset + row);

    for (int q = tid; q < n; q += nthreads) s[q] = a.states[row * n + q];
    __syncthreads();
    if (warp == 0)
        nerf_build_warp(m, s, lane, [&](int res, int at, double x, double y, double z) {
            const int f = 4 * res + at;
            X[f] = x; Y[f] = y; Z[f] = z;
            if (at == 3) { cbx[res] = (float)x; cby[res] = (float)y; cbz[res] = (float)z; }
        });
    __syncthreads();

    double best = INFINITY, e_end = 0.0;
    unsigned long long acc_l = 0, acc_g = 0;
    const long long cyc = (long long)a.n_global + a.n_local;
    const int nspec = max(1, min(nwarps, a.spec_local > 0 ? a.spec_local : nwarps));
    const int draw_warp_u = nwarps > 1 ? 1 : 0;              // the warp that draws the uniforms of the accept test

    auto full_energy = [&]() -> double {     // all threads; returns the same value in every thread
        double e = warp_sum(energy_range_cta(m, cbx, cby, cbz, 0, L - 1, warp, nwarps, lane));
        if (lane == 0) red[warp] = e;
        __syncthreads();
        double tot = 0.0;
        for (int w = 0; w < nwarps; ++w) tot += red[w];
        __syncthreads();
        return tot;
    };
    // the bond the torsion k turns about: phi_c N->CA, psi_c CA->C
    auto step_rot = [&](int k, int bi) -> Rot {
        const int fa = 4 * (k >> 1) + (k & 1), fb = fa + 1;
        return rot_about(X[fa], Y[fa], Z[fa], X[fb], Y[fb], Z[fb], b_cd[bi], b_sd[bi], (k & 1) ? m.inv_len_ca_c : m.inv_len_n_ca);
    };

    for (long long t = a.sweep_offset; t < a.sweep_offset + a.n_sweeps; ++t) {
        const long long r = t % cyc;
        const bool is_global = a.global_first ? (r < a.n_global) : (r >= a.n_local);
        double T;
        if (a.per_chain_T) T = (double)a.per_chain_T[row];
        else if (a.t_start == a.t_end || a.ramp_sweeps <= 1 || t <= 0) T = a.t_start;
        else if (t >= a.ramp_sweeps - 1) T = a.t_end;
        else T = a.t_start * pow(a.t_end / a.t_start, (double)t / (double)(a.ramp_sweeps - 1));
        const double invT = 1.0 / T;

        int k = 0, batch_start = 0, batch_end = 0;
        while (k < n) {
            // ---- a1/a2: draws of the next 32 steps, one lane per step (R5-R7) -----------------------------
            if (k >= batch_end) {
                batch_start = k; batch_end = min(n, k + kDrawBatch);
                const int kk = k + lane;
                if (kk < n && (warp == 0 || warp == draw_warp_u)) {
                    const unsigned long long step = (unsigned long long)t * (unsigned long long)n + (unsigned long long)kk;
                    if (warp == 0) {
                        const uint32_t x0 = draw0(a.seed, chain, step, PURPOSE_PROPOSAL);
                        float sp;
                        if (a.prop_mode == 1) {
                            const int mm = (int)(x0 % (uint32_t)a.grid);
                            sp = __fmul_rn(__fdiv_rn((float)(2 * mm - a.grid), (float)a.grid), 3.14159274101257324f);
                        } else {
                            const int h = (int)(x0 >> 8) - (1 << 23);
                            sp = __fmul_rn((float)h * 1.1920928955078125e-07f, 3.14159274101257324f);
                        }
                        double sd, cd;
                        sincos((double)sp - (double)s[kk], &sd, &cd);
                        b_sp[lane] = sp; b_cd[lane] = cd; b_sd[lane] = sd;
                    }
                    if (warp == draw_warp_u) {
                        const uint32_t x0 = draw0(a.seed, chain, step, PURPOSE_ACCEPT);
                        b_lu[lane] = log((double)((x0 >> 8) + 1u) * 5.9604644775390625e-08);
                    }
                }
                __syncthreads();
            }
            if (is_global) {
                // ======== one proposal, evaluated by the whole CTA ========================================
                const int bi = k - batch_start;
                const int c = k >> 1, split = c + (k & 1);
                const bool inert = (k == 0) || (k == n - 1);
                double dE = 0.0;
                Rot R;
                if (!inert) {
                    // ---- a3: rotation of the right-hand side about the flipped bond ------------------------
                    R = step_rot(k, bi);
                    for (int j = split + tid; j < L; j += nthreads) {
                        double x, y, z;
                        rot_apply(R, X[4 * j + 3], Y[4 * j + 3], Z[4 * j + 3], x, y, z);
                        nwx[j] = (float)x; nwy[j] = (float)y; nwz[j] = (float)z;
                    }
                    __syncthreads();
                    // ---- a5/a6: cross pairs, then the reduction -------------------------------------------
                    double acc = warp_sum(cross_pairs_dE(m, cbx, cby, cbz, nwx, nwy, nwz, 0, 0, split, L - 1, tid, nthreads));
                    if (lane == 0) red[warp] = acc;
                    __syncthreads();
                    for (int w = 0; w < nwarps; ++w) dE += red[w];
                }
                // ---- a7: Metropolis test, accept iff log u <= -dE / T   (Eq. 1a, R14) ---------------------
                const bool accept = b_lu[bi] <= -dE * invT;
                if (tid == 0) {
                    const long long q = (t - a.sweep_offset) * n + k;
                    if (q < a.trace_steps) {
                        const size_t z = (size_t)row * a.trace_steps + q;
                        if (a.trace_prop) a.trace_prop[z] = b_sp[bi];
                        if (a.trace_dE) a.trace_dE[z] = dE;
                        if (a.trace_acc) a.trace_acc[z] = accept ? 1 : 0;
                    }
                }
                if (accept) {
                    ++acc_g;
                    if (tid == 0) s[k] = b_sp[bi];
                    if (!inert) {
                        const int m0 = 4 * c + 2 + 2 * (k & 1);           // first flat atom that moves
                        for (int f = m0 + tid; f < 4 * L; f += nthreads) {
                            double x, y, z;
                            rot_apply(R, X[f], Y[f], Z[f], x, y, z);
                            X[f] = x; Y[f] = y; Z[f] = z;
                            if ((f & 3) == 3) { cbx[f >> 2] = (float)x; cby[f >> 2] = (float)y; cbz[f >> 2] = (float)z; }
                        }
                    }
                }
                __syncthreads();
                ++k;
            } else {
                // ======== up to nspec proposals, warp r evaluating step k + r against the current state ====
                const int S = min(nspec, batch_end - k);
                if (warp < S) {
                    const int kk = k + warp, bi = kk - batch_start;
                    const int c = kk >> 1, split = c + (kk & 1);
                    const bool inert = (kk == 0) || (kk == n - 1);
                    double dE = 0.0;
                    Rot R;
                    if (!inert) {
                        R = step_rot(kk, bi);
                        const int ilo = max(0, c - a.window), jhi = min(L - 1, c + a.window);
                        float *px = lnw + (size_t)warp * 3 * wcap, *py = px + wcap, *pz = py + wcap;
                        for (int j = split + lane; j <= jhi; j += 32) {
                            double x, y, z;
                            rot_apply(R, X[4 * j + 3], Y[4 * j + 3], Z[4 * j + 3], x, y, z);
                            px[j - split] = (float)x; py[j - split] = (float)y; pz[j - split] = (float)z;
                        }
                        __syncwarp();
                        // ---- a4/a6: in-window cross pairs (Eq. 3b), warp reduction ------------------------
                        dE = warp_sum(cross_pairs_dE(m, cbx, cby, cbz, px, py, pz, split, ilo, split, jhi, lane, 32));
                    }
                    if (lane == 0) {
                        sp_dE[warp] = dE;
                        sp_acc[warp] = (b_lu[bi] <= -dE * invT) ? 1 : 0;   // Eq. 2a, R14
                        if (!inert) {
#pragma unroll
                            for (int q = 0; q < 9; ++q) rot_s[12 * warp + q] = R.r[q];
#pragma unroll
                            for (int q = 0; q < 3; ++q) rot_s[12 * warp + 9 + q] = R.t[q];
                        }
                    }
                }
                __syncthreads();
                int rs = S;                                   // first accepted step of the pass
                for (int q = S - 1; q >= 0; --q) if (sp_acc[q]) rs = q;
                const int nvalid = (rs < S) ? rs + 1 : S;     // steps whose result stands
                if (tid < nvalid) {
                    const long long q = (t - a.sweep_offset) * n + k + tid;
                    if (q < a.trace_steps) {
                        const size_t z = (size_t)row * a.trace_steps + q;
                        if (a.trace_prop) a.trace_prop[z] = b_sp[k + tid - batch_start];
                        if (a.trace_dE) a.trace_dE[z] = sp_dE[tid];
                        if (a.trace_acc) a.trace_acc[z] = (unsigned char)sp_acc[tid];
                    }
                }
                if (rs < S) {
                    // ---- a7: commit the accepted step --------------------------------------------------------
                    const int kc = k + rs, c = kc >> 1;
                    ++acc_l;
                    if (tid == 0) s[kc] = b_sp[kc - batch_start];
                    if (kc != 0 && kc != n - 1) {
                        Rot R;
#pragma unroll
                        for (int q = 0; q < 9; ++q) R.r[q] = rot_s[12 * rs + q];
#pragma unroll
                        for (int q = 0; q < 3; ++q) R.t[q] = rot_s[12 * rs + 9 + q];
                        const int m0 = 4 * c + 2 + 2 * (kc & 1);
                        for (int f = m0 + tid; f < 4 * L; f += nthreads) {
                            double x, y, z;
                            rot_apply(R, X[f], Y[f], Z[f], x, y, z);
                            X[f] = x; Y[f] = y; Z[f] = z;
                            if ((f & 3) == 3) { cbx[f >> 2] = (float)x; cby[f >> 2] = (float)y; cbz[f >> 2] = (float)z; }
                        }
                    }
                }
                __syncthreads();
                k += nvalid;
            }
        }
        // ---- a9: book-keeping at the sweep end ----------------------------------------------------
        e_end = full_energy();
        if (e_end < best) {
            best = e_end;
            if (a.best_state)
                for (int q = tid; q < n; q += nthreads) a.best_state[row * n + q] = s[q];
        }
        if (tid == 0 && a.first_hit && (float)e_end <= a.energy_threshold) atomicMin(a.first_hit, (unsigned long long)t);
    }
    if (a.n_sweeps == 0) e_end = full_energy();
    for (int q = tid; q < n; q += nthreads) a.states[row * n + q] = s[q];
    if (tid == 0) {
        if (a.energy) a.energy[row] = (float)e_end;
        if (a.best_energy) a.best_energy[row] = (float)best;
        if (a.n_accept_local) a.n_accept_local[row] = acc_l;
        if (a.n_accept_global) a.n_accept_global[row] = acc_g;
    }
}

}  // namespace amh
