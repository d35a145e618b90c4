// amh_kernels.cuh - the kernels of the AMH hot path (sm_100a): table build, x = G(s), V / V_local of
// a batch, and the per-chain alternating MH sweep kernel.  See DESIGN.md "Kernels" for the layout
// and the roofline of each.
#pragma once
#include "amh_device.cuh"

namespace amh {

// ------------------------------------------------------------------------------------------------
// a0  E = -log(p + eps)   (Eq. 3a; BASELINE.json:7's 1e-8)
// ------------------------------------------------------------------------------------------------
__global__ void table_kernel(const float *__restrict__ p, float *__restrict__ E, long long count, double eps,
                             int *__restrict__ bad)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    int local_bad = 0;
    for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < count; q += stride) {
        const float v = p[q];
        if (!(v >= 0.0f) || isinf(v)) local_bad = 1;
        E[q] = (float)(-log((double)v + eps));
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
        const float *rowi = m.E + (size_t)i * m.L * m.nb;
        for (int j = i + m.min_sep + lane; j <= hi; j += 32) {
            const float dx = xi - cbx[j], dy = yi - cby[j], dz = zi - cbz[j];
            const float d2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
            e += (double)pair_energy(rowi + (size_t)j * m.nb, d2, m.c0, m.inv_delta, m.tmax, m.nb);
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
// shared (per chain):  double X[4L], Y[4L], Z[4L]   N, CA, C, CB of every residue, flat index 4*res + atom
//                      double red[16]; double b_cd[16], b_sd[16], b_lu[16]
//                      float  cb[3][L]   fp32 copy of the C-betas (what the pair loop reads)
//                      float  nw[3][L]   candidate C-betas of the proposal
//                      float  s[n]; float b_sp[16]
// ------------------------------------------------------------------------------------------------
struct RunArgs {
    float *states;
    long long B, n_sweeps, sweep_offset, chain_offset;
    int n_global, n_local, window, global_first;
    double t_start, t_end;
    long long ramp_sweeps;
    const float *per_chain_T;
    int prop_mode, grid;
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

__host__ __device__ inline size_t sweep_smem_bytes(int L)
{
    return sizeof(double) * (12 * (size_t)L + 16 * 4) + sizeof(float) * (6 * (size_t)L + 2 * (size_t)L + 16);
}

struct Rot { double r[9], t[3]; };

__device__ __forceinline__ void rot_apply(const Rot &R, double x, double y, double z, double &ox, double &oy, double &oz)
{
    ox = fma(R.r[0], x, fma(R.r[1], y, fma(R.r[2], z, R.t[0])));
    oy = fma(R.r[3], x, fma(R.r[4], y, fma(R.r[5], z, R.t[1])));
    oz = fma(R.r[6], x, fma(R.r[7], y, fma(R.r[8], z, R.t[2])));
}

// rotation by (cd, sd) = (cos, sin) of the torsion change about the axis a -> b (right-handed about b - a,
// which raises the IUPAC dihedral of everything bonded after b)
__device__ __forceinline__ Rot rot_about(double ax, double ay, double az, double bx, double by, double bz,
                                         double cd, double sd)
{
    double ux = bx - ax, uy = by - ay, uz = bz - az;
    const double inv = rsqrt(fma(ux, ux, fma(uy, uy, uz * uz)));
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

__global__ void __launch_bounds__(512) sweep_kernel(DevModel m, RunArgs a)
{
    extern __shared__ double smem_d[];
    const int L = m.L, n = m.n;
    double *X = smem_d, *Y = X + 4 * L, *Z = Y + 4 * L;
    double *red = Z + 4 * L, *b_cd = red + 16, *b_sd = b_cd + 16, *b_lu = b_sd + 16;
    float *cbx = reinterpret_cast<float *>(b_lu + 16), *cby = cbx + L, *cbz = cby + L;
    float *nwx = cbz + L, *nwy = nwx + L, *nwz = nwy + L;
    float *s = nwz + L;
    float *b_sp = s + n;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nthreads = blockDim.x, nwarps = nthreads >> 5;
    const bool multi = nwarps > 1;
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

    auto full_energy = [&]() -> double {     // all threads; returns the same value in every thread
        double e = warp_sum(energy_range_cta(m, cbx, cby, cbz, 0, L - 1, warp, nwarps, lane));
        if (lane == 0) red[warp] = e;
        __syncthreads();
        double tot = 0.0;
        for (int w = 0; w < nwarps; ++w) tot += red[w];
        __syncthreads();
        return tot;
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

        // local sweeps run on warp 0 alone (<= ~150 pairs per proposal); global sweeps use the whole CTA
        if (is_global || warp == 0) {
            const int nthr = is_global ? nthreads : 32;
            const bool cta_wide = is_global && multi;
            auto sync = [&]() { if (cta_wide) __syncthreads(); else __syncwarp(); };
            for (int k = 0; k < n; ++k) {
                // ---- a1/a2: draws for the next 16 steps, one lane per (step, purpose) -------------
                if ((k & 15) == 0) {
                    if (warp == 0) {
                        const int kk = k + (lane >> 1);
                        if (kk < n) {
                            const unsigned long long step = (unsigned long long)t * (unsigned long long)n + (unsigned long long)kk;
                            const uint32_t x0 = draw0(a.seed, chain, step, lane & 1);
                            if ((lane & 1) == PURPOSE_PROPOSAL) {
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
                                b_sp[lane >> 1] = sp; b_cd[lane >> 1] = cd; b_sd[lane >> 1] = sd;
                            } else {
                                b_lu[lane >> 1] = log((double)((x0 >> 8) + 1u) * 5.9604644775390625e-08);
                            }
                        }
                    }
                    sync();
                }
                const float sp = b_sp[k & 15];
                const double lu = b_lu[k & 15];
                const int c = k >> 1, split = c + (k & 1);
                double dE = 0.0;
                const bool inert = (k == 0) || (k == n - 1);
                Rot R;
                if (!inert) {
                    // ---- a3: rotation of the right-hand side about the flipped bond ---------------
                    const int fa = 4 * c + (k & 1), fb = fa + 1;          // phi: N->CA, psi: CA->C
                    R = rot_about(X[fa], Y[fa], Z[fa], X[fb], Y[fb], Z[fb], b_cd[k & 15], b_sd[k & 15]);
                    const int ilo = is_global ? 0 : max(0, c - a.window);
                    const int jhi = is_global ? L - 1 : min(L - 1, c + a.window);
                    for (int j = split + tid; j <= jhi; j += nthr) {
                        double x, y, z;
                        rot_apply(R, X[4 * j + 3], Y[4 * j + 3], Z[4 * j + 3], x, y, z);
                        nwx[j] = (float)x; nwy[j] = (float)y; nwz[j] = (float)z;
                    }
                    sync();
                    // ---- a4/a5: sum over the pairs that straddle the bond of e(new) - e(old) ------
                    const int nI = split - ilo, nJ = jhi - split + 1;
                    double acc = 0.0;
                    if (nI > 0 && nJ > 0) {
                        const int total = nI * nJ;
                        const int stepI = nthr / nJ, stepJ = nthr - stepI * nJ;
                        int ii = tid / nJ, jj = tid - ii * nJ;
                        for (int q = tid; q < total; q += nthr) {
                            const int i = ilo + ii, j = split + jj;
                            if (j - i >= m.min_sep) {
                                const float xi = cbx[i], yi = cby[i], zi = cbz[i];
                                const float *rowp = m.E + ((size_t)i * L + j) * m.nb;
                                float dx = xi - nwx[j], dy = yi - nwy[j], dz = zi - nwz[j];
                                const float en = pair_energy(rowp, fmaf(dx, dx, fmaf(dy, dy, dz * dz)), m.c0, m.inv_delta, m.tmax, m.nb);
                                dx = xi - cbx[j]; dy = yi - cby[j]; dz = zi - cbz[j];
                                const float eo = pair_energy(rowp, fmaf(dx, dx, fmaf(dy, dy, dz * dz)), m.c0, m.inv_delta, m.tmax, m.nb);
                                acc += (double)(en - eo);
                            }
                            ii += stepI; jj += stepJ;
                            if (jj >= nJ) { jj -= nJ; ++ii; }
                        }
                    }
                    // ---- a6: reduction ------------------------------------------------------------
                    acc = warp_sum(acc);
                    if (cta_wide) {
                        if (lane == 0) red[warp] = acc;
                        __syncthreads();
                        acc = 0.0;
                        for (int w = 0; w < nwarps; ++w) acc += red[w];
                    }
                    dE = acc;
                }
                // ---- a7: Metropolis test, accept iff log u <= -dE / T   (Eq. 1a/2a, R14) -----------
                const bool accept = lu <= -dE * invT;
                if (tid == 0) {
                    const long long q = (t - a.sweep_offset) * n + k;
                    if (q < a.trace_steps) {
                        const size_t z = (size_t)row * a.trace_steps + q;
                        if (a.trace_prop) a.trace_prop[z] = sp;
                        if (a.trace_dE) a.trace_dE[z] = dE;
                        if (a.trace_acc) a.trace_acc[z] = accept ? 1 : 0;
                    }
                }
                if (accept) {
                    if (is_global) ++acc_g; else ++acc_l;
                    if (tid == 0) s[k] = sp;
                    if (!inert) {
                        const int m0 = 4 * c + 2 + 2 * (k & 1);           // first flat atom that moves
                        for (int f = m0 + tid; f < 4 * L; f += nthr) {
                            double x, y, z;
                            rot_apply(R, X[f], Y[f], Z[f], x, y, z);
                            X[f] = x; Y[f] = y; Z[f] = z;
                            if ((f & 3) == 3) { cbx[f >> 2] = (float)x; cby[f >> 2] = (float)y; cbz[f >> 2] = (float)z; }
                        }
                    }
                    sync();
                }
            }
        }
        __syncthreads();
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
