// amh_sweep.cuh - the alternating MH sweep kernel (rows a1-a9 of DESIGN.md section 0), sm_100a.
//
// Launch shape.  One CTA runs C chains; each chain owns W consecutive warps (its "team") and a named
// barrier; one more warp (the last) is the PRODUCER that feeds the table ring by TMA bulk copies.
// Chains are independent: teams never wait for one another except through the ring.
//
// Global sweeps (Eq. 1, 3a): the team evaluates one proposal at a time over its O(L^2/6) straddling
// pairs; rows of far pairs are never touched, near pairs gather 8 bytes from the packed table in L2.
//
// Local sweeps (Eq. 2, 3b): a proposal has only ~65-150 pairs, and Alg. 1 orders the proposals of a
// chain strictly.
//   * Speculation.  The draws are counter-based (R6), so the proposals of steps k, k+1, ... are known in
//     advance: warp r of the team evaluates step k+r AGAINST THE CURRENT STATE, and the results are
//     consumed in order up to and including the first accepted step; later results were computed against
//     a state that no longer exists and are thrown away (their steps are evaluated again in the next
//     pass).  The trajectory is exactly the sequential one.
//   * Table ring.  Every chain of the CTA walks k = 0..n-1, so they all need the same table rows at about
//     the same time: pair (i, j) is needed while the window centre c is in [max(i, j-w), min(j, i+w)].
//     The producer streams "column" j = the rows (i, j), j-2w <= i <= j-min_sep, into slot q mod R of a
//     shared-memory ring (q = a running column number) with cp.async.bulk + mbarrier complete_tx; teams
//     wait on the slot's barrier, gather from shared memory (32 banks instead of one L1 wavefront per
//     lane) and publish their progress; a slot is refilled once every team has passed its column.
#pragma once
#include "amh_device.cuh"

namespace amh {

struct RunArgs {
    float *states;
    long long B, n_sweeps, sweep_offset, chain_offset;
    int n_global, n_local, window, global_first;
    double t_start, t_end;
    long long ramp_sweeps;
    const float *per_chain_T;
    int prop_mode, grid;
    // launch shape
    int C, W;                            // chains per CTA, warps per chain
    int spec_local;                      // local proposals evaluated per pass (<= W)
    int ring_cols;                       // R: slots of the table ring (> window + 2), 0 = gather from L2 instead
    int ring_rows;                       // rows per column: 2w - min_sep + 1
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
constexpr int kMaxWarps = 16;            // array bound of the per-warp scratch of a team
constexpr int kMaxTeamWarps = 15;        // team warps per CTA: chains x warps per chain (+ the producer = 512 threads)
constexpr int kMaxChains = 15;           // chains per CTA (named barriers 1..15)
constexpr int kSweepMaxThreads = 512;    // 15 team warps + the producer: 128 registers per thread

__host__ __device__ inline int sweep_wcap(int L, int window) { return (window + 1 < L) ? window + 1 : L; }

// shared memory of one chain, in bytes (a multiple of 16)
__host__ __device__ inline size_t chain_smem_bytes(int L, int window, int W)
{
    const size_t doubles = 12 * (size_t)L + kMaxWarps + 3 * kDrawBatch + 12 * kMaxWarps + kMaxWarps;
    size_t floats = 6 * (size_t)L + 2 * (size_t)L + kDrawBatch + (size_t)W * 3 * sweep_wcap(L, window) + kMaxWarps;
    floats = (floats + 3) & ~(size_t)3;
    return sizeof(double) * doubles + sizeof(float) * floats;
}

// header: ring barriers, progress words; then the ring; then the chains
__host__ __device__ inline size_t sweep_header_bytes(int ring_cols) { return (8 * (size_t)ring_cols + 8 * 16 + 15) & ~(size_t)15; }

__host__ __device__ inline size_t sweep_smem_bytes(int L, int window, int C, int W, int ring_cols, int ring_rows, int row_stride)
{
    size_t b = sweep_header_bytes(ring_cols) + sizeof(float) * (size_t)ring_cols * ring_rows * row_stride;
    b = (b + 15) & ~(size_t)15;
    return b + (size_t)C * chain_smem_bytes(L, window, W);
}

// ---- PTX: mbarrier, TMA bulk copy, named barriers ----------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(void *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(void *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(void *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(void *bar, uint32_t parity)
{
    const uint32_t a = smem_u32(bar);
    uint32_t ok;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(a), "r"(parity) : "memory");
    } while (!ok);
}
// global -> shared bulk copy (TMA, no tensor map); bytes is a multiple of 16, both addresses 16-byte aligned
__device__ __forceinline__ void tma_bulk_g2s(void *dst, const void *src, uint32_t bytes, void *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void team_bar(int id, int threads)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(threads) : "memory");
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

// the pair term from a plain row E[0..nb-1] in shared memory: the same fp32 operations, in the same order,
// as pair_energy() on the packed row (E[b+1] - E[b] is formed here instead of at create)
__device__ __forceinline__ float pair_energy_row(const float *row, float d2, float c0, float inv_delta, float tmax, int nb)
{
    const float d = sqrtf(d2);
    float t = (d - c0) * inv_delta;
    t = fminf(fmaxf(t, 0.0f), tmax);
    int b = (int)t;
    b = min(b, nb - 2);
    const float f = t - (float)b;
    const float e0 = row[b], e1 = row[b + 1];
    return fmaf(f, e1 - e0, e0);
}

// Where the rows of a local proposal come from: the shared-memory ring or, when the ring is off, the
// packed table in L2.  slot0 = ring slot of column j = split of the step being evaluated.
struct RowSource {
    const float *ring;       // nullptr = gather from m.Epk
    int ring_cols, ring_rows, span, slot0;
};

// sum over the pairs (i, j), ilo <= i < split <= j <= jhi, j - i >= min_sep, of e(new) - e(old); the candidate
// C-beta of residue j is (nx, ny, nz)[j - joff].  Work is dealt to `nthr` threads, this one being `tid`.
template <bool RING>
__device__ __forceinline__ double cross_pairs_dE(const DevModel &m, const RowSource &rs, const float *cbx, const float *cby,
                                                 const float *cbz, const float *nx, const float *ny, const float *nz,
                                                 int joff, int ilo, int split, int jhi, int tid, int nthr)
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
                float en, eo;
                if (RING) {
                    int slot = rs.slot0 + jj;                      // nJ <= w + 1 < ring_cols: one wrap at most
                    if (slot >= rs.ring_cols) slot -= rs.ring_cols;
                    const float *rowp = rs.ring + ((size_t)slot * rs.ring_rows + (i - j + rs.span)) * m.row_stride;
                    en = pair_energy_row(rowp, d2n, m.c0, m.inv_delta, m.tmax, m.nb);
                    eo = pair_energy_row(rowp, d2o, m.c0, m.inv_delta, m.tmax, m.nb);
                } else {
                    const float2 *rowp = m.Epk + (tri_base(i, m.L) + j) * m.nb;
                    en = pair_energy(rowp, d2n, m.c0, m.inv_delta, m.tmax, m.nb);
                    eo = pair_energy(rowp, d2o, m.c0, m.inv_delta, m.tmax, m.nb);
                }
                acc += (double)(en - eo);
            }
        }
        ii += stepI; jj += stepJ;
        if (jj >= nJ) { jj -= nJ; ++ii; }
    }
    return acc;
}

// V (Eq. 3a) of the team's chain from its fp32 C-betas; every thread of the team returns the same value
__device__ __forceinline__ double team_full_energy(const DevModel &m, const float *cbx, const float *cby, const float *cbz,
                                                   double *red, int warp, int nwarps, int lane, int bar_id)
{
    double e = warp_sum(energy_range_cta(m, cbx, cby, cbz, 0, m.L - 1, warp, nwarps, lane));
    if (lane == 0) red[warp] = e;
    team_bar(bar_id, nwarps * 32);
    double tot = 0.0;
    for (int w = 0; w < nwarps; ++w) tot += red[w];
    team_bar(bar_id, nwarps * 32);
    return tot;
}

__global__ void __launch_bounds__(kSweepMaxThreads, 1) sweep_kernel(DevModel m, RunArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int L = m.L, n = m.n;
    const int C = a.C, W = a.W, R = a.ring_cols;
    const int lane = threadIdx.x & 31, warp_cta = threadIdx.x >> 5;
    const int slot = warp_cta / W;                        // chain slot of this warp; C = the producer warp
    const int warp = warp_cta - slot * W;                 // warp within the team
    const int tid = warp * 32 + lane, nthreads = W * 32, nwarps = W;
    const int bar_id = 1 + slot;
    const int wcap = sweep_wcap(L, a.window);
    const int span = min(2 * a.window, L - 1);            // largest j - i of an in-window pair
    const bool use_ring = R > 0;

    unsigned long long *full_bar = reinterpret_cast<unsigned long long *>(smem_raw);                 // [R]
    volatile long long *prog = reinterpret_cast<volatile long long *>(smem_raw + 8 * (size_t)R);      // [16]
    float *ring = reinterpret_cast<float *>(smem_raw + sweep_header_bytes(R));
    const size_t chains_off = (sweep_header_bytes(R) + sizeof(float) * (size_t)R * a.ring_rows * m.row_stride + 15) & ~(size_t)15;

    const long long row0 = (long long)blockIdx.x * C;
    const int nvalid = (int)min((long long)C, a.B - row0);
    const long long cyc = (long long)a.n_global + a.n_local;
    auto sweep_is_global = [&](long long t) -> bool {
        const long long r = t % cyc;
        return a.global_first ? (r < a.n_global) : (r >= a.n_local);
    };

    if (threadIdx.x == 0) {
        for (int q = 0; q < R; ++q) mbar_init(&full_bar[q], 1);
        for (int g = 0; g < 16; ++g) prog[g] = (g < nvalid) ? 0 : 0x7fffffffffffffffLL;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // ================= producer warp: stream the columns of every local sweep through the ring ===========
    if (slot == C) {
        if (!use_ring) return;
        const uint32_t row_bytes = (uint32_t)(m.row_stride * sizeof(float));
        long long q0 = 0;                                   // running number of column j = 0 of the sweep
        for (long long t = a.sweep_offset; t < a.sweep_offset + a.n_sweeps; ++t) {
            if (sweep_is_global(t)) continue;
            for (int j = 0; j < L; ++j) {
                const long long q = q0 + j;
                if (lane == 0) {                            // slot q mod R is free once every team has passed column q - R
                    for (;;) {
                        long long mn = 0x7fffffffffffffffLL;
                        for (int g = 0; g < nvalid; ++g) mn = min(mn, prog[g]);
                        if (q - R < mn) break;
                        __nanosleep(40);
                    }
                }
                __syncwarp();
                const int i_lo = max(0, j - span), i_hi = j - m.min_sep;
                const int nrows = i_hi - i_lo + 1;
                const int s = (int)(q % R);
                void *bar = &full_bar[s];
                if (lane == 0) {
                    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // the teams' reads of the old column come first
                    if (nrows > 0) mbar_expect_tx(bar, (uint32_t)nrows * row_bytes);
                    else mbar_arrive(bar);
                }
                __syncwarp();
                // one lane issues the copies of the column: the operands of a bulk copy live in uniform registers,
                // so a lane-divergent issue loop would be serialised lane by lane anyway
                if (lane == 0)
                    for (int i = i_lo; i <= i_hi; ++i)
                        tma_bulk_g2s(ring + ((size_t)s * a.ring_rows + (i - j + span)) * m.row_stride,
                                     m.Epl + (size_t)(tri_base(i, L) + j) * m.row_stride, row_bytes, bar);
                __syncwarp();
            }
            q0 += L;
        }
        return;
    }
    if (slot >= nvalid) return;

    // ================= team: one chain =====================================================================
    unsigned char *cbase = smem_raw + chains_off + (size_t)slot * chain_smem_bytes(L, a.window, W);
    double *X = reinterpret_cast<double *>(cbase), *Y = X + 4 * L, *Z = Y + 4 * L;
    double *red = Z + 4 * L, *b_cd = red + kMaxWarps, *b_sd = b_cd + kDrawBatch, *b_lu = b_sd + kDrawBatch;
    double *rot_s = b_lu + kDrawBatch, *sp_dE = rot_s + 12 * kMaxWarps;
    float *cbx = reinterpret_cast<float *>(sp_dE + kMaxWarps), *cby = cbx + L, *cbz = cby + L;
    float *nwx = cbz + L, *nwy = nwx + L, *nwz = nwy + L;
    float *s = nwz + L;
    float *b_sp = s + n;
    float *lnw = b_sp + kDrawBatch;
    int *sp_acc = reinterpret_cast<int *>(lnw + (size_t)nwarps * 3 * wcap);

    const long long row = row0 + slot;
    const unsigned long long chain = (unsigned long long)(a.chain_offset + row);

    for (int q = tid; q < n; q += nthreads) s[q] = a.states[row * n + q];
    team_bar(bar_id, nthreads);
    if (warp == 0)
        nerf_build_warp(m, s, lane, [&](int res, int at, double x, double y, double z) {
            const int f = 4 * res + at;
            X[f] = x; Y[f] = y; Z[f] = z;
            if (at == 3) { cbx[res] = (float)x; cby[res] = (float)y; cbz[res] = (float)z; }
        });
    team_bar(bar_id, nthreads);

    double best = INFINITY, e_end = 0.0;
    unsigned long long acc_l = 0, acc_g = 0;
    const int nspec = max(1, min(nwarps, a.spec_local > 0 ? a.spec_local : nwarps));
    const int draw_warp_u = nwarps > 1 ? 1 : 0;              // the warp that draws the uniforms of the accept test
    long long q0 = 0;                                        // running column number of j = 0 (local sweeps)
    RowSource rs;
    rs.ring = use_ring ? ring : nullptr; rs.ring_cols = R; rs.ring_rows = a.ring_rows; rs.span = span; rs.slot0 = 0;

    // the bond the torsion k turns about: phi_c N->CA, psi_c CA->C
    auto step_rot = [&](int k, int bi) -> Rot {
        const int fa = 4 * (k >> 1) + (k & 1), fb = fa + 1;
        return rot_about(X[fa], Y[fa], Z[fa], X[fb], Y[fb], Z[fb], b_cd[bi], b_sd[bi], (k & 1) ? m.inv_len_ca_c : m.inv_len_n_ca);
    };
    // the accepted rotation moves every atom bonded after the turned bond
    auto commit = [&](const Rot &R_, int k) {
        const int m0 = 4 * (k >> 1) + 2 + 2 * (k & 1);       // first flat atom that moves
        for (int f = m0 + tid; f < 4 * L; f += nthreads) {
            double x, y, z;
            rot_apply(R_, X[f], Y[f], Z[f], x, y, z);
            X[f] = x; Y[f] = y; Z[f] = z;
            if ((f & 3) == 3) { cbx[f >> 2] = (float)x; cby[f >> 2] = (float)y; cbz[f >> 2] = (float)z; }
        }
    };

    for (long long t = a.sweep_offset; t < a.sweep_offset + a.n_sweeps; ++t) {
        const bool is_global = sweep_is_global(t);
        double T;
        if (a.per_chain_T) T = (double)a.per_chain_T[row];
        else if (a.t_start == a.t_end || a.ramp_sweeps <= 1 || t <= 0) T = a.t_start;
        else if (t >= a.ramp_sweeps - 1) T = a.t_end;
        else T = a.t_start * pow(a.t_end / a.t_start, (double)t / (double)(a.ramp_sweeps - 1));
        const double invT = 1.0 / T;
        long long seen = q0 - 1;                             // last ring column this team has waited for

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
                team_bar(bar_id, nthreads);
            }
            if (is_global) {
                // ======== one proposal, evaluated by the whole team ========================================
                const int bi = k - batch_start;
                const int c = k >> 1, split = c + (k & 1);
                const bool inert = (k == 0) || (k == n - 1);
                double dE = 0.0;
                Rot Rk;
                if (!inert) {
                    // ---- a3: rotation of the right-hand side about the flipped bond ------------------------
                    Rk = step_rot(k, bi);
                    for (int j = split + tid; j < L; j += nthreads) {
                        double x, y, z;
                        rot_apply(Rk, X[4 * j + 3], Y[4 * j + 3], Z[4 * j + 3], x, y, z);
                        nwx[j] = (float)x; nwy[j] = (float)y; nwz[j] = (float)z;
                    }
                    team_bar(bar_id, nthreads);
                    // ---- a5/a6: cross pairs, then the reduction -------------------------------------------
                    double acc = warp_sum(cross_pairs_dE<false>(m, rs, cbx, cby, cbz, nwx, nwy, nwz, 0, 0, split, L - 1, tid, nthreads));
                    if (lane == 0) red[warp] = acc;
                    team_bar(bar_id, nthreads);
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
                    if (!inert) commit(Rk, k);
                }
                team_bar(bar_id, nthreads);
                ++k;
            } else {
                // ======== up to nspec proposals, warp r evaluating step k + r against the current state ====
                const int S = min(nspec, batch_end - k);
                if (use_ring) {
                    // columns left of the window centre are dead for this chain; wait for the ones the pass needs
                    if (tid == 0) prog[slot] = q0 + (k >> 1);
                    const long long need = q0 + min(L - 1, ((k + S - 1) >> 1) + a.window);
                    while (seen < need) {
                        ++seen;
                        mbar_wait(&full_bar[seen % R], (uint32_t)((seen / R) & 1));
                    }
                }
                if (warp < S) {
                    const int kk = k + warp, bi = kk - batch_start;
                    const int c = kk >> 1, split = c + (kk & 1);
                    const bool inert = (kk == 0) || (kk == n - 1);
                    double dE = 0.0;
                    Rot Rk;
                    if (!inert) {
                        Rk = step_rot(kk, bi);
                        const int ilo = max(0, c - a.window), jhi = min(L - 1, c + a.window);
                        float *px = lnw + (size_t)warp * 3 * wcap, *py = px + wcap, *pz = py + wcap;
                        for (int j = split + lane; j <= jhi; j += 32) {
                            double x, y, z;
                            rot_apply(Rk, X[4 * j + 3], Y[4 * j + 3], Z[4 * j + 3], x, y, z);
                            px[j - split] = (float)x; py[j - split] = (float)y; pz[j - split] = (float)z;
                        }
                        __syncwarp();
                        // ---- a4/a6: in-window cross pairs (Eq. 3b), warp reduction ------------------------
                        if (use_ring) rs.slot0 = (int)((q0 + split) % R);
                        dE = warp_sum(use_ring ? cross_pairs_dE<true>(m, rs, cbx, cby, cbz, px, py, pz, split, ilo, split, jhi, lane, 32)
                                               : cross_pairs_dE<false>(m, rs, cbx, cby, cbz, px, py, pz, split, ilo, split, jhi, lane, 32));
                    }
                    if (lane == 0) {
                        sp_dE[warp] = dE;
                        sp_acc[warp] = (b_lu[bi] <= -dE * invT) ? 1 : 0;   // Eq. 2a, R14
                        if (!inert) {
#pragma unroll
                            for (int q = 0; q < 9; ++q) rot_s[12 * warp + q] = Rk.r[q];
#pragma unroll
                            for (int q = 0; q < 3; ++q) rot_s[12 * warp + 9 + q] = Rk.t[q];
                        }
                    }
                }
                team_bar(bar_id, nthreads);
                int rsel = S;                                 // first accepted step of the pass
                for (int q = S - 1; q >= 0; --q) if (sp_acc[q]) rsel = q;
                const int nstand = (rsel < S) ? rsel + 1 : S; // steps whose result stands
                if (tid < nstand) {
                    const long long q = (t - a.sweep_offset) * n + k + tid;
                    if (q < a.trace_steps) {
                        const size_t z = (size_t)row * a.trace_steps + q;
                        if (a.trace_prop) a.trace_prop[z] = b_sp[k + tid - batch_start];
                        if (a.trace_dE) a.trace_dE[z] = sp_dE[tid];
                        if (a.trace_acc) a.trace_acc[z] = (unsigned char)sp_acc[tid];
                    }
                }
                if (rsel < S) {
                    // ---- a7: commit the accepted step --------------------------------------------------------
                    const int kc = k + rsel;
                    ++acc_l;
                    if (tid == 0) s[kc] = b_sp[kc - batch_start];
                    if (kc != 0 && kc != n - 1) {
                        Rot Rk;
#pragma unroll
                        for (int q = 0; q < 9; ++q) Rk.r[q] = rot_s[12 * rsel + q];
#pragma unroll
                        for (int q = 0; q < 3; ++q) Rk.t[q] = rot_s[12 * rsel + 9 + q];
                        commit(Rk, kc);
                    }
                }
                team_bar(bar_id, nthreads);
                k += nstand;
            }
        }
        if (!is_global) {
            q0 += L;
            if (use_ring && tid == 0) prog[slot] = q0;       // every column of this sweep is dead for this chain
        }
        // ---- a9: book-keeping at the sweep end ----------------------------------------------------
        e_end = team_full_energy(m, cbx, cby, cbz, red, warp, nwarps, lane, bar_id);
        if (e_end < best) {
            best = e_end;
            if (a.best_state)
                for (int q = tid; q < n; q += nthreads) a.best_state[row * n + q] = s[q];
        }
        if (tid == 0 && a.first_hit && (float)e_end <= a.energy_threshold) atomicMin(a.first_hit, (unsigned long long)t);
    }
    if (a.n_sweeps == 0) e_end = team_full_energy(m, cbx, cby, cbz, red, warp, nwarps, lane, bar_id);
    for (int q = tid; q < n; q += nthreads) a.states[row * n + q] = s[q];
    if (tid == 0) {
        if (a.energy) a.energy[row] = (float)e_end;
        if (a.best_energy) a.best_energy[row] = (float)best;
        if (a.n_accept_local) a.n_accept_local[row] = acc_l;
        if (a.n_accept_global) a.n_accept_global[row] = acc_g;
    }
}

}  // namespace amh
