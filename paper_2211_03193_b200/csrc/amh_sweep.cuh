// amh_sweep.cuh - the alternating MH sweep kernel (rows a1-a9 of DESIGN.md section 0), sm_100a.
//
// Launch shape.  One CTA runs C chains; each chain owns W consecutive warps (its "team") and a named
// barrier; one more warp (the last) is the PRODUCER that feeds the table ring by TMA bulk copies.
// Chains are independent: teams never wait for one another except through the ring.
//
// Global sweeps (Eq. 1, 3a): O(L^2/6) straddling pairs per proposal, evaluated either by the whole team one
// proposal at a time (SG = false) or speculatively like the local ones, one warp per step (SG = true).  A thread owns a column j: it turns CB_j itself and walks the rows i in blocks of 8; a block
// whose bounding sphere is beyond the last bin centre for both positions of CB_j is skipped whole, pairs
// clamped before and after are skipped one by one (their term is exactly 0), near pairs gather 8 bytes
// from the packed table in L2, four rows' gathers in flight at a time.
//
// Local sweeps (Eq. 2, 3b): a proposal has only ~65-150 pairs, and Alg. 1 orders the proposals of a
// chain strictly.
//   * Speculation.  The draws are counter-based (R6), so the proposals of steps k, k+1, ... are known in
//     advance: GROUP r (8, 16 or 32 lanes; up to 16 groups per team) evaluates step k+r AGAINST THE
//     CURRENT STATE, and the results are consumed in order up to and including the first accepted step;
//     later results were computed against a state that no longer exists and are thrown away (their steps
//     are evaluated again in the next pass).  The trajectory is exactly the sequential one.
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
    double sigma_start, sigma_end;       // Gaussian mode: linear ramp over ramp_sigma sweeps
    long long ramp_sigma;
    // launch shape
    int C, W;                            // chains per CTA, warps per chain
    int spec_local;                      // local proposals evaluated per pass (<= W * 32 / lanes_per_step, <= 16)
    int lanes_per_step;                  // lanes that share one local proposal: 32, 16 or 8
    int ring_cols;                       // R: slots of the table ring (> window + 2), 0 = gather from L2 instead
    int ring_rows;                       // rows per column: 2w - min_sep + 1
    int cb64;                            // fp64 C-betas kept in shared memory (else rebuilt from N, CA, C)
    unsigned long long seed;
    double guard_local, guard_global;    // exact-decision guard: bound on the fp32 error of dE at 32 A extent (0 = off)
    float *energy, *best_energy, *best_state;
    unsigned long long *n_accept_local, *n_accept_global;
    unsigned long long *first_hit;       // min over chains of the absolute sweep index; ~0ull = none
    float energy_threshold;
    int trace_steps;
    float *trace_prop;
    double *trace_dE;
    unsigned char *trace_acc;
};

constexpr int kDrawBatch = 64;           // steps whose draws are generated together, two per lane
constexpr int kMaxWarps = 16;            // array bound of the per-warp scratch of a team
constexpr int kMaxSpec = 16;             // local proposals evaluated per pass, at most
constexpr int kBlk = 8;                  // residues per culling block of the global phase
constexpr int kMaxTeamWarps = 15;        // team warps per CTA: chains x warps per chain (+ the producer = 512 threads)
constexpr int kMaxChains = 15;           // chains per CTA (named barriers 1..15)
constexpr int kSweepMaxThreads = 512;    // 15 team warps + the producer: 128 registers per thread

// shared memory of one chain, in bytes (a multiple of 16):
//   double X[aL], Y[aL], Z[aL]   atoms, index atom * L + res (atom 0..2 = N, CA, C; a = 3).  The C-beta is a fixed
//                                combination of the three (cb_point); it is kept in fp64 too (atom 3, a = 4) when
//                                that does not cost a resident chain (cb64), else rebuilt where needed
//   double red[16], b_cd[64], b_sd[64], b_lu[64], rot_s[16][12], sp_dE[16]
//   float4 cb4[L]                fp32 copy of the C-betas (what the pair loops read)
//   float4 blk4[ceil(L/8)]       bounding spheres of 8-residue blocks (culling in the global phase)
//   float  s[n], b_sp[64];  int sp_acc[16]
__host__ __device__ inline size_t chain_smem_bytes(int L, int cb64)
{
    const size_t doubles = (cb64 ? 12 : 9) * (size_t)L + (cb64 ? 0 : (L & 1)) + kMaxWarps + 3 * kDrawBatch + 12 * kMaxSpec + kMaxSpec;   // (L & 1): cb4 on 16 bytes
    size_t floats = 4 * (size_t)L + 4 * (((size_t)L + kBlk - 1) / kBlk) + 2 * (size_t)L + kDrawBatch + kMaxSpec;
    floats = (floats + 3) & ~(size_t)3;
    return sizeof(double) * doubles + sizeof(float) * floats;
}

// header: ring barriers, progress words; then the ring; then the chains
__host__ __device__ inline size_t sweep_header_bytes(int ring_cols) { return (8 * (size_t)ring_cols + 8 * 16 + 15) & ~(size_t)15; }

__host__ __device__ inline size_t sweep_smem_bytes(int L, int C, int ring_cols, int ring_rows, int row_stride, int cb64)
{
    size_t b = sweep_header_bytes(ring_cols) + sizeof(float) * (size_t)ring_cols * ring_rows * row_stride;
    b = (b + 15) & ~(size_t)15;
    return b + (size_t)C * chain_smem_bytes(L, cb64);
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
        // the last operand lets the hardware park the thread for up to ~1 us instead of spinning on the barrier
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(a), "r"(parity), "r"(1000u) : "memory");
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

// C-beta of residue `res` from its own N, CA, C (fp64): ideal geometry makes it a fixed combination of them (R3)
__device__ __forceinline__ void cb_point(const DevModel &m, const double *X, const double *Y, const double *Z, int L, int res,
                                         double &x, double &y, double &z)
{
    const double ax = X[L + res], ay = Y[L + res], az = Z[L + res];                                  // CA
    const double ex = (ax - X[res]) * m.inv_len_n_ca, ey = (ay - Y[res]) * m.inv_len_n_ca, ez = (az - Z[res]) * m.inv_len_n_ca;
    const double vx = X[2 * L + res] - ax, vy = Y[2 * L + res] - ay, vz = Z[2 * L + res] - az;        // C - CA
    x = fma(m.cbC, fma(ey, vz, -ez * vy), fma(m.cbB, vx, fma(m.cbA, ex, ax)));
    y = fma(m.cbC, fma(ez, vx, -ex * vz), fma(m.cbB, vy, fma(m.cbA, ey, ay)));
    z = fma(m.cbC, fma(ex, vy, -ey * vx), fma(m.cbB, vz, fma(m.cbA, ez, az)));
}

// bin index and fraction of R8's interpolation at squared distance d2.  d = sqrt.approx.f32(d2): one MUFU instruction,
// maximum relative error 2^-23 (PTX ISA), i.e. within 1 ulp of the correctly rounded root (the
// coordinates feeding d2 are themselves rounded to fp32), instead of sqrtf()'s 9 instructions with its special-case
// branch; d2 = 0 (coincident atoms) gives 0 and lands in the first bin.  Rows in the ring are plain E[0..nb-1]: the
// caller forms E[b+1] - E[b] itself, the same fp32 subtraction the packed table did at create.
__device__ __forceinline__ void lerp_coords(float d2, float t0, float inv_delta, float tmax, int nb, int &b, float &f)
{
    float d;
    asm("sqrt.approx.f32 %0, %1;" : "=f"(d) : "f"(d2));
    float t = fmaf(d, inv_delta, t0);                        // (d - c0) / delta with t0 = -c0 / delta: one fma
    t = fminf(fmaxf(t, 0.0f), tmax);
    b = min((int)t, nb - 2);
    f = t - (float)b;
}

// Where the rows of a local proposal come from: the shared-memory ring or, when the ring is off, the
// packed table in L2.  slot0 = ring slot of column j = split of the step being evaluated.
struct RowSource {
    const float *ring;       // nullptr = gather from m.Epk
    int ring_cols, ring_rows, span, slot0;
};

// floor(a / b) for 0 <= a < 2^16, 1 <= b < 2^10 without the integer-division sequence
__device__ __forceinline__ int small_div(int a, int b)
{
    return __float2int_rd(__fdividef((float)a + 0.5f, (float)b));
}

// row index of the pair i < j in 32 bits (L < 46341)
__device__ __forceinline__ int tri_row(int i, int j, int L) { return (i * (2 * L - i - 1)) / 2 - i - 1 + j; }

// sum over the pairs (i, j), ilo <= i < split <= j <= jhi, j - i >= min_sep, of e(new) - e(old), where new = the
// C-beta of j turned by R.  Work is dealt to `nthr` threads, this one being `tid`: a thread OWNS a column j -
// it turns CB_j itself (fp64, rounded once to fp32) and keeps both positions in registers - and walks the rows
// i; when a round has fewer columns than threads, S threads share a column and take every S-th row.
template <bool RING, bool CULL>
__device__ __forceinline__ double cross_pairs_dE(const DevModel &m, const RowSource &rs, const float4 *cb4, const float4 *blk4,
                                                 const double *X, const double *Y, const double *Z, bool cb64, const Rot &R,
                                                 int ilo, int split, int jhi, int tid, int nthr)
{
    const int nJ = jhi - split + 1;
    double acc = 0.0;
    if (split <= ilo || nJ <= 0) return acc;
    for (int c0 = 0; c0 < nJ; c0 += nthr) {
        const int nc = min(nthr, nJ - c0);
        int S = 1, col = tid, slice = 0;
        if (nc < nthr) {
            S = small_div(nthr, nc); slice = small_div(tid, nc); col = tid - slice * nc;
            if (slice >= S) break;
        }
        const int j = split + c0 + col;
        double x0, y0, z0, x, y, z;
        if (cb64) { x0 = X[3 * m.L + j]; y0 = Y[3 * m.L + j]; z0 = Z[3 * m.L + j]; }
        else cb_point(m, X, Y, Z, m.L, j, x0, y0, z0);
        rot_apply(R, x0, y0, z0, x, y, z);
        const float xn = (float)x, yn = (float)y, zn = (float)z;
        const float4 o = cb4[j];
        const int i_end = min(split - 1, j - m.min_sep);
        const float *colp = nullptr;
        if (RING) {
            int slot = rs.slot0 + (j - split);               // nJ <= w + 1 < ring_cols: one wrap at most
            if (slot >= rs.ring_cols) slot -= rs.ring_cols;
            colp = rs.ring + ((size_t)slot * rs.ring_rows + (rs.span - j)) * m.row_stride;   // + i * row_stride
        }
        // U rows per trip: all distances first, then all gathers, then the sums, so that a thread has 2U loads in
        // flight instead of stalling on each pair's row (the rows of near pairs come from L2, ~600 cycles away)
        constexpr int U = 4;
        auto trip = [&](int i, int stride) {
            float d2n[U], d2o[U];
            int iu[U];
            bool near[U];
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int ii = i + u * stride;
                const bool valid = ii <= i_end;
                iu[u] = valid ? ii : i;
                const float4 ci = cb4[iu[u]];
                float dx = ci.x - xn, dy = ci.y - yn, dz = ci.z - zn;
                d2n[u] = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
                dx = ci.x - o.x; dy = ci.y - o.y; dz = ci.z - o.z;
                d2o[u] = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
                // a pair beyond the last bin centre before and after scores the same clamped value twice:
                // its term is exactly 0 and its row is never touched
                // (in the window of a local proposal nearly every pair is near: the test is skipped there and a far
                // pair goes through the clamped interpolation, which gives the same two values and the same 0)
                near[u] = valid && (!CULL || d2n[u] < m.far2 || d2o[u] < m.far2);
            }
            float fn[U], fo[U];
            int bn[U], bo[U];
            if (RING) {
                float en0[U], en1[U], eo0[U], eo1[U];
#pragma unroll
                for (int u = 0; u < U; ++u) {
                    en0[u] = en1[u] = eo0[u] = eo1[u] = 0.0f;
                    if (near[u]) {
                        lerp_coords(d2n[u], m.t0, m.inv_delta, m.tmax, m.nb, bn[u], fn[u]);
                        lerp_coords(d2o[u], m.t0, m.inv_delta, m.tmax, m.nb, bo[u], fo[u]);
                        const float *rowp = colp + iu[u] * m.row_stride;
                        en0[u] = rowp[bn[u]]; en1[u] = rowp[bn[u] + 1];
                        eo0[u] = rowp[bo[u]]; eo1[u] = rowp[bo[u] + 1];
                    }
                }
#pragma unroll
                for (int u = 0; u < U; ++u)
                    if (near[u]) acc += (double)(fmaf(fn[u], en1[u] - en0[u], en0[u]) - fmaf(fo[u], eo1[u] - eo0[u], eo0[u]));
            } else {
                float2 vn[U], vo[U];
#pragma unroll
                for (int u = 0; u < U; ++u) {
                    vn[u] = vo[u] = make_float2(0.0f, 0.0f);
                    if (near[u]) {
                        lerp_coords(d2n[u], m.t0, m.inv_delta, m.tmax, m.nb, bn[u], fn[u]);
                        lerp_coords(d2o[u], m.t0, m.inv_delta, m.tmax, m.nb, bo[u], fo[u]);
                        const float2 *rowp = m.Epk + (size_t)tri_row(iu[u], j, m.L) * m.nb;
                        vn[u] = __ldg(rowp + bn[u]); vo[u] = __ldg(rowp + bo[u]);
                    }
                }
#pragma unroll
                for (int u = 0; u < U; ++u)
                    if (near[u]) acc += (double)(fmaf(fn[u], vn[u].y, vn[u].x) - fmaf(fo[u], vo[u].y, vo[u].x));
            }
        };
        if (CULL) {
            // rows in blocks of kBlk consecutive residues (ilo = 0): a block whose bounding sphere lies beyond the last
            // bin centre of BOTH positions of CB_j holds only pairs whose term is exactly 0, and is skipped whole;
            // the S threads that share a column take every S-th block
            const int nblk = i_end < 0 ? 0 : i_end / kBlk + 1;
            for (int b = slice; b < nblk; b += S) {
                const float4 bl = blk4[b];
                float dx = bl.x - xn, dy = bl.y - yn, dz = bl.z - zn;
                const float dn = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
                dx = bl.x - o.x; dy = bl.y - o.y; dz = bl.z - o.z;
                const float dq = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
                if (dn >= bl.w && dq >= bl.w) continue;
#pragma unroll
                for (int t = 0; t < kBlk / U; ++t)
                    if (b * kBlk + t * U <= i_end) trip(b * kBlk + t * U, 1);
            }
        } else {
            for (int i = ilo + slice; i <= i_end; i += U * S) trip(i, S);
        }
    }
    return acc;
}

// ---- exact-decision guard (R24) --------------------------------------------------------------
// dE of the proposal at variable k in fp64, every term from the fp64 atoms and from -log(p + eps) itself: this
// thread's share of the sum over (i, j), ilo <= i < split <= j <= jhi, j - i >= min_sep, of e(new) - e(old).
// Pairs beyond the last bin centre before and after contribute exactly 0 (R8's clamp) and are skipped.
__device__ __noinline__ double exact_dE_partial(const DevModel &m, const double *X, const double *Y, const double *Z, int cb64,
                                               int k, double cd, double sd, int ilo, int jhi, int tid, int nthr)
{
    const int L = m.L;
    const int split = (k >> 1) + (k & 1);
    const int nJ = jhi - split + 1, nI = split - ilo;
    if (nJ <= 0 || nI <= 0) return 0.0;
    const int fa = (k & 1) * L + (k >> 1), fb = fa + L;
    const Rot R = rot_about(X[fa], Y[fa], Z[fa], X[fb], Y[fb], Z[fb], cd, sd, (k & 1) ? m.inv_len_ca_c : m.inv_len_n_ca);
    double acc = 0.0;
    for (int idx = tid; idx < nI * nJ; idx += nthr) {
        const int ii = idx / nJ;
        const int i = ilo + ii, j = split + (idx - ii * nJ);
        if (j - i < m.min_sep) continue;
        double xi, yi, zi, xo, yo, zo, xn, yn, zn;
        if (cb64) {
            xi = X[3 * L + i]; yi = Y[3 * L + i]; zi = Z[3 * L + i];
            xo = X[3 * L + j]; yo = Y[3 * L + j]; zo = Z[3 * L + j];
        } else {
            cb_point(m, X, Y, Z, L, i, xi, yi, zi);
            cb_point(m, X, Y, Z, L, j, xo, yo, zo);
        }
        rot_apply(R, xo, yo, zo, xn, yn, zn);
        double dx = xi - xo, dy = yi - yo, dz = zi - zo;
        const double d2o = dx * dx + dy * dy + dz * dz;
        dx = xi - xn; dy = yi - yn; dz = zi - zn;
        const double d2n = dx * dx + dy * dy + dz * dz;
        if (d2o >= m.far2_d && d2n >= m.far2_d) continue;
        const float *prow = m.P + (size_t)tri_row(i, j, L) * m.nb;
        acc += pair_energy_exact(prow, sqrt(d2n), m.c0_d, m.delta_d, m.eps_d, m.nb)
             - pair_energy_exact(prow, sqrt(d2o), m.c0_d, m.delta_d, m.eps_d, m.nb);
    }
    return acc;
}

// sum over the team's threads; every thread returns the total (two team barriers)
__device__ __forceinline__ double team_sum(double v, double *red, int warp, int nwarps, int lane, int bar_id)
{
    v = warp_sum(v);
    if (lane == 0) red[warp] = v;
    team_bar(bar_id, nwarps * 32);
    double tot = 0.0;
    for (int w = 0; w < nwarps; ++w) tot += red[w];
    team_bar(bar_id, nwarps * 32);
    return tot;
}

// largest |coordinate| of the chain's C-betas (the fp32 rounding of a coordinate, hence the error bound of dE, scales with it)
__device__ __forceinline__ float team_extent(const float4 *cb4, int L, double *red, int tid, int nthr, int warp, int nwarps, int lane, int bar_id)
{
    float e = 0.0f;
    for (int i = tid; i < L; i += nthr) { const float4 c = cb4[i]; e = fmaxf(e, fmaxf(fabsf(c.x), fmaxf(fabsf(c.y), fabsf(c.z)))); }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) e = fmaxf(e, __shfl_xor_sync(0xffffffffu, e, d));
    if (lane == 0) red[warp] = (double)e;
    team_bar(bar_id, nwarps * 32);
    double tot = 0.0;
    for (int w = 0; w < nwarps; ++w) tot = fmax(tot, red[w]);
    team_bar(bar_id, nwarps * 32);
    return (float)tot;
}

// bounding spheres of the blocks [first, last] of kBlk consecutive C-betas: blk4[b] = {centre, ((dfar + radius)(1 + 1e-5))^2}
__device__ __forceinline__ void team_blocks(const DevModel &m, const float4 *cb4, float4 *blk4, int first, int tid, int nthr)
{
    const int nblk = (m.L + kBlk - 1) / kBlk;
    for (int b = first + tid; b < nblk; b += nthr) {
        const int lo = b * kBlk, hi = min(m.L, lo + kBlk);
        float cx = 0.0f, cy = 0.0f, cz = 0.0f;
        for (int i = lo; i < hi; ++i) { const float4 c = cb4[i]; cx += c.x; cy += c.y; cz += c.z; }
        const float inv = 1.0f / (float)(hi - lo);
        cx *= inv; cy *= inv; cz *= inv;
        float r2 = 0.0f;
        for (int i = lo; i < hi; ++i) {
            const float4 c = cb4[i];
            const float dx = c.x - cx, dy = c.y - cy, dz = c.z - cz;
            r2 = fmaxf(r2, fmaf(dx, dx, fmaf(dy, dy, dz * dz)));
        }
        const float t = (m.dfar + sqrtf(r2)) * 1.00001f + 1e-4f;
        blk4[b] = make_float4(cx, cy, cz, t * t);
    }
}

// V (Eq. 3a) of the team's chain from its fp32 C-betas; every thread of the team returns the same value
__device__ __forceinline__ double team_full_energy(const DevModel &m, const float4 *cb4, double *red, int warp, int nwarps,
                                                   int lane, int bar_id)
{
    double e = 0.0;
    constexpr int U = 4;                                     // columns per trip: all gathers of a trip in flight together
    for (int i = warp; i < m.L - m.min_sep; i += nwarps) {
        const float4 ci = cb4[i];
        const int rb = tri_row(i, 0, m.L);
        for (int j0 = i + m.min_sep + lane; j0 < m.L; j0 += 32 * U) {
            float d2[U], v[U], f[U];
            float2 g[U];
            bool far[U];
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int j = min(j0 + 32 * u, m.L - 1);
                const float4 cj = cb4[j];
                const float dx = ci.x - cj.x, dy = ci.y - cj.y, dz = ci.z - cj.z;
                d2[u] = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
                far[u] = d2[u] >= m.far2;
            }
            // far pairs take the clamped value from the compact array (coalesced in j), near pairs gather their row
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int j = j0 + 32 * u;
                v[u] = 0.0f; g[u] = make_float2(0.0f, 0.0f); f[u] = 0.0f;
                if (j < m.L) {
                    if (far[u]) v[u] = __ldg(m.Elast + rb + j);
                    else {
                        int b;
                        lerp_coords(d2[u], m.t0, m.inv_delta, m.tmax, m.nb, b, f[u]);
                        g[u] = __ldg(m.Epk + (size_t)(rb + j) * m.nb + b);
                    }
                }
            }
#pragma unroll
            for (int u = 0; u < U; ++u) e += (double)(far[u] ? v[u] : fmaf(f[u], g[u].y, g[u].x));
        }
    }
    e = warp_sum(e);
    if (lane == 0) red[warp] = e;
    team_bar(bar_id, nwarps * 32);
    double tot = 0.0;
    for (int w = 0; w < nwarps; ++w) tot += red[w];
    team_bar(bar_id, nwarps * 32);
    return tot;
}

// SG: global proposals too are evaluated speculatively, one warp per step (separate instantiations, so that neither
// carries the other's pair loop in its register budget)
// RING: the local phase reads its rows from the shared-memory ring (a.ring_cols > 0) or gathers them from L2.
// CB64: the fp64 C-betas are kept in shared memory (a.cb64) or rebuilt from N, CA, C.
template <bool SG, bool RING, bool CB64>
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
    const int span = min(2 * a.window, L - 1);            // largest j - i of an in-window pair
    constexpr bool use_ring = RING;

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
        int s = 0;                                          // ring slot of the next column
        for (long long t = a.sweep_offset; t < a.sweep_offset + a.n_sweeps; ++t) {
            if (sweep_is_global(t)) continue;
            for (int j = 0; j < L; ++j) {
                const long long q = q0 + j;
                if (lane == 0) {                            // slot s is free once every team has passed column q - R
                    for (;;) {
                        long long mn = 0x7fffffffffffffffLL;
                        for (int g = 0; g < nvalid; ++g) mn = min(mn, prog[g]);
                        if (q - R < mn) break;
                        __nanosleep(200);
                    }
                    const int i_lo = max(0, j - span), i_hi = j - m.min_sep;
                    const int nrows = i_hi - i_lo + 1;
                    void *bar = &full_bar[s];
                    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // the teams' reads of the old column come first
                    if (nrows > 0) mbar_expect_tx(bar, (uint32_t)nrows * row_bytes);
                    else mbar_arrive(bar);
                    // one lane issues the copies of the column: the operands of a bulk copy live in uniform registers
                    for (int i = i_lo; i <= i_hi; ++i)
                        tma_bulk_g2s(ring + ((size_t)s * a.ring_rows + (i - j + span)) * m.row_stride,
                                     m.Epl + (size_t)tri_row(i, j, L) * m.row_stride, row_bytes, bar);
                }
                __syncwarp();
                if (++s == R) s = 0;
            }
            q0 += L;
        }
        return;
    }
    if (slot >= nvalid) return;

    // ================= team: one chain =====================================================================
    unsigned char *cbase = smem_raw + chains_off + (size_t)slot * chain_smem_bytes(L, a.cb64);
    constexpr bool cb64 = CB64;
    const int na = cb64 ? 4 : 3;                            // atoms per residue kept in fp64
    double *X = reinterpret_cast<double *>(cbase), *Y = X + na * L, *Z = Y + na * L;
    double *red = Z + na * L + (cb64 ? 0 : (L & 1)), *b_cd = red + kMaxWarps, *b_sd = b_cd + kDrawBatch, *b_lu = b_sd + kDrawBatch;
    double *rot_s = b_lu + kDrawBatch, *sp_dE = rot_s + 12 * kMaxSpec;
    float4 *cb4 = reinterpret_cast<float4 *>(sp_dE + kMaxSpec);
    float4 *blk4 = cb4 + L;
    float *s = reinterpret_cast<float *>(blk4 + (L + kBlk - 1) / kBlk);
    float *b_sp = s + n;
    int *sp_acc = reinterpret_cast<int *>(b_sp + kDrawBatch);

    const long long row = row0 + slot;
    const unsigned long long chain = (unsigned long long)(a.chain_offset + row);

    for (int q = tid; q < n; q += nthreads) s[q] = a.states[row * n + q];
    team_bar(bar_id, nthreads);
    if (warp == 0)
        nerf_build_warp(m, s, lane, [&](int res, int at, double x, double y, double z) {
            if (at == 3) cb4[res] = make_float4((float)x, (float)y, (float)z, 0.0f);
            if (at < na) { const int f = at * L + res; X[f] = x; Y[f] = y; Z[f] = z; }
        });
    team_bar(bar_id, nthreads);

    double best = INFINITY, e_end = 0.0;
    unsigned long long acc_l = 0, acc_g = 0;
    // exact-decision guard: the bound on the fp32 error of dE grows with the size of the coordinates (their fp32 rounding)
    double ext_scale = fmax(1.0, (double)team_extent(cb4, L, red, tid, nthreads, warp, nwarps, lane, bar_id) * (1.0 / 32.0));
    // local proposals are evaluated by groups of gl lanes, 32 / gl groups per warp
    const int gshift = a.lanes_per_step == 8 ? 3 : (a.lanes_per_step == 16 ? 4 : 5);
    const int gl = 1 << gshift, gpw = 32 >> gshift;
    const int grp = lane >> gshift, glane = lane & (gl - 1);
    int nspec = max(1, min(min(nwarps * gpw, kMaxSpec), a.spec_local > 0 ? a.spec_local : kMaxSpec));
    // a pass may not reach beyond what the ring can hold next to the window (else the team would wait for a column
    // whose slot it still occupies itself)
    if (use_ring) nspec = max(1, min(nspec, 2 * (R - min(a.window, L - 1) - 2) - 1));
    const int draw_warp_u = nwarps > 1 ? 1 : 0;              // the warp that draws the uniforms of the accept test
    long long q0 = 0;                                        // running column number of j = 0 (local sweeps)
    int seen_slot = R - 1;                                   // ring slot and phase parity of the last column waited for
    uint32_t seen_par = 1;
    RowSource rs;
    rs.ring = use_ring ? ring : nullptr; rs.ring_cols = R; rs.ring_rows = a.ring_rows; rs.span = span; rs.slot0 = 0;

    // the bond the torsion k turns about: phi_c N->CA, psi_c CA->C
    auto step_rot = [&](int k, int bi) -> Rot {
        const int fa = (k & 1) * L + (k >> 1), fb = fa + L;
        return rot_about(X[fa], Y[fa], Z[fa], X[fb], Y[fb], Z[fb], b_cd[bi], b_sd[bi], (k & 1) ? m.inv_len_ca_c : m.inv_len_n_ca);
    };
    // the accepted rotation moves every atom bonded after the turned bond: phi_c moves C_c, CB_c and all later
    // residues; psi_c moves the residues after c (R19)
    auto commit = [&](const Rot &R_, int k) {
        const int c = k >> 1;
        // a thread takes a residue: turns those of its backbone atoms that move, then rebuilds its C-beta from them
        for (int res = c + ((k & 1) ? 1 : 0) + tid; res < L; res += nthreads) {
#pragma unroll
            for (int at = 0; at < 3; ++at) {
                if (res == c && at < 2) continue;            // phi_c: N_c and CA_c are the axis
                const int f = at * L + res;
                double x, y, z;
                rot_apply(R_, X[f], Y[f], Z[f], x, y, z);
                X[f] = x; Y[f] = y; Z[f] = z;
            }
            double x, y, z;
            if (cb64 && (res > c || (k & 1) == 0)) {         // the stored C-beta turns with its residue
                const int f = 3 * L + res;
                rot_apply(R_, X[f], Y[f], Z[f], x, y, z);
                X[f] = x; Y[f] = y; Z[f] = z;
            } else {
                cb_point(m, X, Y, Z, L, res, x, y, z);
            }
            cb4[res] = make_float4((float)x, (float)y, (float)z, 0.0f);
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
        double sigma_t = a.sigma_start;                      // Gaussian mode: linear in the sweep index
        if (!(a.sigma_start == a.sigma_end || a.ramp_sigma <= 1 || t <= 0))
            sigma_t = (t >= a.ramp_sigma - 1) ? a.sigma_end
                                              : a.sigma_start + (a.sigma_end - a.sigma_start) * ((double)t / (double)(a.ramp_sigma - 1));
        int seen_rel = -1;                                   // last column of this sweep the team has waited for
        const int slot_j0 = (seen_slot + 1 == R) ? 0 : seen_slot + 1;   // ring slot of column 0 of this sweep

        if (is_global) {                                     // the local sweeps moved everything: fresh culling blocks
            team_blocks(m, cb4, blk4, 0, tid, nthreads);
            team_bar(bar_id, nthreads);
        }
        int k = 0, batch_start = 0, batch_end = 0;
        while (k < n) {
            // ---- a1/a2: draws of the next 64 steps, two per lane (R5-R7) ----------------------------------
            if (k >= batch_end) {
                batch_start = k; batch_end = min(n, k + kDrawBatch);
                if (warp == 0 || warp == draw_warp_u) {
#pragma unroll 1
                    for (int bi = lane; bi < kDrawBatch; bi += 32) {
                        const int kk = k + bi;
                        if (kk >= n) break;
                        const unsigned long long step = (unsigned long long)t * (unsigned long long)n + (unsigned long long)kk;
                        if (warp == 0) {
                            uint32_t x1;
                            const uint32_t x0 = draw01(a.seed, chain, step, PURPOSE_PROPOSAL, x1);
                            float sp;
                            if (a.prop_mode == 2) {
                                // the paper's Gaussian flip: Box-Muller in fp64, wrapped to [-pi, pi)
                                const double u1 = ((double)(x0 >> 8) + 1.0) * 5.9604644775390625e-08;
                                const double u2 = (double)(x1 >> 8) * 5.9604644775390625e-08;
                                const double z = sqrt(-2.0 * log(u1)) * cos(6.283185307179586 * u2);
                                double v = (double)s[kk] + sigma_t * z;
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
                            sincos((double)sp - (double)s[kk], &sd, &cd);
                            b_sp[bi] = sp; b_cd[bi] = cd; b_sd[bi] = sd;
                        }
                        if (warp == draw_warp_u) {
                            const uint32_t x0 = draw0(a.seed, chain, step, PURPOSE_ACCEPT);
                            b_lu[bi] = log((double)((x0 >> 8) + 1u) * 5.9604644775390625e-08);
                        }
                    }
                }
                team_bar(bar_id, nthreads);
            }
            if (is_global && !SG) {
                // ======== one proposal, evaluated by the whole team ========================================
                const int bi = k - batch_start;
                const int split = (k >> 1) + (k & 1);
                const bool inert = (k == 0) || (k == n - 1);
                double dE = 0.0;
                if (!inert) {
                    // ---- a3/a5/a6: turn the right-hand side about the flipped bond, cross pairs, reduction ------
                    double acc;
                    {
                        const Rot Rk = step_rot(k, bi);
                        if (tid == 0) {                       // kept in shared memory for the commit, not in registers
#pragma unroll
                            for (int q = 0; q < 9; ++q) rot_s[q] = Rk.r[q];
#pragma unroll
                            for (int q = 0; q < 3; ++q) rot_s[9 + q] = Rk.t[q];
                        }
                        acc = warp_sum(cross_pairs_dE<false, true>(m, rs, cb4, blk4, X, Y, Z, cb64, Rk, 0, split, L - 1, tid, nthreads));
                    }
                    if (lane == 0) red[warp] = acc;
                    team_bar(bar_id, nthreads);
                    for (int w = 0; w < nwarps; ++w) dE += red[w];
                }
                // ---- a7: Metropolis test, accept iff log u <= -dE / T   (Eq. 1a, R14) ---------------------
                // exact-decision guard (R24): a gap inside the fp32 error bound of dE is decided by the fp64 path
                bool exact = false;
                if (!inert && fabs(b_lu[bi] + dE * invT) < a.guard_global * ext_scale * invT) {
                    team_bar(bar_id, nthreads);                      // every thread has read red[]
                    dE = team_sum(exact_dE_partial(m, X, Y, Z, cb64 ? 1 : 0, k, b_cd[bi], b_sd[bi], 0, L - 1, tid, nthreads),
                                  red, warp, nwarps, lane, bar_id);
                    exact = true;
                }
                const bool accept = exact ? (b_lu[bi] <= -dE / T) : (b_lu[bi] <= -dE * invT);
                if (tid == 0) {
                    const long long q = (t - a.sweep_offset) * n + k;
                    if (q < a.trace_steps) {
                        const size_t z = (size_t)row * a.trace_steps + q;
                        if (a.trace_prop) a.trace_prop[z] = b_sp[bi];
                        if (a.trace_dE) a.trace_dE[z] = dE;
                        if (a.trace_acc) a.trace_acc[z] = (accept ? 1 : 0) | (exact ? 2 : 0);
                    }
                }
                if (accept) {
                    ++acc_g;
                    if (tid == 0) s[k] = b_sp[bi];
                    if (!inert) {
                        Rot Rc;
#pragma unroll
                        for (int q = 0; q < 9; ++q) Rc.r[q] = rot_s[q];
#pragma unroll
                        for (int q = 0; q < 3; ++q) Rc.t[q] = rot_s[9 + q];
                        commit(Rc, k);
                        team_bar(bar_id, nthreads);
                        team_blocks(m, cb4, blk4, (k >> 1) / kBlk, tid, nthreads);
                    }
                }
                team_bar(bar_id, nthreads);
                ++k;
            } else {
                // ======== up to nspec proposals, group r evaluating step k + r against the current state ===
                // (a global sweep in speculative mode: the groups are whole warps and the pairs are all straddling ones)
                const bool gp = SG && is_global;
                const int gl_x = gp ? 32 : gl, gpw_x = gp ? 1 : gpw;
                const int grp_x = gp ? 0 : grp, glane_x = gp ? lane : glane;
                const int S = min(gp ? min(nwarps, kMaxSpec) : nspec, batch_end - k);
                if (use_ring && !gp) {
                    // columns left of the window centre are dead for this chain; wait for the ones the pass needs
                    if (tid == 0) prog[slot] = q0 + (k >> 1);
                    const int need = min(L - 1, ((k + S - 1) >> 1) + a.window);
                    while (seen_rel < need) {
                        ++seen_rel;
                        if (++seen_slot == R) { seen_slot = 0; seen_par ^= 1u; }
                        mbar_wait(&full_bar[seen_slot], seen_par);
                    }
                }
                const int r = warp * gpw_x + grp_x;
                const bool active = r < S;
                const int kk = k + r, bi = kk - batch_start;
                const bool inert = (kk == 0) || (kk == n - 1);
                double dE = 0.0;
                Rot Rk;
                if (active && !inert) {
                    const int c = kk >> 1, split = c + (kk & 1);
                    Rk = step_rot(kk, bi);
                    const int ilo = gp ? 0 : max(0, c - a.window), jhi = gp ? L - 1 : min(L - 1, c + a.window);
                    // ---- a4/a5: in-window cross pairs (Eq. 3b), or all of them (Eq. 3a) ------------------------
                    if (gp) {
                        dE = cross_pairs_dE<false, true>(m, rs, cb4, blk4, X, Y, Z, cb64, Rk, 0, split, L - 1, lane, 32);
                    } else {
                        if (RING) {
                            rs.slot0 = slot_j0 + split;
                            if (rs.slot0 >= R) rs.slot0 %= R;
                        }
                        dE = cross_pairs_dE<RING, false>(m, rs, cb4, blk4, X, Y, Z, cb64, Rk, ilo, split, jhi, glane_x, gl_x);
                    }
                }
                // ---- a6: reduction over the group's lanes (every lane of the warp takes part) ----------------
                for (int d = gl_x >> 1; d > 0; d >>= 1) dE += __shfl_xor_sync(0xffffffffu, dE, d);
                if (active && glane_x == 0) {
                    sp_dE[r] = dE;
                    const double gd = (gp ? a.guard_global : a.guard_local) * ext_scale * invT;
                    // Eq. 2a, R14; 2 = the gap is inside the fp32 error bound of dE: decided below by the fp64 path (R24)
                    sp_acc[r] = (!inert && fabs(b_lu[bi] + dE * invT) < gd) ? 2 : ((b_lu[bi] <= -dE * invT) ? 1 : 0);
                    if (!inert) {
#pragma unroll
                        for (int q = 0; q < 9; ++q) rot_s[12 * r + q] = Rk.r[q];
#pragma unroll
                        for (int q = 0; q < 3; ++q) rot_s[12 * r + 9 + q] = Rk.t[q];
                    }
                }
                team_bar(bar_id, nthreads);
                int rsel = 0;                                 // first accepted step of the pass
                bool any_exact = false;
                while (rsel < S) {
                    int f = sp_acc[rsel];                     // the same value in every thread of the team
                    if (f == 2) {
                        const int kx = k + rsel, bx = kx - batch_start, cx = kx >> 1;
                        const double dx = team_sum(exact_dE_partial(m, X, Y, Z, cb64 ? 1 : 0, kx, b_cd[bx], b_sd[bx],
                                                                    gp ? 0 : max(0, cx - a.window), gp ? L - 1 : min(L - 1, cx + a.window),
                                                                    tid, nthreads), red, warp, nwarps, lane, bar_id);
                        f = 2 | ((b_lu[bx] <= -dx / T) ? 1 : 0);
                        if (tid == 0) { sp_dE[rsel] = dx; sp_acc[rsel] = f; }   // after team_sum's barriers: every thread has read the 2
                        any_exact = true;
                    }
                    if (f & 1) break;
                    ++rsel;
                }
                if (any_exact) team_bar(bar_id, nthreads);    // the rewritten entries are read by the tracing threads
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
                    if (gp) ++acc_g; else ++acc_l;
                    if (tid == 0) s[kc] = b_sp[kc - batch_start];
                    if (kc != 0 && kc != n - 1) {
                        Rot Rc;
#pragma unroll
                        for (int q = 0; q < 9; ++q) Rc.r[q] = rot_s[12 * rsel + q];
#pragma unroll
                        for (int q = 0; q < 3; ++q) Rc.t[q] = rot_s[12 * rsel + 9 + q];
                        commit(Rc, kc);
                        if (gp) {
                            team_bar(bar_id, nthreads);
                            team_blocks(m, cb4, blk4, (kc >> 1) / kBlk, tid, nthreads);
                        }
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
        e_end = team_full_energy(m, cb4, red, warp, nwarps, lane, bar_id);
        ext_scale = fmax(1.0, (double)team_extent(cb4, L, red, tid, nthreads, warp, nwarps, lane, bar_id) * (1.0 / 32.0));
        if (e_end < best) {
            best = e_end;
            if (a.best_state)
                for (int q = tid; q < n; q += nthreads) a.best_state[row * n + q] = s[q];
        }
        if (tid == 0 && a.first_hit && (float)e_end <= a.energy_threshold) atomicMin(a.first_hit, (unsigned long long)t);
    }
    if (a.n_sweeps == 0) e_end = team_full_energy(m, cb4, red, warp, nwarps, lane, bar_id);
    for (int q = tid; q < n; q += nthreads) a.states[row * n + q] = s[q];
    if (tid == 0) {
        if (a.energy) a.energy[row] = (float)e_end;
        if (a.best_energy) a.best_energy[row] = (float)best;
        if (a.n_accept_local) a.n_accept_local[row] = acc_l;
        if (a.n_accept_global) a.n_accept_global[row] = acc_g;
    }
}

}  // namespace amh
