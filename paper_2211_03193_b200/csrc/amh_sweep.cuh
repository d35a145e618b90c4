// amh_sweep.cuh - the alternating MH sweep kernel (rows a1-a9 of DESIGN.md section 0), sm_100a.
//
// Launch shape.  One CTA runs C chains; each chain owns W consecutive warps (its "team") and a named
// barrier; one more warp (the last) is the PRODUCER that feeds the table ring by TMA bulk copies.
// Chains are independent: teams never wait for one another except through the ring.
//
// What a proposal costs.  dE = S_new - S_old, both sums over the pairs that straddle the
// flipped bond (all of them in a global sweep, Eq. 1/3a; the in-window ones in a local sweep, Eq. 2/3b), of the
// EXCESS pair energy e'_ij(d) = e_ij(d) - e_ij(infinity) (0 beyond the last bin centre, so far pairs drop out of
// both sums exactly).  Only S_new is evaluated pair by pair.  S_old is carried from step to step: when the step
// index advances, the set of straddling pairs changes by one row and one column (O(w) or O(L) pairs, the
// "transition" T(k)); when a proposal is accepted, S_old becomes that proposal's S_new.
//
// Local sweeps: a proposal has only ~70-150 pairs and Alg. 1 orders the proposals of a chain strictly
// (PAPER.md:105, 114).
//   * Speculation.  The draws are counter-based (R6), so the proposals of steps k, k+1, ... are known in
//     advance: GROUP r (8, 16 or 32 lanes; up to 16 groups per team) evaluates step k+r AGAINST THE
//     CURRENT STATE, and the results are consumed in order up to and including the first accepted step;
//     later results were computed against a state that no longer exists and are thrown away (their steps
//     are evaluated again in the next pass).  The trajectory is exactly the sequential one.
//   * A group first turns the <= w+1 C-betas right of its bond (fp64, rounded once) into shared memory, then
//     deals the nI x nJ pairs of the step evenly to its lanes (pair p = lane, lane + gl, ...).
//   * Table ring.  Every chain of the CTA walks k = 0..n-1, so they all need the same table rows at about
//     the same time: pair (i, j) is needed while the window centre c is in [max(i, j-w), min(j, i+w)].
//     The producer streams "column" j = the rows (i, j), j-2w <= i <= j-min_sep, into slot q mod R of a
//     shared-memory ring (q = a running column number) with cp.async.bulk + mbarrier complete_tx; teams
//     wait on the slot's "full" barrier, read from shared memory, and arrive on the slot's "empty" barrier
//     once the column is dead for them; the producer refills a slot when every team has arrived.
//
// Global sweeps: O(L^2/6) straddling pairs per proposal, evaluated either by the whole team one proposal at a
// time (SG = false) or speculatively, one warp per step (SG = true).  A thread owns a column j: it turns CB_j
// itself and walks the rows i in blocks of 8; a block whose bounding sphere is beyond the last bin centre of
// the new CB_j is skipped whole, far pairs are skipped one by one, near pairs gather 8 bytes from the packed
// table in L2, four rows' gathers in flight at a time.
//
// Exact-decision guard (R24): the sums are fp32; a proposal whose gap |log u + dE/T| is inside the bound on
// their error is evaluated again in fp64 from the fp64 atoms and the probabilities themselves before deciding.
#pragma once
#include "amh_device.cuh"

namespace amh {
// Checked build (-DAMH_CHECK, `python -m paper_2211_03193_b200.build --checked`): every table / ring / shared-memory index the
// pair loops form is range-checked and a violation leaves its code in a device word that amh_check_status() returns.
// (compute-sanitizer is closed on the GPU pool this was developed on; tests/test_gpu_checked.py runs the launch shapes of
// the parity tests through this build instead.)  The product build compiles the checks out.
__device__ int amh_check_word = 0;
#ifdef AMH_CHECK
#define AMH_ASSERT(cond, code) do { if (!(cond)) atomicMax(&amh_check_word, (code)); } while (0)
#else
#define AMH_ASSERT(cond, code) ((void)0)
#endif
#ifndef AMH_UL
#define AMH_UL 3
#endif
#ifndef AMH_UG
#define AMH_UG 4
#endif

struct RunArgs {
    float *states;
    long long B, n_sweeps, sweep_offset, chain_offset;
    int n_global, n_local, window, global_first;
    int local_stride;                    // NEXT-4: 0 = Alg. 1's order; s > 0 = strided order of the local sweeps
    double t_start, t_end;
    long long ramp_sweeps;
    const float *per_chain_T;
    int prop_mode, grid;
    double sigma_start, sigma_end;       // Gaussian mode: linear ramp over ramp_sigma sweeps
    long long ramp_sigma;
    // launch shape
    int C, W;                            // chains per CTA, warps per chain
    int nspec;                           // local proposals evaluated per pass (<= W * 32 / lanes_per_step, <= 16)
    int lanes_per_step;                  // lanes that share one local proposal: 32, 16 or 8
    int ring_cols;                       // R: slots of the table ring (> window + 2), 0 = gather from L2 instead
    int ring_rows;                       // rows per column: 2w - min_sep + 1
    int wpts;                            // C-betas a local proposal turns, at most: min(window, L-1) + 1
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
constexpr int kMaxSpec = 16;             // proposals evaluated per pass, at most
constexpr int kBlk = 8;                  // residues per culling block of the global phase
constexpr int kSup = 4;                  // blocks per super-block (second culling level)
constexpr int kMaxTeamWarps = 15;        // team warps per CTA: chains x warps per chain (+ the producer = 512 threads)
constexpr int kMaxChains = 15;           // chains per CTA (named barriers 1..15)
constexpr int kSweepMaxThreads = 512;    // 15 team warps + the producer: 128 registers per thread
constexpr int kRingPadRows = 4;          // rows in front of the first ring slot that masked-off evaluations (j - i < min_sep) may touch

// shared memory of one chain, in bytes (a multiple of 16):
//   double X[aL], Y[aL], Z[aL]   atoms, index atom * L + res (atom 0..2 = N, CA, C; a = 3).  The C-beta is a fixed
//                                combination of the three (cb_point); it is kept in fp64 too (atom 3, a = 4) when
//                                that does not cost a resident chain (cb64), else rebuilt where needed
//   double red[32], b_cd[64], b_sd[64], b_lu[64], rot_s[16][12], sp_new[16], sp_T[16]
//   float4 cb4[L]                fp32 copy of the C-betas (what the pair loops read); .w = byte offset of the
//                                residue's term in a table address (as the ROW index i of a pair)
//   float4 blk4[ceil(L/8) + ceil(L/32)]   bounding spheres of the 8-residue blocks, then of the 32-residue super-blocks
//                                (two-level culling in the global phase)
//   float4 cbn[nspec][wpts]      the turned C-betas of the local proposals of a pass; .w = the column's term
//   float  s[n], b_sp[64];  int ctr[4]  (chunk counter of the whole-team global proposals)
__host__ __device__ inline size_t chain_smem_bytes(int L, int cb64, int nspec, int wpts, int W)
{
    size_t doubles = (cb64 ? 12 : 9) * (size_t)L;
    doubles += doubles & 1;                                  // float4 arrays on 16 bytes
    doubles += 2 * kMaxWarps + 3 * kDrawBatch + 12 * kMaxSpec + 2 * kMaxSpec;
    const size_t nblk = ((size_t)L + kBlk - 1) / kBlk;
    size_t floats = 4 * (size_t)L + 4 * (nblk + (nblk + kSup - 1) / kSup) + 4 * (size_t)nspec * wpts + 2 * (size_t)L + kDrawBatch + 4;
    floats = (floats + 3) & ~(size_t)3;
    return sizeof(double) * doubles + sizeof(float) * floats;
}

// header: full barriers [R], empty barriers [R]; then the ring; then the chains
__host__ __device__ inline size_t sweep_header_bytes(int ring_cols) { return (16 * (size_t)ring_cols + 15) & ~(size_t)15; }

__host__ __device__ inline size_t ring_bytes(int ring_cols, int ring_rows, int row_stride)
{
    if (ring_cols <= 0) return 0;
    return (sizeof(float) * ((size_t)ring_cols * ring_rows + kRingPadRows) * row_stride + 15) & ~(size_t)15;
}

__host__ __device__ inline size_t sweep_smem_bytes(int L, int C, int W, int ring_cols, int ring_rows, int row_stride, int cb64, int nspec, int wpts)
{
    return sweep_header_bytes(ring_cols) + ring_bytes(ring_cols, ring_rows, row_stride) + (size_t)C * chain_smem_bytes(L, cb64, nspec, wpts, W);
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
// arrive (release at CTA scope: the caller's earlier reads of the slot are ordered before it)
__device__ __forceinline__ void mbar_arrive(void *bar)
{
    asm volatile("mbarrier.arrive.release.cta.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait_u32(uint32_t a, uint32_t parity)
{
    uint32_t ok;
    do {
        // the last operand lets the hardware park the thread for up to ~1 us instead of spinning on the barrier
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.acquire.cta.shared::cta.b64 p, [%1], %2, %3;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(a), "r"(parity), "r"(1000u) : "memory");
    } while (!ok);
}
__device__ __forceinline__ void mbar_wait(void *bar, uint32_t parity) { mbar_wait_u32(smem_u32(bar), parity); }
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
template <class Model>
__device__ __forceinline__ void cb_point(const Model &m, const double *X, const double *Y, const double *Z, int L, int res,
                                         double &x, double &y, double &z)
{
    const double ax = X[L + res], ay = Y[L + res], az = Z[L + res];                                  // CA
    const double ex = (ax - X[res]) * m.inv_len_n_ca, ey = (ay - Y[res]) * m.inv_len_n_ca, ez = (az - Z[res]) * m.inv_len_n_ca;
    const double vx = X[2 * L + res] - ax, vy = Y[2 * L + res] - ay, vz = Z[2 * L + res] - az;        // C - CA
    x = fma(m.cbC, fma(ey, vz, -ez * vy), fma(m.cbB, vx, fma(m.cbA, ex, ax)));
    y = fma(m.cbC, fma(ez, vx, -ex * vz), fma(m.cbB, vy, fma(m.cbA, ey, ay)));
    z = fma(m.cbC, fma(ex, vy, -ey * vx), fma(m.cbB, vz, fma(m.cbA, ez, az)));
}

// bin index b and fraction f of R8's interpolation at squared distance d2: t = (d - c0) / delta clamped to
// [0, nb-1], b <= t <= b + 1, b <= nb - 2, f = t - b.
//   d = sqrt.approx.ftz.f32(d2): one MUFU instruction, maximum relative error 2^-23 (PTX ISA); d2 = 0 (or a
//   subnormal: coincident atoms) gives 0.
//   b = round-to-nearest-even(t - 1/2), read off the low mantissa bits of (t - 1/2) + 1.5 * 2^23: conversion
//   instructions (F2I, I2F) run at the MUFU rate on sm_100 (16 per clock and SM, measured), these are plain FADDs.
//   At an integer t either neighbour bin gives the same value (the interpolant is continuous), and
//   min(t - 1/2, nb - 1.75) keeps b <= nb - 2.
__device__ __forceinline__ void bin_frac(float d2, float t0, float inv_delta, float tmax, float thmax, int &b, float &f)
{
    float d;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(d) : "f"(d2));
    float t = fmaf(d, inv_delta, t0);                        // (d - c0) / delta with t0 = -c0 / delta: one fma
    t = fminf(fmaxf(t, 0.0f), tmax);
    const float u = __fadd_rn(fminf(__fadd_rn(t, -0.5f), thmax), 12582912.0f);
    f = __fadd_rn(t, -__fadd_rn(u, -12582912.0f));
    b = __float_as_int(u) & 0x3fffff;
}

// floor(a / b) for 0 <= a < 2^16, 1 <= b < 2^10 without the integer-division sequence
__device__ __forceinline__ int small_div(int a, int b)
{
    return __float2int_rd(__fdividef((float)a + 0.5f, (float)b));
}

// row index of the pair i < j in 32 bits (L < 46341)
__device__ __forceinline__ int tri_row(int i, int j, int L) { return (i * (2 * L - i - 1)) / 2 - i - 1 + j; }

// ---- local phase: tables addressed as base + rowterm(i) + colterm(j) + bin ----------------------------------
// RING: rows of plain E' in the shared-memory ring, row j - i - min_sep of slot(j): rowterm = -i * row_stride * 4,
// colterm = ((slot(j) * ring_rows + j - min_sep) * row_stride) * 4.
// else: packed {E', dE'} in L2: rowterm = tri_base(i) * nb * 8, colterm = j * nb * 8.
struct LocalTab {
    const unsigned char *base;
    int ring_cols, ring_rows, min_sep, stride4;              // stride4 = row_stride * 4 (RING)
    int slot_c, c_ref;                                       // ring slot of column c_ref (RING)
    int nb8;                                                 // nb * 8 (L2)
    long long lo, hi;                                        // checked build: valid byte offsets from base are [lo, hi)
};

template <bool RING>
__device__ __forceinline__ int col_term(const LocalTab &tb, int j)
{
    if (RING) {
        int s = tb.slot_c + (j - tb.c_ref);                  // 0 <= j - c_ref < ring_cols: one wrap at most
        if (s >= tb.ring_cols) s -= tb.ring_cols;
        return (s * tb.ring_rows + j - tb.min_sep) * tb.stride4;
    }
    return j * tb.nb8;
}

// excess energy e'_ij of one pair from its two points; ci.w / pj.w carry the row / column terms of the address
template <bool RING>
__device__ __forceinline__ float local_pair(const DevModel &m, const LocalTab &tb, const float4 ci, const float4 pj)
{
    const float dx = ci.x - pj.x, dy = ci.y - pj.y, dz = ci.z - pj.z;
    const float d2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
    int b;
    float f;
    bin_frac(d2, m.t0, m.inv_delta, m.tmax, m.thmax, b, f);
    const unsigned char *row = tb.base + (__float_as_int(ci.w) + __float_as_int(pj.w));
    AMH_ASSERT(b >= 0 && b <= m.nb - 2, 1);
    AMH_ASSERT((long long)(__float_as_int(ci.w) + __float_as_int(pj.w)) + (long long)b * (RING ? 4 : 8) >= tb.lo &&
               (long long)(__float_as_int(ci.w) + __float_as_int(pj.w)) + (long long)(b + 1) * (RING ? 4 : 8) + (RING ? 4 : 0) <= tb.hi, 2);
    if (RING) {
        const float *r = reinterpret_cast<const float *>(row) + b;
        const float e0 = r[0], e1 = r[1];
        return fmaf(f, e1 - e0, e0);
    } else {
        const float2 v = __ldg(reinterpret_cast<const float2 *>(row) + b);
        return fmaf(f, v.y, v.x);
    }
}

// S_new of a local proposal: sum of e' over the pairs (i, j), ilo <= i < split <= j <= jhi, j - i >= min_sep, with the
// turned C-betas cbn[j - split].  The nI x nJ pairs are dealt to the gl lanes of the group: pair p = glane + t * gl,
// i = ilo + p / nJ, j = split + p % nJ.  Returns this lane's partial sum.
template <bool RING>
__device__ __forceinline__ float local_new_sum(const DevModel &m, const LocalTab &tb, const float4 *cb4, const float4 *cbn,
                                               int ilo, int split, int nI, int nJ, int glane, int gl)
{
    constexpr int U = AMH_UL;
    const int nP = nI * nJ;
    float acc[U];
#pragma unroll
    for (int u = 0; u < U; ++u) acc[u] = 0.0f;
    if (nP <= 0) return 0.0f;
    // p / nJ by a 32-bit reciprocal (one IMAD.HI per pair instead of carrying (i, j) along): exact for p * nJ < 2^32
    const unsigned rcp = 0xffffffffu / (unsigned)nJ + 1u;
    const bool one_col = nJ == 1;                            // 2^32 / 1 does not fit
    const int dsep = split - ilo - m.min_sep;                // valid iff ju - iu + dsep >= 0
    for (int p = glane; p < nP; p += U * gl) {
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int q = p + u * gl;
            const bool in = q < nP;
            const int qq = in ? q : 0;
            const int iu = one_col ? qq : (int)__umulhi((unsigned)qq, rcp), ju = qq - iu * nJ;
            AMH_ASSERT(ilo + iu >= 0 && ilo + iu < m.L && ju >= 0 && ju < nJ && iu < nI, 3);
            const float4 ci = cb4[ilo + iu];
            const float4 pj = cbn[ju];
            const bool valid = in && ju - iu + dsep >= 0;
            const float e = local_pair<RING>(m, tb, ci, pj);
            acc[u] += valid ? e : 0.0f;
        }
    }
    float s = acc[0];
#pragma unroll
    for (int u = 1; u < U; ++u) s += acc[u];
    return s;
}

// T(k) = S_old(k) - S_old(k - 1) for the CURRENT state: the straddling set of step k minus that of step k - 1
// (DESIGN.md section 7 "Transitions").  w >= L - 1 makes the window the whole chain (global sweeps).
//   k odd  (c = k >> 1): the split moves from c to c + 1: column c leaves (rows lo..c - ms), row c enters (columns c + ms..hi)
//   k even (c >= 1):     the window moves from c - 1 to c: row c - 1 - w leaves (columns c..c - 1 + w), column c + w enters
// Each is a line of pairs (i0 + t * di, j0 + t * dj), t < count.
struct Line { int i0, j0, di, dj, cnt; };

__device__ __forceinline__ void transition_lines(int k, int L, int w, int ms, Line &leave, Line &enter)
{
    const int c = k >> 1;
    leave.cnt = 0; leave.i0 = leave.j0 = leave.di = leave.dj = 0;
    enter = leave;
    if (k <= 0) return;
    if (k & 1) {
        const int lo = max(0, c - w), hi = min(L - 1, c + w);
        leave.i0 = lo; leave.j0 = c; leave.di = 1; leave.dj = 0; leave.cnt = max(0, c - ms - lo + 1);
        enter.i0 = c; enter.j0 = c + ms; enter.di = 0; enter.dj = 1; enter.cnt = max(0, hi - c - ms + 1);
    } else {
        const int il = c - 1 - w;
        if (il >= 0) {
            const int j0 = max(c, il + ms), j1 = min(L - 1, c - 1 + w);
            leave.i0 = il; leave.j0 = j0; leave.di = 0; leave.dj = 1; leave.cnt = max(0, j1 - j0 + 1);
        }
        const int je = c + w;
        if (je <= L - 1) {
            const int i0 = max(0, c - w), i1 = min(c - 1, je - ms);
            enter.i0 = i0; enter.j0 = je; enter.di = 1; enter.dj = 0; enter.cnt = max(0, i1 - i0 + 1);
        }
    }
}

template <bool RING>
__device__ __forceinline__ float local_transition(const DevModel &m, const LocalTab &tb, const float4 *cb4, int k, int w,
                                                  int glane, int gl)
{
    Line lv, en;
    transition_lines(k, m.L, w, m.min_sep, lv, en);
    float acc0 = 0.0f, acc1 = 0.0f;
    const int tot = lv.cnt + en.cnt;
    // two pairs per lane and trip (the two lines hold 2 (w + 1) pairs at most, i.e. two trips of a group of 8)
    for (int q0 = glane; q0 < tot; q0 += 2 * gl) {
        float e[2];
        bool isl[2], in[2];
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            const int q = q0 + u * gl;
            in[u] = q < tot;
            const int qq = in[u] ? q : q0;
            isl[u] = qq < lv.cnt;
            const int t = isl[u] ? qq : qq - lv.cnt;
            const int i = isl[u] ? lv.i0 + t * lv.di : en.i0 + t * en.di;
            const int j = isl[u] ? lv.j0 + t * lv.dj : en.j0 + t * en.dj;
            AMH_ASSERT(i >= 0 && i < j && j < m.L && j - i >= m.min_sep, 4);
            const float4 ci = cb4[i];
            float4 cj = cb4[j];
            cj.w = __int_as_float(col_term<RING>(tb, j));
            e[u] = local_pair<RING>(m, tb, ci, cj);
        }
        acc0 += isl[0] ? -e[0] : e[0];
        acc1 += in[1] ? (isl[1] ? -e[1] : e[1]) : 0.0f;
    }
    return acc0 + acc1;
}

// ---- global phase -------------------------------------------------------------------------------------------
// Sum of e' over the pairs (i, j), i < split, jlo <= j <= jhi, j - i >= min_sep, with CB_j turned by R (turn = true) or
// left where it is (turn = false: a transition line).  Work is dealt to `nthr` threads, this one being `tid`:
// a thread OWNS a column j - it turns CB_j itself (fp64, rounded once to fp32) - and walks the rows i in blocks of kBlk
// residues whose bounding spheres are kept in blk4: a block beyond the last bin centre holds only pairs whose term is
// exactly 0 and is skipped whole.  When a round has fewer columns than threads, S threads share a column and take
// every S-th block.
__device__ __forceinline__ double global_cols_sum(const DevModel &m, const float4 *cb4, const float4 *blk4,
                                                  const double *X, const double *Y, const double *Z, bool cb64, bool turn, const Rot &R,
                                                  int split, int jlo, int jhi, int tid_, int nthr_, int *ctr = nullptr)
{
    const int nJ = jhi - jlo + 1;
    double acc = 0.0;
    if (split <= 0 || nJ <= 0) return acc;
    // ctr (a shared-memory counter, 0 at entry; whole-team calls only): when there are at least as many columns as threads, the
    // team's warps do not take fixed rounds of columns but GRAB chunks of 32 columns as they finish (culling makes the chunks
    // uneven; with fixed rounds the fast warps wait at the reduction).  The sum does not depend on who takes which chunk.
    const bool dyn = ctr != nullptr && nthr_ > 32 && nJ >= nthr_;
    const int nthr = dyn ? 32 : nthr_, tid = dyn ? (tid_ & 31) : tid_;
    for (int c0 = 0;; c0 += dyn ? 0 : nthr) {
        if (dyn) {
            int ch = 0;
            if (tid == 0) ch = atomicAdd(ctr, 1);
            c0 = __shfl_sync(0xffffffffu, ch, 0) * 32;
        }
        if (c0 >= nJ) break;
        const int nc = min(nthr, nJ - c0);
        int S = 1, col = tid, slice = 0;
        if (nc < nthr) {
            S = small_div(nthr, nc); slice = small_div(tid, nc); col = tid - slice * nc;
            if (slice >= S) { if (dyn) continue; else break; }
        }
        const int j = jlo + c0 + col;
        float xn, yn, zn;
        if (turn) {
            double x0, y0, z0, x, y, z;
            if (cb64) { x0 = X[3 * m.L + j]; y0 = Y[3 * m.L + j]; z0 = Z[3 * m.L + j]; }
            else cb_point(m, X, Y, Z, m.L, j, x0, y0, z0);
            rot_apply(R, x0, y0, z0, x, y, z);
            xn = (float)x; yn = (float)y; zn = (float)z;
        } else {
            const float4 o = cb4[j];
            xn = o.x; yn = o.y; zn = o.z;
        }
        const int i_end = min(split - 1, j - m.min_sep);
        const int nblk = i_end < 0 ? 0 : i_end / kBlk + 1;
        const int nblk_all = (m.L + kBlk - 1) / kBlk;
        int b = slice;
        while (b < nblk) {
            // second culling level: a super-block of kSup blocks beyond the last bin centre is skipped whole
            const int sb = b / kSup;
            if (nblk_all > 4 * kSup) {                                      // long chains only: short ones have too few blocks to gain
                const float4 sl = blk4[nblk_all + sb];
                const float dx = sl.x - xn, dy = sl.y - yn, dz = sl.z - zn;
                if (fmaf(dx, dx, fmaf(dy, dy, dz * dz)) >= sl.w) {
                    const int nb0 = (sb + 1) * kSup;                       // this slice's first block at or after nb0
                    b = (S == 1) ? nb0 : slice + small_div(max(nb0 - slice, 0) + S - 1, S) * S;
                    continue;
                }
            }
            const int bend = min(nblk, (sb + 1) * kSup);
            for (; b < bend; b += S) {
            const float4 bl = blk4[b];
            {
                const float dx = bl.x - xn, dy = bl.y - yn, dz = bl.z - zn;
                if (fmaf(dx, dx, fmaf(dy, dy, dz * dz)) >= bl.w) continue;
            }
            // U rows per trip: all distances first, then all gathers, then the sums, so that a thread has U loads in
            // flight instead of stalling on each pair's row (the rows of near pairs come from L2, ~600 cycles away)
            constexpr int U = AMH_UG;
            float part = 0.0f;
#pragma unroll
            for (int t = 0; t < kBlk / U; ++t) {
                const int i = b * kBlk + t * U;
                if (i <= i_end) {
                    float d2[U], f[U];
                    float2 v[U];
                    bool near[U];
#pragma unroll
                    for (int u = 0; u < U; ++u) {
                        const float4 ci = cb4[min(i + u, i_end)];
                        const float dx = ci.x - xn, dy = ci.y - yn, dz = ci.z - zn;
                        d2[u] = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
                        near[u] = (i + u <= i_end) && d2[u] < m.far2;
                    }
#pragma unroll
                    for (int u = 0; u < U; ++u) {
                        v[u] = make_float2(0.0f, 0.0f); f[u] = 0.0f;
                        if (near[u]) {
                            int bn;
                            bin_frac(d2[u], m.t0, m.inv_delta, m.tmax, m.thmax, bn, f[u]);
                            AMH_ASSERT(bn >= 0 && bn <= m.nb - 2 && i + u >= 0 && i + u < j && j < m.L, 5);
                            v[u] = __ldg(m.Epk + (size_t)tri_row(i + u, j, m.L) * m.nb + bn);
                        }
                    }
#pragma unroll
                    for (int u = 0; u < U; ++u) part += fmaf(f[u], v[u].y, v[u].x);
                }
            }
            acc += (double)part;
            }
        }
    }
    return acc;
}

// the column line of a global transition: sum of e' over (i, j), i = 0 .. cnt - 1, at the current positions
__device__ __forceinline__ double global_col_sum(const DevModel &m, const float4 *cb4, int j, int cnt, int tid, int nthr)
{
    double acc = 0.0;
    if (cnt <= 0) return acc;
    const float4 cj = cb4[j];
    for (int i = tid; i < cnt; i += nthr) {
        const float4 ci = cb4[i];
        const float dx = ci.x - cj.x, dy = ci.y - cj.y, dz = ci.z - cj.z;
        const float d2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
        if (d2 < m.far2) {
            int b;
            float f;
            bin_frac(d2, m.t0, m.inv_delta, m.tmax, m.thmax, b, f);
            const float2 v = __ldg(m.Epk + (size_t)tri_row(i, j, m.L) * m.nb + b);
            acc += (double)fmaf(f, v.y, v.x);
        }
    }
    return acc;
}

// the row line of a global transition: sum of e' over (i, j), j = j0 .. j0 + cnt - 1, at the current positions
__device__ __forceinline__ double global_row_sum(const DevModel &m, const float4 *cb4, int i, int j0, int cnt, int tid, int nthr)
{
    double acc = 0.0;
    if (cnt <= 0) return acc;
    const float4 ci = cb4[i];
    const int rb = tri_row(i, 0, m.L);
    for (int q = tid; q < cnt; q += nthr) {
        const int j = j0 + q;
        const float4 cj = cb4[j];
        const float dx = ci.x - cj.x, dy = ci.y - cj.y, dz = ci.z - cj.z;
        const float d2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
        if (d2 < m.far2) {
            int b;
            float f;
            bin_frac(d2, m.t0, m.inv_delta, m.tmax, m.thmax, b, f);
            const float2 v = __ldg(m.Epk + (size_t)(rb + j) * m.nb + b);
            acc += (double)fmaf(f, v.y, v.x);
        }
    }
    return acc;
}

// ---- exact-decision guard (R24) --------------------------------------------------------------
// what the fp64 path needs of the model, passed BY VALUE: a reference to the kernel's DevModel parameter would force
// that whole struct into local memory and turn every m.field of the hot loops into a local load
struct ExactModel {
    const float *P;
    int L, nb, min_sep;
    double c0_d, delta_d, eps_d, far2_d, inv_len_n_ca, inv_len_ca_c, cbA, cbB, cbC;
};
__device__ __forceinline__ ExactModel exact_model(const DevModel &m)
{
    ExactModel e;
    e.P = m.P; e.L = m.L; e.nb = m.nb; e.min_sep = m.min_sep;
    e.c0_d = m.c0_d; e.delta_d = m.delta_d; e.eps_d = m.eps_d; e.far2_d = m.far2_d;
    e.inv_len_n_ca = m.inv_len_n_ca; e.inv_len_ca_c = m.inv_len_ca_c; e.cbA = m.cbA; e.cbB = m.cbB; e.cbC = m.cbC;
    return e;
}

// dE of the proposal at variable k in fp64, every term from the fp64 atoms and from -log(p + eps) itself: this
// thread's share of the sum over (i, j), ilo <= i < split <= j <= jhi, j - i >= min_sep, of e(new) - e(old).
// Pairs beyond the last bin centre before and after contribute exactly 0 (R8's clamp) and are skipped.
__device__ __noinline__ double exact_dE_partial(const ExactModel m, const double *X, const double *Y, const double *Z, int cb64,
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

// two sums at once
__device__ __forceinline__ void team_sum2(double &a, double &b, double *red, int warp, int nwarps, int lane, int bar_id)
{
    a = warp_sum(a); b = warp_sum(b);
    if (lane == 0) { red[warp] = a; red[kMaxWarps + warp] = b; }
    team_bar(bar_id, nwarps * 32);
    a = 0.0; b = 0.0;
    for (int w = 0; w < nwarps; ++w) { a += red[w]; b += red[kMaxWarps + w]; }
    team_bar(bar_id, nwarps * 32);
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
    auto sphere = [&](int lo, int hi) -> float4 {
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
        return make_float4(cx, cy, cz, t * t);
    };
    for (int b = first + tid; b < nblk; b += nthr) blk4[b] = sphere(b * kBlk, min(m.L, (b + 1) * kBlk));
    // the super-blocks of kSup blocks each, from the points themselves (the last threads take them, so that both levels run at once)
    const int nsup = (nblk + kSup - 1) / kSup;
    for (int sb = first / kSup + (nthr - 1 - tid); sb < nsup; sb += nthr)
        blk4[nblk + sb] = sphere(sb * kSup * kBlk, min(m.L, (sb + 1) * kSup * kBlk));
}

// V (Eq. 3a) of the team's chain from its fp32 C-betas: v_far (every pair at its clamped value) + the excess of the
// near pairs; every thread of the team returns the same value
__device__ __forceinline__ double team_full_energy(const DevModel &m, const float4 *cb4, double *red, int warp, int nwarps,
                                                   int lane, int bar_id)
{
    double e = 0.0;
    // Work item = (row i, chunk q): the 32 columns j = i + min_sep + 32 q + lane.  A warp takes U rows of the same chunk
    // per trip, so that U gathers are in flight per lane (a trip costs one L2 round trip whatever U is).
    constexpr int U = 8;
    const int nrow = m.L - m.min_sep;                        // rows with at least one column
    for (int c0 = 0; c0 < nrow; c0 += 32) {
        const int nr = nrow - c0;                            // rows that still have columns in this chunk
        for (int i0 = warp; i0 < nr; i0 += nwarps * U) {
            float d2[U], f[U];
            float2 g[U];
            int rj[U];
            float part = 0.0f;
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int i = i0 + u * nwarps;
                const bool ok = i < nr;
                const int ic = ok ? i : 0;
                const int j = ic + m.min_sep + c0 + lane;
                const float4 ci = cb4[ic];
                const float4 cj = cb4[min(j, m.L - 1)];
                const float dx = ci.x - cj.x, dy = ci.y - cj.y, dz = ci.z - cj.z;
                d2[u] = (ok && j < m.L) ? fmaf(dx, dx, fmaf(dy, dy, dz * dz)) : m.far2;
                rj[u] = tri_row(ic, 0, m.L) + j;
            }
#pragma unroll
            for (int u = 0; u < U; ++u) {
                g[u] = make_float2(0.0f, 0.0f); f[u] = 0.0f;
                if (d2[u] < m.far2) {
                    int b;
                    bin_frac(d2[u], m.t0, m.inv_delta, m.tmax, m.thmax, b, f[u]);
                    g[u] = __ldg(m.Epk + (size_t)rj[u] * m.nb + b);
                }
            }
#pragma unroll
            for (int u = 0; u < U; ++u) part += fmaf(f[u], g[u].y, g[u].x);
            e += (double)part;
        }
    }
    return m.v_far + team_sum(e, red, warp, nwarps, lane, bar_id);
}

// SG: global proposals too are evaluated speculatively, one warp per step (separate instantiations, so that neither
// carries the other's pair loop in its register budget)
// RING: the local phase reads its rows from the shared-memory ring (a.ring_cols > 0) or gathers them from L2.
// CB64: the fp64 C-betas are kept in shared memory (a.cb64) or rebuilt from N, CA, C.
// STRIDED: the local sweeps take NEXT-4's strided order (its own instantiations: Alg. 1's kernels do not carry that code).
template <bool SG, bool RING, bool CB64, bool STRIDED = false>
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
    const int w_eff = min(a.window, L - 1);
    const int span = min(2 * a.window, L - 1);            // largest j - i of an in-window pair
    constexpr bool use_ring = RING;

    unsigned long long *full_bar = reinterpret_cast<unsigned long long *>(smem_raw);                 // [R]
    unsigned long long *empty_bar = full_bar + R;                                                     // [R]
    const uint32_t full_bar_u32 = smem_u32(full_bar);
    float *ring = reinterpret_cast<float *>(smem_raw + sweep_header_bytes(R)) + (R > 0 ? kRingPadRows * m.row_stride : 0);
    const size_t chains_off = sweep_header_bytes(R) + ring_bytes(R, a.ring_rows, m.row_stride);

    const long long row0 = (long long)blockIdx.x * C;
    const int nvalid = (int)min((long long)C, a.B - row0);
    const long long cyc = (long long)a.n_global + a.n_local;
    auto sweep_is_global = [&](long long t) -> bool {
        const long long r = t % cyc;
        return a.global_first ? (r < a.n_global) : (r >= a.n_local);
    };

    if (threadIdx.x == 0) {
        for (int q = 0; q < R; ++q) { mbar_init(&full_bar[q], 1); mbar_init(&empty_bar[q], (uint32_t)nvalid); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // ================= producer warp: stream the columns of every local sweep through the ring ===========
    if (slot == C) {
        if (!use_ring || lane != 0) return;
        const uint32_t row_bytes = (uint32_t)(m.row_stride * sizeof(float));
        int s = 0;                                          // ring slot of the next column
        long long rev = 0;                                  // revolutions of the ring so far
        for (long long t = a.sweep_offset; t < a.sweep_offset + a.n_sweeps; ++t) {
            if (sweep_is_global(t)) continue;
            for (int j = 0; j < L; ++j) {
                // slot s is free once every team has arrived on its empty barrier for the column it held before
                if (rev > 0) mbar_wait(&empty_bar[s], (uint32_t)((rev - 1) & 1));
                const int nrows = min(span, j) - m.min_sep + 1;   // rows j - i = min_sep .. min(span, j): contiguous in Ebd
                void *bar = &full_bar[s];
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // the teams' reads of the old column come first
                if (nrows > 0) {
                    mbar_expect_tx(bar, (uint32_t)nrows * row_bytes);
                    AMH_ASSERT(nrows <= a.ring_rows && nrows <= m.band_rows && s >= 0 && s < R, 6);
                    tma_bulk_g2s(ring + (size_t)s * a.ring_rows * m.row_stride, m.Ebd + (size_t)j * m.band_rows * m.row_stride,
                                 (uint32_t)nrows * row_bytes, bar);
                } else {
                    mbar_arrive(bar);
                }
                if (++s == R) { s = 0; ++rev; }
            }
        }
        return;
    }
    if (slot >= nvalid) return;

    // ================= team: one chain =====================================================================
    const int cbn_rows = a.local_stride > 0 ? 2 * a.nspec : a.nspec;   // strided sweeps also keep the columns' current C-betas
    unsigned char *cbase = smem_raw + chains_off + (size_t)slot * chain_smem_bytes(L, a.cb64, cbn_rows, a.wpts, W);
    constexpr bool cb64 = CB64;
    const int na = cb64 ? 4 : 3;                            // atoms per residue kept in fp64
    double *X = reinterpret_cast<double *>(cbase), *Y = X + na * L, *Z = Y + na * L;
    double *red = Z + na * L + ((3 * na * L) & 1), *b_cd = red + 2 * kMaxWarps, *b_sd = b_cd + kDrawBatch, *b_lu = b_sd + kDrawBatch;
    double *rot_s = b_lu + kDrawBatch, *sp_new = rot_s + 12 * kMaxSpec, *sp_T = sp_new + kMaxSpec;
    float4 *cb4 = reinterpret_cast<float4 *>(sp_T + kMaxSpec);
    float4 *blk4 = cb4 + L;
    float4 *cbn = blk4 + (L + kBlk - 1) / kBlk + ((L + kBlk - 1) / kBlk + kSup - 1) / kSup;
    float *s = reinterpret_cast<float *>(cbn + (size_t)cbn_rows * a.wpts);
    float *b_sp = s + n;
    int *ctr = reinterpret_cast<int *>(b_sp + kDrawBatch);

    const long long row = row0 + slot;
    const unsigned long long chain = (unsigned long long)(a.chain_offset + row);

    for (int q = tid; q < n; q += nthreads) s[q] = a.states[row * n + q];
    if (tid == 0) ctr[0] = 0;
    team_bar(bar_id, nthreads);
    // the row term of residue i in a local table address (see LocalTab)
    auto row_term = [&](int i) -> float {
        return __int_as_float(use_ring ? -i * m.row_stride * 4 : (int)(tri_base(i, L) * m.nb * 8));
    };
    if (warp == 0)
        nerf_build_warp(m, s, lane, [&](int res, int at, double x, double y, double z) {
            if (at == 3) cb4[res] = make_float4((float)x, (float)y, (float)z, row_term(res));
            if (at < na) { const int f = at * L + res; X[f] = x; Y[f] = y; Z[f] = z; }
        });
    team_bar(bar_id, nthreads);

    double best = INFINITY, e_end = 0.0;
    unsigned long long acc_l = 0, acc_g = 0;
    // exact-decision guard: the bound on the fp32 error of dE grows with the size of the coordinates (their fp32 rounding)
    double ext_scale = fmax(1.0, (double)team_extent(cb4, L, red, tid, nthreads, warp, nwarps, lane, bar_id) * (1.0 / 32.0));
    // local proposals are evaluated by groups of gl lanes, 32 / gl groups per warp
    const int gshift = a.lanes_per_step == 4 ? 2 : (a.lanes_per_step == 8 ? 3 : (a.lanes_per_step == 16 ? 4 : 5));
    const int gl = 1 << gshift, gpw = 32 >> gshift;
    const int grp = lane >> gshift, glane = lane & (gl - 1);
    const int nspec = a.nspec;
    // ring bookkeeping of this team: the slot of column 0 of the current local sweep, the columns it has waited for and
    // the columns it has released
    int slot_j0 = 0;                                         // ring slot of column 0 of this sweep
    int seen_slot = R - 1;                                   // ring slot and phase parity of the last column waited for
    uint32_t seen_par = 1;
    int dead_slot = 0;                                       // ring slot of the next column to release
    LocalTab tb;
    tb.base = use_ring ? reinterpret_cast<const unsigned char *>(ring) : reinterpret_cast<const unsigned char *>(m.Epk);
    tb.ring_cols = R; tb.ring_rows = a.ring_rows; tb.min_sep = m.min_sep; tb.stride4 = m.row_stride * 4; tb.nb8 = m.nb * 8;
    tb.slot_c = 0; tb.c_ref = 0;
    tb.lo = use_ring ? -(long long)kRingPadRows * m.row_stride * 4 : 0;
    tb.hi = use_ring ? (long long)R * a.ring_rows * m.row_stride * 4 : (long long)((size_t)L * (L - 1) / 2) * m.nb * 8;

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
            if (cb64) {                                      // the stored C-beta turns with its residue
                const int f = 3 * L + res;
                rot_apply(R_, X[f], Y[f], Z[f], x, y, z);
                X[f] = x; Y[f] = y; Z[f] = z;
            } else {
                cb_point(m, X, Y, Z, L, res, x, y, z);
            }
            cb4[res] = make_float4((float)x, (float)y, (float)z, row_term(res));
        }
    };

    for (long long t = a.sweep_offset; t < a.sweep_offset + a.n_sweeps; ++t) {
        const bool gp = sweep_is_global(t);                  // proposals judged on all pairs (Eq. 1) or on the window (Eq. 2)
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
        tb.c_ref = 0; tb.slot_c = slot_j0;                   // ring slot of the window centre, advanced with it
        int dead_rel = 0;                                    // columns < dead_rel of this sweep have been released (tid 0)
        const double guard = (gp ? a.guard_global : a.guard_local) * ext_scale * invT;
        double S_base = 0.0;                                 // S_old of step k - 1 for the current state (every thread holds it)

        if (gp) {                                            // the local sweeps moved everything: fresh culling blocks
            team_blocks(m, cb4, blk4, 0, tid, nthreads);
            team_bar(bar_id, nthreads);
        }
        int k = 0, batch_start = 0, batch_end = 0;
        if (STRIDED && !gp && a.local_stride > 0) {
            // ======== NEXT-4: strided local sweep (R26) ========================================================
            // The residues are visited in colour classes o = 0 .. s-1 (c = o, o + s, ...), phi_c then psi_c.  With
            // s >= 2w + 1 the windows of a class do not overlap: an accepted move turns everything right of it rigidly, which
            // changes no distance inside another window, so the proposals of a class do not interact and the order inside a
            // class is immaterial.  A pass evaluates the same variable (phi, then psi) of up to nspec residues of a class
            // against the current state, one group each, decides them all, and commits every accepted one together.
            // Nothing is speculative here: every evaluation stands.  (s < 2w + 1: one proposal per pass, in the same order.)
            const int sd = a.local_stride;
            const bool indep = sd >= 2 * w_eff + 1;
            float4 *cbo = cbn + (size_t)nspec * a.wpts;             // the current C-betas of the columns (the old state's sum)
            int pos_class = 0;                                      // position of the class's first variable in the sweep
            for (int o = 0; o < sd && o < L; ++o) {
                const int cnt = (L - o + sd - 1) / sd;
                const int chunk = indep ? nspec : 1;
                for (int r0 = 0; r0 < cnt; r0 += indep ? chunk : 1) {
                  for (int par = 0; par < 2; ++par) {
                    // the independent order: all phi of the chunk, then all psi; the sequential one: phi_c, psi_c per residue
                    const int S = min(chunk, cnt - r0);
                    // ---- draws of the pass: lane r of warp 0 the proposal, of the last warp the uniform -------------
                    if (lane < S && (warp == 0 || warp == nwarps - 1)) {
                        const int kk = 2 * (o + (r0 + lane) * sd) + par;
                        const unsigned long long step = (unsigned long long)t * (unsigned long long)n + (unsigned long long)kk;
                        if (warp == 0) {
                            uint32_t x1;
                            const uint32_t x0 = draw01(a.seed, chain, step, PURPOSE_PROPOSAL, x1);
                            float sp;
                            if (a.prop_mode == 2) {
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
                            double sdl, cdl;
                            sincos((double)sp - (double)s[kk], &sdl, &cdl);
                            b_sp[lane] = sp; b_cd[lane] = cdl; b_sd[lane] = sdl;
                        }
                        if (warp == nwarps - 1) {
                            const uint32_t x0 = draw0(a.seed, chain, step, PURPOSE_ACCEPT);
                            b_lu[lane] = log((double)((x0 >> 8) + 1u) * 5.9604644775390625e-08);
                        }
                    }
                    team_bar(bar_id, nthreads);
                    // ---- evaluation: group r takes residue r0 + r of the class ---------------------------------------------
                    const int r = warp * gpw + grp;
                    const bool active = r < S;
                    const int c = o + (r0 + min(r, S - 1)) * sd, kk = 2 * c + par, split = c + par;
                    const bool inert = (kk == 0) || (kk == n - 1);
                    const int ilo = max(0, c - w_eff), jhi = min(L - 1, c + w_eff);
                    const int nI = split - ilo, nJ = jhi - split + 1;
                    float4 *cbn_r = cbn + (size_t)min(r, nspec - 1) * a.wpts, *cbo_r = cbo + (size_t)min(r, nspec - 1) * a.wpts;
                    double p_dE = 0.0;
                    if (active && !inert) {
                        const Rot Rk = step_rot(kk, r);
                        if (glane == 0) {
#pragma unroll
                            for (int q = 0; q < 9; ++q) rot_s[12 * r + q] = Rk.r[q];
#pragma unroll
                            for (int q = 0; q < 3; ++q) rot_s[12 * r + 9 + q] = Rk.t[q];
                        }
                        for (int jj = glane; jj < nJ; jj += gl) {
                            const int j = split + jj;
                            double x0, y0, z0, x, y, z;
                            if (cb64) { x0 = X[3 * L + j]; y0 = Y[3 * L + j]; z0 = Z[3 * L + j]; }
                            else cb_point(m, X, Y, Z, L, j, x0, y0, z0);
                            rot_apply(Rk, x0, y0, z0, x, y, z);
                            const float ct = __int_as_float(col_term<RING>(tb, j));
                            cbn_r[jj] = make_float4((float)x, (float)y, (float)z, ct);
                            const float4 cur = cb4[j];
                            cbo_r[jj] = make_float4(cur.x, cur.y, cur.z, ct);
                        }
                    }
                    __syncwarp();
                    if (active && !inert)
                        p_dE = (double)local_new_sum<RING>(m, tb, cb4, cbn_r, ilo, split, nI, nJ, glane, gl)
                             - (double)local_new_sum<RING>(m, tb, cb4, cbo_r, ilo, split, nI, nJ, glane, gl);
                    for (int d = gl >> 1; d > 0; d >>= 1) p_dE += __shfl_xor_sync(0xffffffffu, p_dE, d);
                    if (active && glane == 0) sp_new[r] = p_dE;
                    team_bar(bar_id, nthreads);
                    // ---- decisions: lane q holds step q of the pass; all of them stand ---------------------------------------
                    const int cq = o + (r0 + min(lane, S - 1)) * sd, kq = 2 * cq + par;
                    const bool inert_q = (kq == 0) || (kq == n - 1);
                    double dE = (lane < S && !inert_q) ? sp_new[lane] : 0.0;
                    const double lu = b_lu[min(lane, S - 1)];
                    const bool unc = lane < S && !inert_q && fabs(lu + dE * invT) < guard;
                    bool acc = lane < S && (lu <= -dE * invT);
                    unsigned m_unc = __ballot_sync(0xffffffffu, unc), m_exact = 0;
                    while (m_unc) {
                        const int r1 = __ffs(m_unc) - 1;
                        const int cx = o + (r0 + r1) * sd, kx = 2 * cx + par;
                        const double dx = team_sum(exact_dE_partial(exact_model(m), X, Y, Z, cb64 ? 1 : 0, kx, b_cd[r1], b_sd[r1],
                                                                    max(0, cx - w_eff), min(L - 1, cx + w_eff), tid, nthreads),
                                                   red, warp, nwarps, lane, bar_id);
                        const bool ax = b_lu[r1] <= -dx / T;
                        if (lane == r1) { dE = dx; acc = ax; }
                        m_exact |= 1u << r1;
                        m_unc &= ~(1u << r1);
                    }
                    const unsigned m_acc = __ballot_sync(0xffffffffu, acc);
                    if (warp == 0 && lane < S) {
                        const long long q = (t - a.sweep_offset) * n + pos_class + 2 * (r0 + lane) + par;
                        if (q < a.trace_steps) {
                            const size_t z = (size_t)row * a.trace_steps + q;
                            if (a.trace_prop) a.trace_prop[z] = b_sp[lane];
                            if (a.trace_dE) a.trace_dE[z] = dE;
                            if (a.trace_acc) a.trace_acc[z] = (unsigned char)((acc ? 1 : 0) | (((m_exact >> lane) & 1u) ? 2 : 0));
                        }
                    }
                    acc_l += (unsigned long long)__popc(m_acc);
                    // ---- commit: the accepted rotations (all given in the frame before the pass) compose from the left:
                    // a residue right of the accepted bonds c_1 < ... < c_j moves by M_j = R_1 R_2 ... R_j -----------------------
                    if (tid == 0) {
                        Xf cum = xf_identity();
                        for (unsigned mm = m_acc; mm; mm &= mm - 1) {
                            const int r1 = __ffs(mm) - 1;
                            const int k1 = 2 * (o + (r0 + r1) * sd) + par;
                            s[k1] = b_sp[r1];
                            if (k1 == 0 || k1 == n - 1) { for (int q = 0; q < 9; ++q) rot_s[12 * r1 + q] = cum.r[q]; for (int q = 0; q < 3; ++q) rot_s[12 * r1 + 9 + q] = cum.t[q]; continue; }
                            Xf Rr;
                            for (int q = 0; q < 9; ++q) Rr.r[q] = rot_s[12 * r1 + q];
                            for (int q = 0; q < 3; ++q) Rr.t[q] = rot_s[12 * r1 + 9 + q];
                            cum = xf_mul(cum, Rr);
                            for (int q = 0; q < 9; ++q) rot_s[12 * r1 + q] = cum.r[q];
                            for (int q = 0; q < 3; ++q) rot_s[12 * r1 + 9 + q] = cum.t[q];
                        }
                    }
                    team_bar(bar_id, nthreads);
                    if (m_acc) {
                        const int first = __ffs(m_acc) - 1;
                        const int res0 = o + (r0 + first) * sd;                       // the leftmost residue that may move
                        for (int res = res0 + tid; res < L; res += nthreads) {
                            // the accepted move that governs this residue: the last one with c_r <= res (phi) or c_r < res (psi)
                            int jr = -1, jprev = -1;
                            for (unsigned mm = m_acc; mm; mm &= mm - 1) {
                                const int r1 = __ffs(mm) - 1;
                                const int c1 = o + (r0 + r1) * sd;
                                if (c1 + par <= res) { jprev = jr; jr = r1; }
                            }
                            if (jr < 0) continue;
                            const int cj = o + (r0 + jr) * sd;
                            const bool on_axis = (par == 0 && res == cj) && !(2 * cj == 0);      // phi_c: N_c and CA_c stay with the left side
#pragma unroll
                            for (int at = 0; at < 4; ++at) {
                                if (at == 3 && !cb64) break;
                                const int jm = (on_axis && at < 2) ? jprev : jr;
                                if (jm < 0) continue;
                                Rot Mj;
#pragma unroll
                                for (int q = 0; q < 9; ++q) Mj.r[q] = rot_s[12 * jm + q];
#pragma unroll
                                for (int q = 0; q < 3; ++q) Mj.t[q] = rot_s[12 * jm + 9 + q];
                                const int f = at * L + res;
                                double x, y, z;
                                rot_apply(Mj, X[f], Y[f], Z[f], x, y, z);
                                X[f] = x; Y[f] = y; Z[f] = z;
                            }
                            double x, y, z;
                            if (cb64) { x = X[3 * L + res]; y = Y[3 * L + res]; z = Z[3 * L + res]; }
                            else cb_point(m, X, Y, Z, L, res, x, y, z);
                            cb4[res] = make_float4((float)x, (float)y, (float)z, row_term(res));
                        }
                    }
                    team_bar(bar_id, nthreads);
                  }
                }
                pos_class += 2 * cnt;
            }
            k = n;                                                   // the sweep is done: skip Alg. 1's loop below
        }
        while (k < n) {
            // ---- a1/a2: draws of the next 64 steps, two per lane (R5-R7) ----------------------------------
            if (k >= batch_end) {
                batch_start = k; batch_end = min(n, k + kDrawBatch);
                const int draw_warp_u = nwarps > 1 ? 1 : 0;   // the warp that draws the uniforms of the accept test
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
            // ---- a pass: S proposals, group r evaluating step k + r against the current state -------------------
            // local sweeps: groups of gl lanes; global sweeps: SG = one warp per step, else one step by the whole team
            const bool teamwide = gp && !SG;
            const int S = teamwide ? 1 : min(gp ? min(nwarps, kMaxSpec) : nspec, batch_end - k);
            double my_new = 0.0, my_T = 0.0;                 // S_new and T of step k + lane, lane < S (filled below)
            if (teamwide) {
                // ======== one proposal, evaluated by the whole team (a3/a5/a6) =================================
                const int bi = k - batch_start;
                const int split = (k >> 1) + (k & 1);
                const bool inert = (k == 0) || (k == n - 1);
                double p_new = 0.0, p_T = 0.0;
                Rot Rk;
                if (!inert) {
                    Rk = step_rot(k, bi);
                    if (tid == 0) {                           // kept in shared memory for the commit, not in registers
#pragma unroll
                        for (int q = 0; q < 9; ++q) rot_s[q] = Rk.r[q];
#pragma unroll
                        for (int q = 0; q < 3; ++q) rot_s[9 + q] = Rk.t[q];
                    }
                    p_new = global_cols_sum(m, cb4, blk4, X, Y, Z, cb64, true, Rk, split, split, L - 1, tid, nthreads, ctr);
                }
                if (k & 1) {                                  // the split moved: column c leaves, row c enters
                    const int c = k >> 1;
                    p_T = global_row_sum(m, cb4, c, c + m.min_sep, L - c - m.min_sep, tid, nthreads)
                        - global_col_sum(m, cb4, c, c - m.min_sep + 1, tid, nthreads);
                }
                team_sum2(p_new, p_T, red, warp, nwarps, lane, bar_id);
                if (tid == 0) ctr[0] = 0;                     // every warp is past its last grab; the pass ends with a barrier
                my_new = p_new; my_T = p_T;
            } else {
                if (use_ring && !gp) {
                    // columns left of the window centre are dead for this chain; wait for the ones the pass needs
                    const int c_now = k >> 1;
                    if (tid == 0)
                        while (dead_rel < c_now) {
                            mbar_arrive(&empty_bar[dead_slot]);
                            ++dead_rel;
                            if (++dead_slot == R) dead_slot = 0;
                        }
                    const int need = min(L - 1, ((k + S - 1) >> 1) + a.window);
                    while (seen_rel < need) {
                        ++seen_rel;
                        if (++seen_slot == R) { seen_slot = 0; seen_par ^= 1u; }
                        mbar_wait_u32(full_bar_u32 + 8u * (uint32_t)seen_slot, seen_par);
                    }
                    if (tb.c_ref < c_now) {                   // a pass advances by less than R columns
                        tb.slot_c += c_now - tb.c_ref;
                        if (tb.slot_c >= R) tb.slot_c -= R;
                        tb.c_ref = c_now;
                    }
                }
                const int r = gp ? warp : warp * gpw + grp;
                const int gl_x = gp ? 32 : gl, glane_x = gp ? lane : glane;
                const bool active = r < S;
                const int kk = k + r, bi = min(kk, batch_end - 1) - batch_start;
                const bool inert = (kk == 0) || (kk == n - 1);
                const int c = kk >> 1, split = c + (kk & 1);
                double p_new = 0.0, p_T = 0.0;
                if (gp) {
                    // ---- a5: all straddling pairs (Eq. 3a), one warp ---------------------------------------------
                    if (active) {
                        Rot Rk;
                        if (!inert) {
                            Rk = step_rot(kk, bi);
                            if (lane == 0) {
#pragma unroll
                                for (int q = 0; q < 9; ++q) rot_s[12 * r + q] = Rk.r[q];
#pragma unroll
                                for (int q = 0; q < 3; ++q) rot_s[12 * r + 9 + q] = Rk.t[q];
                            }
                            p_new = global_cols_sum(m, cb4, blk4, X, Y, Z, cb64, true, Rk, split, split, L - 1, lane, 32);
                        }
                        if (kk & 1)
                            p_T = global_row_sum(m, cb4, c, c + m.min_sep, L - c - m.min_sep, lane, 32)
                                - global_col_sum(m, cb4, c, c - m.min_sep + 1, lane, 32);
                    }
                } else {
                    // ---- a3/a4: in-window straddling pairs (Eq. 3b) ------------------------------------------------
                    const int ilo = max(0, c - w_eff), jhi = min(L - 1, c + w_eff);
                    const int nI = split - ilo, nJ = jhi - split + 1;
                    float4 *cbn_r = cbn + (size_t)min(r, nspec - 1) * a.wpts;
                    if (active && !inert) {
                        const Rot Rk = step_rot(kk, bi);
                        if (glane_x == 0) {
#pragma unroll
                            for (int q = 0; q < 9; ++q) rot_s[12 * r + q] = Rk.r[q];
#pragma unroll
                            for (int q = 0; q < 3; ++q) rot_s[12 * r + 9 + q] = Rk.t[q];
                        }
                        // two columns per lane and trip, loads first (w + 1 = gl + 1 columns is the common case)
                        for (int jj = glane_x; jj < nJ; jj += 2 * gl_x) {
                            const int jj2 = jj + gl_x;
                            const bool two = jj2 < nJ;
                            const int j = split + jj, j2 = split + (two ? jj2 : jj);
                            double x0, y0, z0, x, y, z, u0, v0, w0, u, v, w_;
                            if (cb64) {
                                x0 = X[3 * L + j]; y0 = Y[3 * L + j]; z0 = Z[3 * L + j];
                                u0 = X[3 * L + j2]; v0 = Y[3 * L + j2]; w0 = Z[3 * L + j2];
                            } else {
                                cb_point(m, X, Y, Z, L, j, x0, y0, z0);
                                cb_point(m, X, Y, Z, L, j2, u0, v0, w0);
                            }
                            rot_apply(Rk, x0, y0, z0, x, y, z);
                            rot_apply(Rk, u0, v0, w0, u, v, w_);
                            AMH_ASSERT(jj < a.wpts && r < nspec && j < L && (!two || (jj2 < a.wpts && j2 < L)), 7);
                            cbn_r[jj] = make_float4((float)x, (float)y, (float)z, __int_as_float(col_term<RING>(tb, j)));
                            if (two) cbn_r[jj2] = make_float4((float)u, (float)v, (float)w_, __int_as_float(col_term<RING>(tb, j2)));
                        }
                    }
                    __syncwarp();
                    if (active) {
                        if (!inert) p_new = (double)local_new_sum<RING>(m, tb, cb4, cbn_r, ilo, split, nI, nJ, glane_x, gl_x);
                        p_T = (double)local_transition<RING>(m, tb, cb4, kk, w_eff, glane_x, gl_x);
                    }
                }
                // ---- a6: reduction over the group's lanes (every lane of the warp takes part) ----------------
                for (int d = gl_x >> 1; d > 0; d >>= 1) {
                    p_new += __shfl_xor_sync(0xffffffffu, p_new, d);
                    p_T += __shfl_xor_sync(0xffffffffu, p_T, d);
                }
                if (active && glane_x == 0) { sp_new[r] = p_new; sp_T[r] = p_T; }
                team_bar(bar_id, nthreads);
                if (lane < S) { my_new = sp_new[lane]; my_T = sp_T[lane]; }
            }
            // ---- a7: Metropolis tests in step order; lane r holds step k + r ---------------------------------------------
            // S_old(k + r) = S_base + T(k) + ... + T(k + r)  (inclusive prefix over the lanes)
            double pre = my_T;
#pragma unroll
            for (int d = 1; d < kMaxSpec; d <<= 1) {
                const double v = __shfl_up_sync(0xffffffffu, pre, d);
                if (lane >= d) pre += v;
            }
            const double s_old = S_base + pre;
            const int kq = k + lane;                          // this lane's step (meaningful for lane < S)
            const int bq = min(kq, batch_end - 1) - batch_start;
            const bool inert_q = (kq == 0) || (kq == n - 1);
            double dE = inert_q ? 0.0 : my_new - s_old;
            const double lu = b_lu[bq];
            // exact-decision guard (R24): a gap inside the fp32 error bound of dE is decided by the fp64 path
            const bool unc = lane < S && !inert_q && fabs(lu + dE * invT) < guard;
            bool acc = lane < S && (lu <= -dE * invT);        // Eq. 1a/2a, R14
            const unsigned m_unc = __ballot_sync(0xffffffffu, unc);
            unsigned m_go = __ballot_sync(0xffffffffu, acc || unc);
            unsigned m_exact = 0;
            int rsel = S;                                     // first accepted step of the pass
            while (m_go) {
                const int r0 = __ffs(m_go) - 1;
                if (!((m_unc >> r0) & 1u)) { rsel = r0; break; }
                const int kx = k + r0, bx = kx - batch_start, cx = kx >> 1;
                const double dx = team_sum(exact_dE_partial(exact_model(m), X, Y, Z, cb64 ? 1 : 0, kx, b_cd[bx], b_sd[bx],
                                                            gp ? 0 : max(0, cx - w_eff), gp ? L - 1 : min(L - 1, cx + w_eff),
                                                            tid, nthreads), red, warp, nwarps, lane, bar_id);
                const bool ax = b_lu[bx] <= -dx / T;
                if (lane == r0) { dE = dx; acc = ax; }
                m_exact |= 1u << r0;
                if (ax) { rsel = r0; break; }
                m_go &= ~(1u << r0);
            }
            const int nstand = (rsel < S) ? rsel + 1 : S;     // steps whose result stands
            if (warp == 0 && lane < nstand) {
                const long long q = (t - a.sweep_offset) * n + kq;
                if (q < a.trace_steps) {
                    const size_t z = (size_t)row * a.trace_steps + q;
                    if (a.trace_prop) a.trace_prop[z] = b_sp[bq];
                    if (a.trace_dE) a.trace_dE[z] = dE;
                    if (a.trace_acc) a.trace_acc[z] = (unsigned char)((lane == rsel ? 1 : 0) | (((m_exact >> lane) & 1u) ? 2 : 0));
                }
            }
            // S_old carried to the next pass: an accepted proposal's S_new is the S_old of its step for the new state
            // (an inert one moves nothing); without an accept, the S_old of the last step evaluated
            {
                const int src = (rsel < S) ? rsel : S - 1;
                const bool take_new = (rsel < S) && !((k + rsel == 0) || (k + rsel == n - 1));
                S_base = __shfl_sync(0xffffffffu, take_new ? my_new : s_old, src);
            }
            if (rsel < S) {
                // ---- commit the accepted step --------------------------------------------------------
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
        if (!gp && use_ring) {
            // every column of this sweep is dead for this chain
            if (tid == 0)
                while (dead_rel < L) {
                    mbar_arrive(&empty_bar[dead_slot]);
                    ++dead_rel;
                    if (++dead_slot == R) dead_slot = 0;
                }
            slot_j0 = (slot_j0 + L) % R;
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
