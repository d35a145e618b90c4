/*
 * amh.h - C ABI of the B200-native Alternating Metropolis-Hastings (AMH) hot path.
 *
 * Method: Ghantasala, Jaiswal, Datta, "An Efficient MCMC Approach to Energy Function Optimization in
 * Protein Structure Prediction", arXiv 2211.03193.  "PAPER.md:<line>" cites the text of that paper,
 * "Rn" a reading listed in DESIGN.md (taken where the paper is silent, ambiguous or garbled).
 *
 * What the library computes (one GPU, hand-written CUDA for sm_100a, no CPU fallback):
 *   state        s in R^n, n = 2L, s[2i] = phi_i, s[2i+1] = psi_i, radians        PAPER.md:25, Fig. 2 (:67); R15, R16
 *   geometry     x = G(s): backbone by NeRF with ideal geometry, C-beta from N/CA/C   PAPER.md:39, 77; R1-R4
 *   energy       V(x) = sum_{i<j, j-i>=min_sep} e_ij(|CB_i - CB_j|)   (Eq. 3a)      PAPER.md:75; R8, R9
 *                e_ij(d): -log(p_ij + eps) interpolated linearly between bin centres, clamped at the ends
 *   local energy V_local(x,k,w): the same sum restricted to residues floor(k/2)-w .. floor(k/2)+w
 *                (Eq. 3b)                                                          PAPER.md:81-86; R12
 *   MH           single-flip proposal of s_k, accept iff log u <= -dE/T   (Eq. 1a-1c, 2a-2b)
 *                                                                                  PAPER.md:27-49; R5, R7, R14
 *   alternation  cycles of n_global sweeps judged on V, then n_local sweeps judged on V_local;
 *                one sweep = k = 0..n-1 in order   (Alg. 1, Fig. 1)                 PAPER.md:55, 97-123, 129; R10
 *   RNG          Philox4x32-10, key = seed, counter = (step_lo, step_hi, chain, purpose), step = t*n + k   R6
 *
 * Conventions
 *   - "device" pointers are CUDA device memory of the current device; "host" pointers are ordinary
 *     host memory.  Each argument says which.  The caller owns every buffer it passes in.
 *   - All device work is enqueued on `cuda_stream` (a cudaStream_t passed as void*; NULL = the legacy
 *     default stream).  amh_run / amh_energy / amh_energy_local / amh_coords do not synchronise and
 *     do not allocate; the *_host variants and amh_create / amh_destroy synchronise.
 *   - Every function returns an amh_status; nothing throws or exits.  amh_last_error() returns a
 *     thread-local, NUL-terminated description of the last failure on this thread.
 *   - Chain ids: row b of a state batch is chain (chain_offset + b); the id, not the row, keys the RNG,
 *     so a batch may be sharded across calls or GPUs without changing any trajectory.
 */
#ifndef AMH_H_
#define AMH_H_

#ifdef __cplusplus
extern "C" {
#endif

typedef struct amh_ctx amh_ctx;   /* opaque; owns the device energy table and the geometry constants */

typedef enum {
    AMH_OK = 0,
    AMH_ERR_INVALID_ARG = 1,   /* NULL where a pointer is required, sizes < 1, T <= 0, NaN/Inf/negative p, ... */
    AMH_ERR_UNSUPPORTED = 2,   /* non-uniform bins, AMH_PARAM_TR5, L beyond the shared-memory plan */
    AMH_ERR_CUDA = 3,          /* a CUDA runtime call failed; see amh_last_error() */
    AMH_ERR_OOM = 4
} amh_status;

typedef enum {
    AMH_PARAM_PHI_PSI = 0,     /* 2 variables per residue (the paper's AlphaFold1 mapping) */
    AMH_PARAM_TR5 = 1          /* 5 variables per residue (trRosetta2; config 3): contexts of this kind are
                                  built by amh_create_tr5(), which also takes the orientation maps */
} amh_param;

/* Geometry, energy and numerics options (the MODEL; nothing about the launch).  amh_default_options() fills the
 * values every config of BASELINE.json uses (R2, R3, R9).  Lengths in Angstrom, angles in radians. */
typedef struct {
    double len_n_ca, len_ca_c, len_c_n;          /* 1.458, 1.525, 1.329 */
    double ang_n_ca_c, ang_ca_c_n, ang_c_n_ca;   /* 111.2, 116.2, 121.7 degrees */
    double omega;                                /* pi (trans) */
    double cb_len, cb_ang, cb_dih;               /* |CA-CB| 1.522, angle N-CA-CB 1.927, dihedral C-N-CA-CB -2.143 */
    double eps;                                  /* 1e-8, added to p inside the log */
    double guard_scale;                          /* exact-decision guard (R24): pair energies are
                                                    summed in fp32; a proposal whose gap |log u + dE/T| is below
                                                    guard_scale * G(L, window, extent) / T - G being the bound on the fp32
                                                    error of dE - is re-evaluated in fp64 (coordinates, root, -log(p + eps),
                                                    interpolation) before the decision is taken, so that every decision is
                                                    the one fp64 arithmetic gives WHERE G BOUNDS THAT ERROR.  G is calibrated,
                                                    not proven: about 4 x the largest error measured on distograms with a 5 %
                                                    uniform floor (excess energies and bin-to-bin steps of the table up to 7.1),
                                                    raised by (max(|E'|max, largest step) / 7.2)^2 for sharper tables - checked
                                                    down to one-bin peaks without a floor at eps = 1e-8, where the error stays
                                                    below a third of G (R24).  A smaller eps, or a chain that grows
                                                    several-fold beyond 32 A within one sweep (the extent is sampled at sweep
                                                    ends), is outside what was measured: raise guard_scale there.
                                                    1 = default; 0 = off (fp32 decisions); a huge value sends every proposal
                                                    through the fp64 path */
    int    min_sep;                              /* 3: pairs need j - i >= min_sep; >= 1 */
    int    pad_;
} amh_options;

/* Launch shape of amh_run (kernel internals, not part of the model; every field 0 / -1 = let the library choose).
 * Set with amh_set_launch_options(); the parity tests run many shapes and require the same trajectory from all. */
typedef struct {
    int    warps_per_chain;                      /* 0 = choose from L and B; else 1..15 */
    int    spec_local;                           /* local proposals evaluated per pass (results consumed in order up to the
                                                    first accept: same trajectory); 0 = as many as the team has lane groups,
                                                    at most 16 */
    int    lanes_per_step;                       /* lanes that share one local proposal: 0 = choose; else 4, 8, 16 or 32 */
    int    spec_global;                          /* global proposals: 1 = one warp per step, speculative like the local ones;
                                                    0 = one step at a time by the whole team; -1 = choose */
    int    chains_per_cta;                       /* chains sharing one CTA and its table ring: 0 = choose; else 1..15,
                                                    chains_per_cta * warps_per_chain <= 15 */
    int    ring_cols;                            /* slots of the shared-memory table ring of the local phase: 0 = choose,
                                                    -1 = off (rows gathered from L2), else >= window + 3 */
} amh_launch_options;

/* Alg. 1 / Fig. 1, R10, R12. */
typedef struct {
    int n_global;       /* sweeps per cycle judged on V            (>= 0) */
    int n_local;        /* sweeps per cycle judged on V_local      (>= 0; n_global + n_local >= 1) */
    int window;         /* radius w in residues, inclusive, clamped at the chain ends (>= 0) */
    int global_first;   /* 1 = Alg. 1 order (global sweeps first in each cycle); 0 = local first */
    int local_stride;   /* NEXT-4 (a VARIANT of Alg. 1; R26): 0 = the paper's order k = 0..n-1.
                           s >= 1: local sweeps visit the residues in colour classes o = 0..s-1 (c = o, o+s, o+2s, ...), phi_c
                           then psi_c; with s >= 2 * window + 1 the windows of a class do not overlap, their proposals do not
                           interact, and the kernel evaluates a class in parallel with nothing speculative.  The draws stay
                           keyed by (sweep, variable).  Global sweeps keep k = 0..n-1.  AMH_PARAM_PHI_PSI only. */
} amh_schedule;

/* R13.  T_t = t_start * (t_end/t_start)^(t/(ramp_sweeps-1)) for absolute sweep index t, constant
 * within a sweep, clamped to t_end for t >= ramp_sweeps-1; t_start == t_end or ramp_sweeps <= 1 means
 * constant t_start.  per_chain_T (DEVICE float[B], or NULL) overrides the ramp with one constant
 * temperature per row (config 4's replicas).  All temperatures must be > 0: t_start / t_end are checked
 * (INVALID_ARG); per_chain_T is checked by amh_run_host (host memory) and NOT by amh_run (device memory: a check
 * would synchronise) - a row with T <= 0 there makes that row's decisions undefined. */
typedef struct {
    double t_start, t_end;
    long long ramp_sweeps;
    const float *per_chain_T;
} amh_temperature;

typedef enum {
    AMH_PROP_UNIFORM = 0,   /* s'_k = fp32(h * 2^-23) * fp32(pi), h = (x0 >> 8) - 2^23    (BASELINE.json configs; R5) */
    AMH_PROP_GRID = 1,      /* s'_k = fp32((2m - G)/G) * fp32(pi), m = x0 mod G           (tests: Boltzmann pins P4/P5) */
    AMH_PROP_GAUSSIAN = 2   /* the paper's single flip (Eq. 1b, 129, 145): s'_k = wrap(s_k + sigma_t z),
                               z = sqrt(-2 ln u1) cos(2 pi u2) (Box-Muller), u1 = ((x0 >> 8) + 1) 2^-24, u2 = (x1 >> 8) 2^-24,
                               evaluated in fp64, wrapped to [-pi, pi), rounded once to fp32 */
} amh_prop_mode;

/* sigma_t = sigma_start + (sigma_end - sigma_start) * t / (ramp_sweeps - 1) for absolute sweep index t (the paper
 * anneals 10 -> 4 degrees over a run), clamped to sigma_end for t >= ramp_sweeps - 1; sigma_start ==
 * sigma_end or ramp_sweeps <= 1 means constant.  Radians, > 0; read in Gaussian mode only. */
typedef struct { int mode; int grid; double sigma_start, sigma_end; long long ramp_sweeps; } amh_proposal;

/* Results of amh_run.  Every pointer is optional (NULL = not wanted).  DEVICE memory for amh_run,
 * HOST memory for amh_run_host.  B = rows of the batch, n = 2L. */
typedef struct {
    float *energy;                        /* [B] V of the final state */
    float *best_energy;                   /* [B] min over this call's sweep ends of V */
    float *best_state;                    /* [B][n] the state at that sweep end */
    unsigned long long *n_accept_local;   /* [B] accepted proposals in local sweeps */
    unsigned long long *n_accept_global;  /* [B] accepted proposals in global sweeps */
    long long *first_hit_sweep;           /* [1] smallest absolute sweep index at whose end some chain of the
                                                 batch had V <= energy_threshold; -1 if none */
    float energy_threshold;
    int   trace_steps;                    /* the first trace_steps proposals of the call are traced per chain */
    float *trace_prop;                    /* [B][trace_steps] proposed value s'_k */
    double *trace_dE;                     /* [B][trace_steps] dE the decision used */
    unsigned char *trace_acc;             /* [B][trace_steps] bit 0 = accepted; bit 1 = the decision was taken by the
                                                 fp64 path of the exact-decision guard (trace_dE is then the fp64 dE) */
} amh_outputs;

/* Fill *opt with the defaults above.  opt: host. */
amh_status amh_default_options(amh_options *opt);
amh_status amh_default_launch_options(amh_launch_options *opt);

/* Force (parts of) the launch shape of later amh_run calls on this context; NULL restores the defaults.
 * INVALID_ARG when a field is out of range.  Host. */
amh_status amh_set_launch_options(amh_ctx *ctx, const amh_launch_options *opt);

/* Build a context: validate, compute E = -log(p + eps) (Eq. 3a) into device memory.
 *   out         host; receives the context
 *   n_res       L >= 1 (L < min_sep + 1 is valid: no pairs, energy 0)
 *   param       AMH_PARAM_PHI_PSI (AMH_PARAM_TR5: INVALID_ARG, use amh_create_tr5)
 *   distogram   HOST or DEVICE float [L][L][n_bins] row-major, p_ij(b) >= 0 finite; only i < j is read.
 *               Copied: the caller may free it after the call.
 *   bin_edges   HOST float [n_bins + 1], increasing, evenly spaced to 1e-5 relative (else UNSUPPORTED)
 *   n_bins      >= 2; UNSUPPORTED when the packed pair table L (L - 1) / 2 x n_bins x 8 bytes (plus one row per residue)
 *               reaches 2^31 bytes - the sweep kernel addresses it with 32-bit offsets (L = 600 allows 1,488 bins)
 *   opt         host, or NULL for the defaults
 * Synchronises the stream. */
amh_status amh_create(amh_ctx **out, int n_res, amh_param param, const float *distogram,
                      const float *bin_edges, int n_bins, const amh_options *opt, void *cuda_stream);

/* Config 3 (NEXT-2; BASELINE.json:11; PAPER.md:25 "trRosetta2 follows a 5 angle parameterization", :125 "(phi, theta,
 * omega)"; reading R25 of DESIGN.md - the paper fixes neither the parameterisation nor the orientation conventions).
 *   state   n = 5 L variables per chain: s[5i+0] = phi_i, s[5i+1] = psi_i, s[5i+2] = omega_i (torsion of the peptide bond
 *           C_i - N_{i+1}; geometry as R1 with this omega instead of the constant), s[5i+3], s[5i+4] = two slots that move
 *           no backbone atom and no C-beta (their proposals have dE = 0 and are always accepted); the residue of variable
 *           k is floor(k / 5)
 *   energy  V = sum over i < j, j - i >= min_sep of
 *               e_d(|CB_i CB_j|)                                 distogram, n_bins over the given edges (R8)
 *             + e_o(dihedral CA_i, CB_i, CB_j, CA_j)             omega map, nb_omega bins over [-pi, pi), periodic
 *             + e_t[i][j](dihedral N_i, CA_i, CB_i, CB_j) + e_t[j][i](dihedral N_j, CA_j, CB_j, CB_i)     theta map, periodic
 *             + e_p[i][j](angle CA_i, CB_i, CB_j) + e_p[j][i](angle CA_j, CB_j, CB_i)    phi map, nb_phi bins over [0, pi]
 *           every e = -log(p + eps) interpolated linearly between bin centres: clamped beyond the end centres (distance,
 *           phi), circularly (omega, theta); IUPAC dihedrals in (-pi, pi]
 *   maps    HOST or DEVICE float, row-major: omega [L][L][nb_omega] (only i < j is read), theta [L][L][nb_theta] and
 *           phi [L][L][nb_phi] (entry [i][j] scores the geometry seen from residue i: both orders are read)
 * amh_energy, amh_energy_local, amh_coords, amh_run and amh_run_host work on such a context with n = 5 L; the arithmetic
 * is fp64 throughout (no decision guard is needed: trace_acc carries bit 1 on every step); amh_exchange / amh_run_pt too. */
typedef struct {
    const float *omega, *theta, *phi;
    int nb_omega, nb_theta, nb_phi;
} amh_orientation_maps;

amh_status amh_create_tr5(amh_ctx **out, int n_res, const float *distogram, const float *bin_edges, int n_bins,
                          const amh_orientation_maps *maps, const amh_options *opt, void *cuda_stream);

/* The inter-residue geometry of config 3 for a batch of 5-slot states (the reference structure's values, from which
 * synthetic orientation maps are drawn): DEVICE double [B][L][L] each, entry [i][j] = the ORDERED pair (i, j) - distance
 * |CB_i CB_j|, omega_ij, theta_ij, phi_ij (0 on the diagonal); any output may be NULL.  TR5 contexts only. */
amh_status amh_pair_geometry(amh_ctx *ctx, const float *states, long long B, double *d_out, double *omega_out,
                             double *theta_out, double *phi_out, void *cuda_stream);

/* Free the context and everything it owns (synchronises the device). NULL is allowed. */
amh_status amh_destroy(amh_ctx *ctx);

/* V(G(s)) for a batch (Eq. 3a).  states: DEVICE float [B][n]; energy_out: DEVICE float [B]. B >= 0. */
amh_status amh_energy(amh_ctx *ctx, const float *states, long long B, float *energy_out, void *cuda_stream);

/* V_local(G(s), k, window) for a batch (Eq. 3b, R12).  0 <= k < n, window >= 0.  Same layouts. */
amh_status amh_energy_local(amh_ctx *ctx, const float *states, long long B, int k, int window,
                            float *energy_out, void *cuda_stream);

/* x = G(s) in the canonical frame (R1, R4: N_0 at the origin, CA_0 on +x, C_0 in the xy plane, y > 0).
 *   cb_out     DEVICE float  [B][L][3] C-beta, or NULL
 *   atoms_out  DEVICE double [B][L][4][3] N, CA, C, CB, or NULL */
amh_status amh_coords(amh_ctx *ctx, const float *states, long long B, float *cb_out, double *atoms_out,
                      void *cuda_stream);

/* Alg. 1 on a batch of independent chains.
 *   states        DEVICE float [B][n], in/out
 *   n_sweeps      sweeps of this call (>= 0), all kinds counted (R10)
 *   sweep_offset  absolute index of the first sweep (>= 0): it positions the call in the cycle, in the
 *                 temperature ramp and in the RNG counter, so run(a) then run(b, offset a) == run(a+b)
 *   chain_offset  chain id of row 0
 *   sched, temp   host, required
 *   prop          host, or NULL for AMH_PROP_UNIFORM
 *   out           host struct of DEVICE pointers, or NULL */
amh_status amh_run(amh_ctx *ctx, float *states, long long B, long long n_sweeps, long long sweep_offset,
                   long long chain_offset, const amh_schedule *sched, const amh_temperature *temp,
                   const amh_proposal *prop, unsigned long long seed, const amh_outputs *out,
                   void *cuda_stream);

/* NEXT-3, replica exchange (PAPER.md:160 names parallel tempering as the companion of multi-block runs; DESIGN.md
 * R23).  Chains chain_offset + b are grouped by `replicas` consecutive ids (B and chain_offset multiples of
 * replicas >= 2).  After cycle `cycle` the pairs (r, r+1) of every group with r = cycle (mod 2) are tested:
 *     accept iff log u <= (1/T_a - 1/T_b) (V_a - V_b),  u = ((x0 >> 8) + 1) 2^-24,
 *     x0 = word 0 of Philox(key = seed; counter = (cycle_lo, cycle_hi, chain id of r, 3)),
 * in fp64 on the fp32 inputs; an accepted pair swaps its TEMPERATURES (states stay in their rows).
 *   energies    DEVICE float [B]  current V of every chain (amh_run's `energy` output)
 *   per_chain_T DEVICE float [B]  in/out
 *   n_tried, n_accepted  DEVICE unsigned long long [1], incremented (not reset); NULL = not wanted */
amh_status amh_exchange(amh_ctx *ctx, const float *energies, float *per_chain_T, long long B, int replicas,
                        long long cycle, long long chain_offset, unsigned long long seed,
                        unsigned long long *n_tried, unsigned long long *n_accepted, void *cuda_stream);

/* Alternating MH with an exchange step after every cycle: n_cycles times { amh_run for one cycle
 * (sched->n_global + sched->n_local sweeps, sweep_offset = cycle * that) at the chains' current temperatures;
 * amh_exchange on the sweep-end energies }, all enqueued on the stream, nothing synchronised.
 *   per_chain_T  DEVICE float [B], in/out (the temperatures each row holds at the end)
 *   energy       DEVICE float [B], required: V of the final states (also the scratch the exchange reads)
 *   best_energy  DEVICE float [B] or NULL: min over all sweep ends of the call
 *   n_tried, n_accepted  DEVICE unsigned long long [1] or NULL; reset to 0 by the call */
amh_status amh_run_pt(amh_ctx *ctx, float *states, long long B, long long n_cycles, long long cycle_offset,
                      long long chain_offset, const amh_schedule *sched, float *per_chain_T, int replicas,
                      const amh_proposal *prop, unsigned long long seed, float *energy, float *best_energy,
                      unsigned long long *n_tried, unsigned long long *n_accepted, void *cuda_stream);

/* amh_run_pt for callers that must not allocate device memory while they sample.
 *
 * amh_run_pt keeps one float per chain between a cycle's sweep kernel (which writes the cycle's best energy there) and
 * the kernel that folds it into best_energy; it takes that room from the context's staging arena, which it grows with
 * cudaMalloc (and cudaFree of the old arena) whenever a larger batch arrives.  Three kinds of caller cannot afford
 * that inside their sampling loop:
 *   - a sampler sharing the GPU with a framework whose caching allocator has already claimed nearly all of HBM
 *     (PyTorch next to a resident model): a raw cudaMalloc then fails, or succeeds only after the framework is made
 *     to hand blocks back;
 *   - a service with a latency budget: cudaMalloc and cudaFree serialise against the whole device, so one call
 *     stalls every other stream of the process, not just ours;
 *   - code running under a "no allocation after start-up" rule (a fixed memory plan checked at start, or a region
 *     in which the runtime refuses allocation calls outright).
 * This entry point does the same work, enqueues the same kernels in the same order and leaves the same results, but
 * its per-cycle scratch is a fixed array compiled into the library (file-scope __device__ storage,
 * AMH_RUN_PT_STATIC_MAX_CHAINS floats = 256 KiB; every GPU on which the library is loaded carries it until the process
 * exits).  It calls no cudaMalloc, no cudaFree and no library routine that allocates; the context itself is still
 * built by amh_create, at start-up.
 *
 * Arguments, layouts and results: exactly amh_run_pt's (states, per_chain_T, energy, best_energy, n_tried, n_accepted
 * are the caller's DEVICE buffers).  Differences:
 *   - B > AMH_RUN_PT_STATIC_MAX_CHAINS returns AMH_ERR_UNSUPPORTED (amh_last_error names the limit) and enqueues
 *     nothing.  Split a larger batch into several calls with chain_offset, one after the other.
 *   - The device current at the call must be the one the context was created on (INVALID_ARG otherwise).
 *   - The first call on each device looks up the array's device address (cudaGetSymbolAddress; it may also make the
 *     runtime load the library's kernels).  Make that first call during start-up, before any stream capture begins
 *     anywhere in the process.  Later calls on that device reuse the address.
 *   - The array is shared by every call and every context of the process on that device, and keeps what the last
 *     call left in it.  Nothing in it has to start at zero: each cycle's sweep kernel overwrites entries [0, B)
 *     before they are read, so no call sees another's values - PROVIDED calls do not overlap on the GPU.  Two
 *     calls in flight at once on different streams (or from different threads) race on it; order them on one
 *     stream or with events. */
#define AMH_RUN_PT_STATIC_MAX_CHAINS 65536
amh_status amh_run_pt_static(amh_ctx *ctx, float *states, long long B, long long n_cycles, long long cycle_offset,
                             long long chain_offset, const amh_schedule *sched, float *per_chain_T, int replicas,
                             const amh_proposal *prop, unsigned long long seed, float *energy, float *best_energy,
                             unsigned long long *n_tried, unsigned long long *n_accepted, void *cuda_stream);

/* The same call on HOST buffers: states, temp->per_chain_T and every pointer in *out are host memory.
 * Copies in, runs, copies out and synchronises the stream; device staging buffers are owned by the
 * context and grow on demand. */
amh_status amh_run_host(amh_ctx *ctx, float *states, long long B, long long n_sweeps, long long sweep_offset,
                        long long chain_offset, const amh_schedule *sched, const amh_temperature *temp,
                        const amh_proposal *prop, unsigned long long seed, const amh_outputs *out,
                        void *cuda_stream);

/* HOST-buffer energy: states host float [B][n] -> energy_out host float [B]; synchronises. */
amh_status amh_energy_host(amh_ctx *ctx, const float *states, long long B, float *energy_out, void *cuda_stream);

/* Launch shape amh_run would use for a batch of B rows and a schedule with this window: threads per
 * chain-CTA, dynamic shared memory bytes per CTA, CTAs resident per SM, SM count.  Any pointer may be
 * NULL.  Host. */
amh_status amh_launch_info(amh_ctx *ctx, long long B, int window, int *threads_per_chain, int *smem_bytes,
                           int *ctas_per_sm, int *n_sm);

/* The rest of the launch shape: chains per CTA, warps per chain, slots and rows per slot of the table
 * ring (0, 0 = ring off).  Any pointer may be NULL.  Host. */
amh_status amh_launch_shape(amh_ctx *ctx, long long B, int window, int *chains_per_cta, int *warps_per_chain,
                            int *ring_cols, int *ring_rows);

/* Test hook (pin P0 on the device): out[q][0..3] = Philox4x32-10(ctr[q][0..3], key[q][0..1]).
 * ctr: DEVICE uint32 [count][4]; key: DEVICE uint32 [count][2]; out: DEVICE uint32 [count][4]. */
amh_status amh_philox_test(const unsigned int *ctr, const unsigned int *key, unsigned int *out,
                           long long count, void *cuda_stream);

/* Measurement hooks (SURVEY.md 8(d) "BW_L2 is not in MEASURED_PEAKS.json - measure it"): the two
 * memory ceilings of the pair loops on the current device.  Both allocate a scratch buffer, run their kernel `reps` times
 * (after one warm-up), time it with CUDA events on the stream, free the buffer and synchronise.  Host outputs.
 *   amh_probe_l2_read   every SM sweeps a buffer of `bytes` with 16-byte loads that bypass L1: *gb_per_s = bytes read
 *                       from L2 (all SMs together) / time.  bytes <= L2 size measures L2 -> SM bandwidth, larger
 *                       buffers fall to HBM.
 *   amh_probe_gather    8-byte gathers at pseudo-random entries of a table of `bytes` (a power of two is used):
 *                       *gathers_per_s.  This is the ceiling of the near-pair table look-ups of the global phase
 *                       (one L1 wavefront per lane: about one gather per clock and SM whatever the table size in L2). */
amh_status amh_probe_l2_read(long long bytes, int reps, double *gb_per_s, void *cuda_stream);
amh_status amh_probe_gather(long long bytes, int reps, double *gathers_per_s, void *cuda_stream);

/* Which variant of the sweep kernel amh_run would launch for a batch of B rows and this window (for reports):
 * spec_global 1 = one warp per global proposal, ring 1 = shared-memory table ring on, cb64 1 = fp64 C-betas kept in
 * shared memory, nspec = local proposals per pass, lanes = lanes per local proposal.  Any pointer may be NULL.  Host. */
amh_status amh_launch_variant(amh_ctx *ctx, long long B, int window, int *spec_global, int *ring, int *cb64, int *nspec, int *lanes);

/* Checked build only (python -m paper_2211_03193_b200.build --checked: every table, ring and shared-memory index of the
 * pair loops is range-checked on the device): *code = 0 if no check has failed since the library was loaded, else the
 * largest code of a failed check; *checked = 1 in a checked build, 0 in the product build (whose *code stays 0).
 * Synchronises the device.  Host outputs. */
amh_status amh_check_status(int *code, int *checked);

const char *amh_last_error(void);
const char *amh_version(void);

#ifdef __cplusplus
}
#endif
#endif /* AMH_H_ */
