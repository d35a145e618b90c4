/*
 * amh_oracle.c - plain, slow, fp64 CPU statement of the Alternating Metropolis-Hastings hot path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may call it.  It shares no code, header,
 * table or constant generator with the CUDA path under paper_2211_03193_b200/csrc/.
 *
 * What it follows (PAPER.md = /root/reference/PAPER.md, arXiv 2211.03193; readings Rn = DESIGN.md):
 *   - state s, n = 2r variables, s_even = phi, s_odd = psi            PAPER.md:25, Fig. 2 (:67)   R15
 *   - x = G(s): C-beta coordinates from the torsions                  PAPER.md:39, 77             R1-R3
 *   - V(x)      = -sum log P(|x_i - x_j|)                Eq. 3a       PAPER.md:75                 R8, R9
 *   - V_local(x,k,d): same sum restricted to the window  Eq. 3b       PAPER.md:81-86              R12
 *   - accept with min[1, P(s')/P(s)], P = e^{-V}         Eq. 1a/1c, 2a/2b  PAPER.md:27-49         R14
 *   - cycles of N_global then N_local sweeps, k = 0..n-1 Alg. 1       PAPER.md:97-123, 129        R10
 *   - inverse temperature beta in the acceptance                      PAPER.md:172, 192-194       R13
 *   - minimum energy observed over a run
 * The paper's RNG (two LFSRs) is replaced by Philox4x32-10 keyed by
 * (seed, chain, step, purpose) as BASELINE.json north_star fixes (R6); the proposal is the configs'
 * uniform resampling (BASELINE.json:7, R5) with the paper's Gaussian single flip (PAPER.md:25, 31,
 * 129) as a second mode.
 *
 * Every proposal rebuilds ALL coordinates from the torsions and re-sums the FULL global or window
 * energy of both the current and the proposed state - the plain definitions, none of the GPU's
 * shortcuts (no rotation of one side, no cross-pair difference, no cached energies).
 *
 * Parity pins: tests/test_oracle_*.py (P0-P7 of DESIGN.md).  Parity unpinned: the ideal bond-angle
 * and C-beta constants of R2/R3 (any self-consistent choice passes every pin).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ------------------------------------------------------------------------------------------- */
/* Philox4x32-10 (Salmon et al., SC'11), written from the algorithm description.  R6, pin P0.   */
/* ------------------------------------------------------------------------------------------- */
void amho_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int r = 0; r < 10; ++r) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

enum { AMHO_PURPOSE_PROPOSAL = 0, AMHO_PURPOSE_ACCEPT = 1 };
enum { AMHO_PROP_UNIFORM = 0, AMHO_PROP_GRID = 1, AMHO_PROP_GAUSSIAN = 2 };

static void draw(uint64_t seed, uint64_t chain, uint64_t step, uint32_t purpose, uint32_t out[4])
{
    /* R6: key = (seed_lo, seed_hi); counter = (step_lo, step_hi, chain, purpose) */
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    uint32_t ctr[4] = { (uint32_t)step, (uint32_t)(step >> 32), (uint32_t)chain, purpose };
    amho_philox4x32_10(ctr, key, out);
}

/* ------------------------------------------------------------------------------------------- */
/* Geometry  x = G(s)   (R1-R3)                                                 */
/* ------------------------------------------------------------------------------------------- */
typedef struct {
    double len_n_ca, len_ca_c, len_c_n;          /* A   (BASELINE.json:7) */
    double ang_n_ca_c, ang_ca_c_n, ang_c_n_ca;   /* rad (R2) */
    double omega;                                /* rad (BASELINE.json:7: 180 deg) */
    double cb_len, cb_ang, cb_dih;               /* R3: |CA-CB|, angle N-CA-CB, dihedral C-N-CA-CB */
    double eps;                                  /* 1e-8 inside the log (BASELINE.json:7) */
    int    min_sep;                              /* pairs need j - i >= min_sep (R9) */
    int    pad_;
} amho_geom;

void amho_default_geom(amho_geom *g)
{
    g->len_n_ca = 1.458; g->len_ca_c = 1.525; g->len_c_n = 1.329;
    g->ang_n_ca_c = 1.9408061282176943;   /* 111.2 deg */
    g->ang_ca_c_n = 2.028072590817411;    /* 116.2 deg */
    g->ang_c_n_ca = 2.124065699677099;    /* 121.7 deg */
    g->omega = 3.141592653589793;
    g->cb_len = 1.522; g->cb_ang = 1.927; g->cb_dih = -2.143;
    g->eps = 1e-8; g->min_sep = 3; g->pad_ = 0;
}

static void sub3(const double a[3], const double b[3], double o[3]) { o[0]=a[0]-b[0]; o[1]=a[1]-b[1]; o[2]=a[2]-b[2]; }
static void cross3(const double a[3], const double b[3], double o[3])
{
    o[0] = a[1]*b[2] - a[2]*b[1];
    o[1] = a[2]*b[0] - a[0]*b[2];
    o[2] = a[0]*b[1] - a[1]*b[0];
}
static void unit3(double a[3]) { double r = sqrt(a[0]*a[0] + a[1]*a[1] + a[2]*a[2]); a[0]/=r; a[1]/=r; a[2]/=r; }

/* place(a,b,c; len, ang, tor): the point d with |c-d| = len, angle b-c-d = ang and IUPAC dihedral
 * a-b-c-d = tor (natural extension reference frame, R1). */
static void place(const double a[3], const double b[3], const double c[3],
                  double len, double ang, double tor, double d[3])
{
    double bc[3], ab[3], nrm[3], m[3];
    sub3(c, b, bc); unit3(bc);
    sub3(b, a, ab);
    cross3(ab, bc, nrm); unit3(nrm);
    cross3(nrm, bc, m);
    double dx = -len * cos(ang);
    double dy =  len * sin(ang) * cos(tor);
    double dz =  len * sin(ang) * sin(tor);
    for (int q = 0; q < 3; ++q) d[q] = c[q] + dx * bc[q] + dy * m[q] + dz * nrm[q];
}

/* Sequential NeRF in the canonical frame of R1/R4.  s = [phi_0, psi_0, phi_1, psi_1, ...] (R15),
 * radians (R16).  N, CA, C, CB are [L][3]; any of them may be NULL except that all three backbone
 * arrays are needed internally (scratch is allocated when NULL). */
void amho_coords(const amho_geom *g, int L, const float *s, double *N, double *CA, double *C, double *CB)
{
    if (L <= 0) return;
    double *own = NULL;
    if (!N || !CA || !C) {
        own = (double *)malloc(sizeof(double) * 9 * (size_t)L);
        if (!N) N = own; if (!CA) CA = own + 3 * (size_t)L; if (!C) C = own + 6 * (size_t)L;
    }
    N[0] = 0; N[1] = 0; N[2] = 0;
    CA[0] = g->len_n_ca; CA[1] = 0; CA[2] = 0;
    C[0] = CA[0] - g->len_ca_c * cos(g->ang_n_ca_c);      /* angle N-CA-C at CA, C in the xy plane, y > 0 */
    C[1] = g->len_ca_c * sin(g->ang_n_ca_c);
    C[2] = 0;
    for (int i = 0; i + 1 < L; ++i) {
        double psi_i  = (double)s[2 * i + 1];
        double phi_n  = (double)s[2 * (i + 1)];
        place(N  + 3*i, CA + 3*i, C  + 3*i,         g->len_c_n,  g->ang_ca_c_n, psi_i,    N  + 3*(i+1));
        place(CA + 3*i, C  + 3*i, N  + 3*(i+1),     g->len_n_ca, g->ang_c_n_ca, g->omega, CA + 3*(i+1));
        place(C  + 3*i, N  + 3*(i+1), CA + 3*(i+1), g->len_ca_c, g->ang_n_ca_c, phi_n,    C  + 3*(i+1));
    }
    if (CB)
        for (int i = 0; i < L; ++i)     /* R3: CB_i = place(C_i, N_i, CA_i; cb_len, cb_ang, cb_dih) */
            place(C + 3*i, N + 3*i, CA + 3*i, g->cb_len, g->cb_ang, g->cb_dih, CB + 3*i);
    free(own);
}

/* ------------------------------------------------------------------------------------------- */
/* Energy  (Eq. 3a / 3b; R8, R9, R12)                                       */
/* ------------------------------------------------------------------------------------------- */
typedef struct {
    int L, nb;
    const double *E;       /* [L][L][nb], E = -log(p + eps) */
    double c0, delta;      /* first bin centre, bin width */
    amho_geom g;
} amho_model;

/* E[i][j][b] = -log((double)p_f32 + eps)   (Eq. 3a with BASELINE.json:7's 1e-8) */
void amho_table(const float *p, long long count, double eps, double *E)
{
    for (long long q = 0; q < count; ++q) E[q] = -log((double)p[q] + eps);
}

/* R8: linear interpolation of the -log values between bin centres, constant beyond the end centres */
double amho_pair(const double *Erow, int nb, double c0, double delta, double d)
{
    double t = (d - c0) / delta;
    if (t < 0.0) t = 0.0;
    if (t > (double)(nb - 1)) t = (double)(nb - 1);
    int b = (int)floor(t);
    if (b > nb - 2) b = nb - 2;
    double f = t - (double)b;
    return Erow[b] + f * (Erow[b + 1] - Erow[b]);
}

static double dist3(const double *a, const double *b)
{
    double x = a[0]-b[0], y = a[1]-b[1], z = a[2]-b[2];
    return sqrt(x*x + y*y + z*z);
}

/* V restricted to residues lo..hi inclusive: sum over lo <= i < j <= hi, j - i >= min_sep */
static double energy_range(const amho_model *m, const double *CB, int lo, int hi)
{
    double v = 0.0;
    for (int i = lo; i <= hi; ++i)
        for (int j = i + m->g.min_sep; j <= hi; ++j)
            v += amho_pair(m->E + ((size_t)i * m->L + j) * m->nb, m->nb, m->c0, m->delta,
                           dist3(CB + 3*i, CB + 3*j));
    return v;
}

double amho_energy_cb(const amho_model *m, const double *CB) { return energy_range(m, CB, 0, m->L - 1); }

/* Eq. 3b with R12: residue c = floor(k/2), window c-w .. c+w inclusive, clamped at the chain ends */
double amho_energy_local_cb(const amho_model *m, const double *CB, int k, int w)
{
    int c = k / 2;
    int lo = c - w < 0 ? 0 : c - w;
    int hi = c + w > m->L - 1 ? m->L - 1 : c + w;
    return energy_range(m, CB, lo, hi);
}

double amho_energy(const amho_model *m, const float *s)
{
    double *CB = (double *)malloc(sizeof(double) * 3 * (size_t)m->L);
    amho_coords(&m->g, m->L, s, NULL, NULL, NULL, CB);
    double v = amho_energy_cb(m, CB);
    free(CB);
    return v;
}

double amho_energy_local(const amho_model *m, const float *s, int k, int w)
{
    double *CB = (double *)malloc(sizeof(double) * 3 * (size_t)m->L);
    amho_coords(&m->g, m->L, s, NULL, NULL, NULL, CB);
    double v = amho_energy_local_cb(m, CB, k, w);
    free(CB);
    return v;
}

void amho_energy_batch(const amho_model *m, const float *states, long long B, double *out, int n_threads)
{
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
    long long n = 2LL * m->L;
    #pragma omp parallel for schedule(dynamic, 1)
    for (long long b = 0; b < B; ++b) out[b] = amho_energy(m, states + b * n);
}

/* ------------------------------------------------------------------------------------------- */
/* Alternating MH  (Alg. 1)                                                     */
/* ------------------------------------------------------------------------------------------- */
typedef struct {
    long long n_sweeps, sweep_offset;     /* absolute sweep index t runs over [offset, offset+n_sweeps) */
    int n_global, n_local, window, global_first;   /* R10, R12 */
    double t_start, t_end;                /* R13: geometric per sweep over ramp_sweeps; equal => constant */
    long long ramp_sweeps;
    const float *per_chain_T;             /* [B] or NULL; overrides the ramp (cfg 4) */
    int prop_mode, grid;                  /* R5 */
    double sigma_start, sigma_end;        /* Gaussian mode: sigma_t geometric-free linear ramp over ramp_sigma sweeps (rad) */
    long long ramp_sigma;
    unsigned long long seed;
    long long chain_offset;               /* chain id used by the RNG = chain_offset + row */
    int only_k;                           /* test hook (pin P5 iii): propose only this variable; -1 = all */
    int trace_steps;                      /* first trace_steps proposals of the call are traced */
    int n_threads;                        /* OpenMP threads over chains; <= 0 = default */
    int local_stride;                     /* NEXT-4: 0 = Alg. 1's order k = 0..n-1; s > 0 = the strided order of local sweeps */
} amho_run_params;

typedef struct {                          /* every pointer optional */
    double *energy;                       /* [B] global energy of the final state */
    double *best_energy;                  /* [B] min over sweep ends of this call */
    float  *best_state;                   /* [B][n] */
    long long *n_accept_local, *n_accept_global, *n_prop_local, *n_prop_global;   /* [B] */
    double *sweep_energy;                 /* [B][n_sweeps] global energy at every sweep end */
    float  *trace_prop;                   /* [B][trace_steps] proposed value s'_k */
    double *trace_dE;                     /* [B][trace_steps] */
    double *trace_g;                      /* [B][trace_steps] near-tie gap g = log u + dE/T (R14) */
    unsigned char *trace_acc;             /* [B][trace_steps] */
} amho_outputs;

static int phase_is_global(const amho_run_params *p, long long t)
{
    long long cyc = (long long)p->n_global + p->n_local;
    long long r = t % cyc;
    if (p->global_first) return r < p->n_global;
    return r >= p->n_local;
}

double amho_temperature(const amho_run_params *p, long long t, long long row)
{
    if (p->per_chain_T) return (double)p->per_chain_T[row];
    if (p->t_start == p->t_end || p->ramp_sweeps <= 1 || t <= 0) return p->t_start;
    if (t >= p->ramp_sweeps - 1) return p->t_end;
    return p->t_start * pow(p->t_end / p->t_start, (double)t / (double)(p->ramp_sweeps - 1));
}

static double sigma_at(const amho_run_params *p, long long t)
{
    if (p->sigma_start == p->sigma_end || p->ramp_sigma <= 1 || t <= 0) return p->sigma_start;
    if (t >= p->ramp_sigma - 1) return p->sigma_end;
    return p->sigma_start + (p->sigma_end - p->sigma_start) * ((double)t / (double)(p->ramp_sigma - 1));
}

/* NEXT-4 (PAPER.md:105, 114 give the order being changed): the variable visited at position p of a sweep.
 * Alg. 1 (stride <= 0, and every global sweep): k = p.  Strided local sweep with stride s: the residues are visited in
 * colour classes o = 0 .. s-1 (c = o, o + s, o + 2s, ...), both variables of a residue in turn (phi_c, then psi_c).  With
 * s >= 2w + 1 the windows of the residues of one class do not overlap, so their proposals do not interact: an accepted
 * move turns everything right of it rigidly and leaves every other window's internal distances unchanged (R26). */
int amho_sweep_order(int p, int is_global, int L, int stride)
{
    if (is_global || stride <= 0) return p;
    int r = p / 2;
    const int par = p % 2;
    for (int o = 0; o < stride && o < L; ++o) {
        const int cnt = (L - o + stride - 1) / stride;
        if (r < cnt) return 2 * (o + r * stride) + par;
        r -= cnt;
    }
    return p;
}

/* R5: the proposed value for variable k.  UNIFORM and GRID are a single IEEE fp32 operation chain
 * on integers, so an fp32 implementation reproduces them bit for bit. */
static float propose(const amho_run_params *p, uint64_t chain, uint64_t step, long long t, float s_k)
{
    uint32_t x[4];
    draw(p->seed, chain, step, AMHO_PURPOSE_PROPOSAL, x);
    const float pi_f = 3.14159274101257324f;
    if (p->prop_mode == AMHO_PROP_UNIFORM) {
        int32_t h = (int32_t)(x[0] >> 8) - (1 << 23);          /* h * 2^-23 in [-1, 1) exactly */
        float a = (float)h * 1.1920928955078125e-07f;
        return (float)((double)a * (double)pi_f);               /* one fp32 rounding of an exact product */
    }
    if (p->prop_mode == AMHO_PROP_GRID) {
        int32_t m = (int32_t)(x[0] % (uint32_t)p->grid);
        float a = (float)((double)(2 * m - p->grid) / (double)p->grid);   /* fp32 division, correctly rounded */
        return (float)((double)a * (double)pi_f);
    }
    /* GAUSSIAN: Box-Muller, added to s_k, wrapped to [-pi, pi) */
    double u1 = ((double)(x[0] >> 8) + 1.0) * 5.9604644775390625e-08;   /* (0,1] */
    double u2 = (double)(x[1] >> 8) * 5.9604644775390625e-08;          /* [0,1) */
    double z = sqrt(-2.0 * log(u1)) * cos(6.283185307179586 * u2);
    double v = (double)s_k + sigma_at(p, t) * z;
    v -= 6.283185307179586 * floor((v + 3.141592653589793) / 6.283185307179586);
    float vf = (float)v;
    if (vf >= pi_f) vf -= 2.0f * pi_f;
    return vf;
}

static double uniform01(const amho_run_params *p, uint64_t chain, uint64_t step)
{
    uint32_t x[4];
    draw(p->seed, chain, step, AMHO_PURPOSE_ACCEPT, x);
    return ((double)(x[0] >> 8) + 1.0) * 5.9604644775390625e-08;   /* R7: ((x0>>8)+1) * 2^-24 in (0,1] */
}

/* One proposal from the current state s (length n): returns dE and the proposed value; the caller
 * takes the decision.  Both states are rebuilt from scratch and fully re-summed. */
static double proposal_dE(const amho_model *m, const amho_run_params *p, int is_global, int k,
                          float *s, float s_new, double *CB, double *CBn)
{
    amho_coords(&m->g, m->L, s, NULL, NULL, NULL, CB);
    float keep = s[k];
    s[k] = s_new;
    amho_coords(&m->g, m->L, s, NULL, NULL, NULL, CBn);
    s[k] = keep;
    if (is_global) return amho_energy_cb(m, CBn) - amho_energy_cb(m, CB);
    return amho_energy_local_cb(m, CBn, k, p->window) - amho_energy_local_cb(m, CB, k, p->window);
}

/* Free-running AMH over B chains.  states is [B][n], in/out. */
int amho_run(const amho_model *m, const amho_run_params *p, float *states, long long B, const amho_outputs *o)
{
    const int L = m->L, n = 2 * L;
    if (L < 1 || B < 0 || p->n_global + p->n_local <= 0 || p->window < 0) return 1;
#ifdef _OPENMP
    if (p->n_threads > 0) omp_set_num_threads(p->n_threads);
#endif
    #pragma omp parallel
    {
        double *CB  = (double *)malloc(sizeof(double) * 3 * (size_t)L);
        double *CBn = (double *)malloc(sizeof(double) * 3 * (size_t)L);
        #pragma omp for schedule(dynamic, 1)
        for (long long row = 0; row < B; ++row) {
            float *s = states + row * n;
            const uint64_t chain = (uint64_t)(p->chain_offset + row);
            long long acc_l = 0, acc_g = 0, prop_l = 0, prop_g = 0, traced = 0;
            double best = INFINITY, e_end = NAN;
            for (long long t = p->sweep_offset; t < p->sweep_offset + p->n_sweeps; ++t) {
                const int is_global = phase_is_global(p, t);
                const double T = amho_temperature(p, t, row);
                for (int pos = 0; pos < n; ++pos) {
                    const int k = amho_sweep_order(pos, is_global, L, p->local_stride);
                    if (p->only_k >= 0 && k != p->only_k) continue;
                    const uint64_t step = (uint64_t)t * (uint64_t)n + (uint64_t)k;
                    const float s_new = propose(p, chain, step, t, s[k]);
                    const double dE = proposal_dE(m, p, is_global, k, s, s_new, CB, CBn);
                    const double lu = log(uniform01(p, chain, step));
                    const int accept = lu <= -dE / T;                 /* R14 */
                    if (traced < p->trace_steps) {
                        size_t q = (size_t)row * p->trace_steps + traced;
                        if (o->trace_prop) o->trace_prop[q] = s_new;
                        if (o->trace_dE)   o->trace_dE[q] = dE;
                        if (o->trace_g)    o->trace_g[q] = lu + dE / T;
                        if (o->trace_acc)  o->trace_acc[q] = (unsigned char)accept;
                        ++traced;
                    }
                    if (is_global) { ++prop_g; acc_g += accept; } else { ++prop_l; acc_l += accept; }
                    if (accept) s[k] = s_new;
                }
                e_end = amho_energy(m, s);                            /* book-keeping at the sweep end */
                if (o->sweep_energy) o->sweep_energy[(size_t)row * p->n_sweeps + (t - p->sweep_offset)] = e_end;
                if (e_end < best) {
                    best = e_end;
                    if (o->best_state) memcpy(o->best_state + row * n, s, sizeof(float) * n);
                }
            }
            if (p->n_sweeps == 0) e_end = amho_energy(m, s);
            if (o->energy) o->energy[row] = e_end;
            if (o->best_energy) o->best_energy[row] = best;
            if (o->n_accept_local)  o->n_accept_local[row]  = acc_l;
            if (o->n_accept_global) o->n_accept_global[row] = acc_g;
            if (o->n_prop_local)    o->n_prop_local[row]    = prop_l;
            if (o->n_prop_global)   o->n_prop_global[row]   = prop_g;
        }
        free(CB); free(CBn);
    }
    return 0;
}

/* Follow mode: replay the first `steps` proposals of
 * a run with sweep_offset as given, taking at every step the decision in `forced_acc` (the other
 * implementation's accept bits) while recording this implementation's own proposal, dE, gap g and
 * decision from the SHARED current state.  states is [B][n], in/out (ends at the forced path).
 * forced_prop (may be NULL): the other implementation's proposed values.  DESIGN.md R5: a Gaussian
 * proposal goes through log/sqrt/cos, which two math libraries round differently in the last place,
 * so there the replay is teacher-forced - this implementation still records its OWN proposal in
 * own_prop (the test checks it within 2 ulp) but evaluates and applies the forced value, so that
 * both stay on one path.  For UNIFORM and GRID the two are bit-identical and NULL is passed. */
int amho_follow(const amho_model *m, const amho_run_params *p, float *states, long long B, int steps,
                const unsigned char *forced_acc, const float *forced_prop, float *own_prop, double *own_dE,
                double *own_g, unsigned char *own_acc)
{
    const int L = m->L, n = 2 * L;
    if (L < 1 || p->n_global + p->n_local <= 0) return 1;
#ifdef _OPENMP
    if (p->n_threads > 0) omp_set_num_threads(p->n_threads);
#endif
    #pragma omp parallel
    {
        double *CB  = (double *)malloc(sizeof(double) * 3 * (size_t)L);
        double *CBn = (double *)malloc(sizeof(double) * 3 * (size_t)L);
        #pragma omp for schedule(dynamic, 1)
        for (long long row = 0; row < B; ++row) {
            float *s = states + row * n;
            const uint64_t chain = (uint64_t)(p->chain_offset + row);
            for (int q = 0; q < steps; ++q) {
                const uint64_t at = (uint64_t)p->sweep_offset * (uint64_t)n + (uint64_t)q;
                const long long t = (long long)(at / (uint64_t)n);
                const int is_global = phase_is_global(p, t);
                const int k = amho_sweep_order((int)(at % (uint64_t)n), is_global, L, p->local_stride);
                const uint64_t step = (uint64_t)t * (uint64_t)n + (uint64_t)k;      /* the draws are keyed by the variable */
                const double T = amho_temperature(p, t, row);
                size_t z = (size_t)row * steps + q;
                const float s_own = propose(p, chain, step, t, s[k]);
                const float s_new = forced_prop ? forced_prop[z] : s_own;
                const double dE = proposal_dE(m, p, is_global, k, s, s_new, CB, CBn);
                const double lu = log(uniform01(p, chain, step));
                own_prop[z] = s_own; own_dE[z] = dE; own_g[z] = lu + dE / T;
                own_acc[z] = (unsigned char)(lu <= -dE / T);
                if (forced_acc[z]) s[k] = s_new;
            }
        }
        free(CB); free(CBn);
    }
    return 0;
}

int amho_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* =========================================================================================== */
/* NEXT-2: config 3, trRosetta2-style energy on a 5-slot state (BASELINE.json:11; R25) */
/* =========================================================================================== */
/*
 * The paper says only that "trRosetta2 follows a 5 angle parameterization" whose
 * inter-residue geometry is "(phi, theta, omega)" and that "once the information is
 * captured in the angle vector (s), the remaining procedure is unchanged".  Reading R25:
 *   state   n = 5L, s[5i+0] = phi_i, s[5i+1] = psi_i, s[5i+2] = omega_i (the torsion of the peptide bond
 *           C_i - N_{i+1}, a variable here instead of the constant 180 degrees of R1), s[5i+3], s[5i+4] = two
 *           slots that move no backbone atom and no C-beta (their proposals have dE = 0: always accepted)
 *   energy  V = sum over i < j, j - i >= min_sep of
 *             e_d(|CB_i CB_j|)                                   37 bins over 2-20 A, R8's interpolation and clamp
 *           + e_o(dihedral CA_i, CB_i, CB_j, CA_j)               24 bins over [-pi, pi), periodic, symmetric
 *           + e_t[i][j](dihedral N_i, CA_i, CB_i, CB_j) + e_t[j][i](dihedral N_j, CA_j, CB_j, CB_i)   24 bins, periodic
 *           + e_p[i][j](angle CA_i, CB_i, CB_j) + e_p[j][i](angle CA_j, CB_j, CB_i)                  12 bins over [0, pi], clamped
 *           every e = -log(p + eps) interpolated linearly between bin centres (circularly for the periodic ones)
 *   window  residue of variable k is floor(k/5); Eq. 3b and R12 unchanged
 * Parity unpinned: the CHOICE of the parameterisation and of the orientation conventions (the paper fixes neither).
 * That amho_tr5_pair_geometry computes the conventions written above - which atoms, which order, which sign - is
 * pinned by P16 (tests/test_oracle_tr5.py: two residues placed by hand, values derived from the coordinates).
 */
typedef struct {
    int L, nb_d, nb_o, nb_t, nb_p;
    const double *Ed;      /* [L][L][nb_d]  i < j read */
    const double *Eo;      /* [L][L][nb_o]  i < j read */
    const double *Et;      /* [L][L][nb_t]  ordered: row (i, j) scores the dihedral seen from residue i */
    const double *Ep;      /* [L][L][nb_p]  ordered */
    double c0, delta;      /* distance bins: first centre, width */
    amho_geom g;
} amho_tr5_model;

static double dot3(const double a[3], const double b[3]) { return a[0]*b[0] + a[1]*b[1] + a[2]*b[2]; }

/* IUPAC dihedral a-b-c-d in (-pi, pi]: the angle between the projections of a-b and d-c on the plane normal to b-c */
double amho_dihedral(const double a[3], const double b[3], const double c[3], const double d[3])
{
    double b0[3], b1[3], b2[3], v[3], w[3], x[3];
    sub3(a, b, b0); sub3(c, b, b1); sub3(d, c, b2);
    unit3(b1);
    double p0 = dot3(b0, b1), p2 = dot3(b2, b1);
    for (int q = 0; q < 3; ++q) { v[q] = b0[q] - p0 * b1[q]; w[q] = b2[q] - p2 * b1[q]; }
    cross3(b1, v, x);
    return atan2(dot3(x, w), dot3(v, w));
}

/* angle a-b-c at b in [0, pi] */
double amho_angle(const double a[3], const double b[3], const double c[3])
{
    double u[3], v[3];
    sub3(a, b, u); sub3(c, b, v);
    double q = dot3(u, v) / sqrt(dot3(u, u) * dot3(v, v));
    if (q > 1.0) q = 1.0;
    if (q < -1.0) q = -1.0;
    return acos(q);
}

/* periodic table over [-pi, pi): bin centres -pi + (b + 1/2) 2 pi / nb, circular linear interpolation */
double amho_interp_periodic(const double *Erow, int nb, double x)
{
    const double two_pi = 6.283185307179586, delta = two_pi / nb;
    double t = (x + 3.141592653589793) / delta - 0.5;
    double fl = floor(t);
    double f = t - fl;
    long b = (long)fl % nb;
    if (b < 0) b += nb;
    long b1 = (b + 1) % nb;
    return Erow[b] + f * (Erow[b1] - Erow[b]);
}

void amho_tr5_coords(const amho_geom *g, int L, const float *s, double *N, double *CA, double *C, double *CB)
{
    if (L <= 0) return;
    N[0] = 0; N[1] = 0; N[2] = 0;
    CA[0] = g->len_n_ca; CA[1] = 0; CA[2] = 0;
    C[0] = CA[0] - g->len_ca_c * cos(g->ang_n_ca_c);
    C[1] = g->len_ca_c * sin(g->ang_n_ca_c);
    C[2] = 0;
    for (int i = 0; i + 1 < L; ++i) {
        double psi_i = (double)s[5 * i + 1], om_i = (double)s[5 * i + 2], phi_n = (double)s[5 * (i + 1)];
        place(N  + 3*i, CA + 3*i, C  + 3*i,         g->len_c_n,  g->ang_ca_c_n, psi_i, N  + 3*(i+1));
        place(CA + 3*i, C  + 3*i, N  + 3*(i+1),     g->len_n_ca, g->ang_c_n_ca, om_i,  CA + 3*(i+1));
        place(C  + 3*i, N  + 3*(i+1), CA + 3*(i+1), g->len_ca_c, g->ang_n_ca_c, phi_n, C  + 3*(i+1));
    }
    for (int i = 0; i < L; ++i)
        place(C + 3*i, N + 3*i, CA + 3*i, g->cb_len, g->cb_ang, g->cb_dih, CB + 3*i);
}

/* the four inter-residue coordinates of the ordered pair (i, j): d, omega (symmetric), theta_ij, phi_ij */
void amho_tr5_pair_geometry(const double *N, const double *CA, const double *CB, int i, int j,
                            double *d, double *omega, double *theta, double *phi)
{
    *d = dist3(CB + 3*i, CB + 3*j);
    *omega = amho_dihedral(CA + 3*i, CB + 3*i, CB + 3*j, CA + 3*j);
    *theta = amho_dihedral(N + 3*i, CA + 3*i, CB + 3*i, CB + 3*j);
    *phi = amho_angle(CA + 3*i, CB + 3*i, CB + 3*j);
}

/* one unordered pair i < j: the six terms */
double amho_tr5_pair(const amho_tr5_model *m, const double *N, const double *CA, const double *CB, int i, int j)
{
    const double pi = 3.141592653589793;
    double d, om, th_ij, ph_ij, d2, om2, th_ji, ph_ji;
    amho_tr5_pair_geometry(N, CA, CB, i, j, &d, &om, &th_ij, &ph_ij);
    amho_tr5_pair_geometry(N, CA, CB, j, i, &d2, &om2, &th_ji, &ph_ji);
    const size_t ij = (size_t)i * m->L + j, ji = (size_t)j * m->L + i;
    const double dp = pi / m->nb_p;
    double e = amho_pair(m->Ed + ij * m->nb_d, m->nb_d, m->c0, m->delta, d);
    e += amho_interp_periodic(m->Eo + ij * m->nb_o, m->nb_o, om);
    e += amho_interp_periodic(m->Et + ij * m->nb_t, m->nb_t, th_ij);
    e += amho_interp_periodic(m->Et + ji * m->nb_t, m->nb_t, th_ji);
    e += amho_pair(m->Ep + ij * m->nb_p, m->nb_p, 0.5 * dp, dp, ph_ij);
    e += amho_pair(m->Ep + ji * m->nb_p, m->nb_p, 0.5 * dp, dp, ph_ji);
    return e;
}

static double tr5_energy_range(const amho_tr5_model *m, const double *N, const double *CA, const double *CB, int lo, int hi)
{
    double v = 0.0;
    for (int i = lo; i <= hi; ++i)
        for (int j = i + m->g.min_sep; j <= hi; ++j)
            v += amho_tr5_pair(m, N, CA, CB, i, j);
    return v;
}

/* V (k < 0) or V_local(k, w) of one state; scratch = 12 L doubles */
double amho_tr5_energy(const amho_tr5_model *m, const float *s, int k, int w, double *scratch)
{
    const int L = m->L;
    double *own = scratch ? NULL : (double *)malloc(sizeof(double) * 12 * (size_t)L);
    double *N = scratch ? scratch : own, *CA = N + 3 * L, *C = CA + 3 * L, *CB = C + 3 * L;
    amho_tr5_coords(&m->g, L, s, N, CA, C, CB);
    int lo = 0, hi = L - 1;
    if (k >= 0) {
        int c = k / 5;
        lo = c - w < 0 ? 0 : c - w;
        hi = c + w > L - 1 ? L - 1 : c + w;
    }
    double v = tr5_energy_range(m, N, CA, CB, lo, hi);
    free(own);
    return v;
}

void amho_tr5_energy_batch(const amho_tr5_model *m, const float *states, long long B, double *out, int n_threads)
{
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
    long long n = 5LL * m->L;
    #pragma omp parallel for schedule(dynamic, 1)
    for (long long b = 0; b < B; ++b) out[b] = amho_tr5_energy(m, states + b * n, -1, 0, NULL);
}

static double tr5_proposal_dE(const amho_tr5_model *m, const amho_run_params *p, int is_global, int k,
                              float *s, float s_new, double *scratch)
{
    const int kk = is_global ? -1 : k;
    double v0 = amho_tr5_energy(m, s, kk, p->window, scratch);
    float keep = s[k];
    s[k] = s_new;
    double v1 = amho_tr5_energy(m, s, kk, p->window, scratch);
    s[k] = keep;
    return v1 - v0;
}

/* Alg. 1 on the 5-slot state: free-running (forced_acc == NULL) or follow mode (the first `steps` proposals
 * of a run at sweep_offset, taking the decisions in forced_acc), exactly like amho_run / amho_follow */
int amho_tr5_run(const amho_tr5_model *m, const amho_run_params *p, float *states, long long B, const amho_outputs *o)
{
    const int L = m->L, n = 5 * L;
    if (L < 1 || B < 0 || p->n_global + p->n_local <= 0 || p->window < 0) return 1;
#ifdef _OPENMP
    if (p->n_threads > 0) omp_set_num_threads(p->n_threads);
#endif
    #pragma omp parallel
    {
        double *scratch = (double *)malloc(sizeof(double) * 12 * (size_t)L);
        #pragma omp for schedule(dynamic, 1)
        for (long long row = 0; row < B; ++row) {
            float *s = states + row * n;
            const uint64_t chain = (uint64_t)(p->chain_offset + row);
            long long acc_l = 0, acc_g = 0, traced = 0;
            double best = INFINITY, e_end = NAN;
            for (long long t = p->sweep_offset; t < p->sweep_offset + p->n_sweeps; ++t) {
                const int is_global = phase_is_global(p, t);
                const double T = amho_temperature(p, t, row);
                for (int k = 0; k < n; ++k) {
                    const uint64_t step = (uint64_t)t * (uint64_t)n + (uint64_t)k;
                    const float s_new = propose(p, chain, step, t, s[k]);
                    const double dE = tr5_proposal_dE(m, p, is_global, k, s, s_new, scratch);
                    const double lu = log(uniform01(p, chain, step));
                    const int accept = lu <= -dE / T;
                    if (traced < p->trace_steps) {
                        size_t q = (size_t)row * p->trace_steps + traced;
                        if (o->trace_prop) o->trace_prop[q] = s_new;
                        if (o->trace_dE)   o->trace_dE[q] = dE;
                        if (o->trace_g)    o->trace_g[q] = lu + dE / T;
                        if (o->trace_acc)  o->trace_acc[q] = (unsigned char)accept;
                        ++traced;
                    }
                    if (is_global) acc_g += accept; else acc_l += accept;
                    if (accept) s[k] = s_new;
                }
                e_end = amho_tr5_energy(m, s, -1, 0, scratch);
                if (e_end < best) {
                    best = e_end;
                    if (o->best_state) memcpy(o->best_state + row * n, s, sizeof(float) * n);
                }
            }
            if (p->n_sweeps == 0) e_end = amho_tr5_energy(m, s, -1, 0, scratch);
            if (o->energy) o->energy[row] = e_end;
            if (o->best_energy) o->best_energy[row] = best;
            if (o->n_accept_local)  o->n_accept_local[row]  = acc_l;
            if (o->n_accept_global) o->n_accept_global[row] = acc_g;
        }
        free(scratch);
    }
    return 0;
}

int amho_tr5_follow(const amho_tr5_model *m, const amho_run_params *p, float *states, long long B, int steps,
                    const unsigned char *forced_acc, float *own_prop, double *own_dE, double *own_g, unsigned char *own_acc)
{
    const int L = m->L, n = 5 * L;
    if (L < 1 || p->n_global + p->n_local <= 0) return 1;
#ifdef _OPENMP
    if (p->n_threads > 0) omp_set_num_threads(p->n_threads);
#endif
    #pragma omp parallel
    {
        double *scratch = (double *)malloc(sizeof(double) * 12 * (size_t)L);
        #pragma omp for schedule(dynamic, 1)
        for (long long row = 0; row < B; ++row) {
            float *s = states + row * n;
            const uint64_t chain = (uint64_t)(p->chain_offset + row);
            for (int q = 0; q < steps; ++q) {
                const uint64_t step = (uint64_t)p->sweep_offset * (uint64_t)n + (uint64_t)q;
                const long long t = (long long)(step / (uint64_t)n);
                const int k = (int)(step % (uint64_t)n);
                const int is_global = phase_is_global(p, t);
                const double T = amho_temperature(p, t, row);
                size_t z = (size_t)row * steps + q;
                const float s_new = propose(p, chain, step, t, s[k]);
                const double dE = tr5_proposal_dE(m, p, is_global, k, s, s_new, scratch);
                const double lu = log(uniform01(p, chain, step));
                own_prop[z] = s_new; own_dE[z] = dE; own_g[z] = lu + dE / T;
                own_acc[z] = (unsigned char)(lu <= -dE / T);
                if (forced_acc[z]) s[k] = s_new;
            }
        }
        free(scratch);
    }
    return 0;
}
