// amh_api.cu - host side of the C ABI declared in include/amh.h: argument checks, the geometry
// constants of the bond-frame recursion, launches.  No arithmetic of the method runs on the host
// except those constants (closed forms of the ideal bond geometry, R1-R3).
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <vector>

#include "../../include/amh.h"
#include "amh_kernels.cuh"
#include "amh_sweep.cuh"
#include "amh_tr5.cuh"

namespace {

thread_local char g_err[512] = "";

amh_status fail(amh_status st, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
    return st;
}

#define AMH_CUDA(call)                                                                              \
    do {                                                                                            \
        cudaError_t e_ = (call);                                                                    \
        if (e_ != cudaSuccess)                                                                      \
            return fail(e_ == cudaErrorMemoryAllocation ? AMH_ERR_OOM : AMH_ERR_CUDA, "%s: %s", #call, \
                        cudaGetErrorString(e_));                                                    \
    } while (0)

// Mplus(ang, tor, len) of DESIGN.md "Geometry": the bond frame reached by one NeRF placement
amh::Xf mplus(double ang, double tor, double len)
{
    const double ca = std::cos(ang), sa = std::sin(ang), ct = std::cos(tor), st = std::sin(tor);
    amh::Xf M;
    M.r[0] = -ca;     M.r[1] = -sa;      M.r[2] = 0.0;
    M.r[3] = sa * ct; M.r[4] = -ca * ct; M.r[5] = -st;
    M.r[6] = sa * st; M.r[7] = -ca * st; M.r[8] = ct;
    M.t[0] = len * M.r[0]; M.t[1] = len * M.r[3]; M.t[2] = len * M.r[6];
    return M;
}

}  // namespace

struct amh_ctx {
    amh::DevModel m;
    amh_options opt;
    amh_launch_options lopt;
    float2 *Epk = nullptr;       // upper-triangle lerp table (see DevModel)
    float *Elast = nullptr;
    float *Ebd = nullptr;        // the band j - i <= band_dmax of the same E', column-major, rows padded to row_stride floats (TMA source)
    int band_dmax = 0;
    float *P = nullptr;          // the probabilities themselves (fp64 path of the exact-decision guard)
    float tab_emax = 0.0f, tab_step = 0.0f;   // max |E'| and max |E'[b+1] - E'[b]| of the table (table_kernel): scale the guard
    int param = AMH_PARAM_PHI_PSI;
    amh::Tr5Model tm;            // config 3 (AMH_PARAM_TR5): fp64 tables
    double *tE[4] = {nullptr, nullptr, nullptr, nullptr};
    int device = 0, n_sm = 0, max_smem = 0;
    // staging for the *_host calls (grow-only)
    void *stage = nullptr;
    size_t stage_bytes = 0;
};

static amh_status check_launch_options(const amh_launch_options &o)
{
    const int w = o.warps_per_chain;
    if (w < 0 || w > amh::kMaxTeamWarps)
        return fail(AMH_ERR_INVALID_ARG, "launch options: warps_per_chain = %d outside [0, %d]", w, amh::kMaxTeamWarps);
    const int cc = o.chains_per_cta;
    if (cc < 0 || cc > amh::kMaxChains)
        return fail(AMH_ERR_INVALID_ARG, "launch options: chains_per_cta = %d outside [0, %d]", cc, amh::kMaxChains);
    if (w > 0 && cc > 0 && w * cc > amh::kMaxTeamWarps)
        return fail(AMH_ERR_INVALID_ARG, "launch options: warps_per_chain * chains_per_cta = %d > %d", w * cc, amh::kMaxTeamWarps);
    if (!(o.lanes_per_step == 0 || o.lanes_per_step == 4 || o.lanes_per_step == 8 || o.lanes_per_step == 16 || o.lanes_per_step == 32))
        return fail(AMH_ERR_INVALID_ARG, "launch options: lanes_per_step = %d not in {0, 4, 8, 16, 32}", o.lanes_per_step);
    if (o.spec_local < 0 || o.spec_local > amh::kMaxSpec)
        return fail(AMH_ERR_INVALID_ARG, "launch options: spec_local = %d outside [0, %d]", o.spec_local, amh::kMaxSpec);
    return AMH_OK;
}

// ---- scratch of amh_run_pt_static (include/amh.h): the per-cycle best energies, one float per chain ---------------
// Storage that is part of the library image instead of a cudaMalloc: each GPU that loads the library holds these
// 256 KiB until the process exits.  Shared by every call on a device; see the header for what that means for callers.
static __device__ __align__(256) float amh_pt_static_scratch[AMH_RUN_PT_STATIC_MAX_CHAINS];

// In host code `amh_pt_static_scratch` is only a handle for the runtime, not something a kernel can dereference: the
// address a kernel needs comes from cudaGetSymbolAddress, differs from device to device, and is looked up once per
// device with that device current.  Host callers must never pass the bare name to a kernel.
namespace {
constexpr int kPtStaticMaxDevices = 64;
std::mutex g_pt_static_mu;
float *g_pt_static_addr[kPtStaticMaxDevices] = {};       // [device ordinal] -> device address, nullptr = not looked up yet
}  // namespace

static amh_status pt_static_scratch(int device, float **addr)
{
    if (device < 0 || device >= kPtStaticMaxDevices)
        return fail(AMH_ERR_UNSUPPORTED, "amh_run_pt_static: device ordinal %d outside [0, %d)", device, kPtStaticMaxDevices);
    std::lock_guard<std::mutex> lock(g_pt_static_mu);
    if (!g_pt_static_addr[device]) {
        void *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, amh_pt_static_scratch);     // for the CURRENT device (checked by the caller)
        if (e != cudaSuccess || !p)
            return fail(AMH_ERR_CUDA, "amh_run_pt_static: cudaGetSymbolAddress on device %d: %s", device,
                        e != cudaSuccess ? cudaGetErrorString(e) : "null address");
        g_pt_static_addr[device] = static_cast<float *>(p);
    }
    *addr = g_pt_static_addr[device];
    return AMH_OK;
}

extern "C" {

const char *amh_last_error(void) { return g_err; }
const char *amh_version(void) { return "amh-b200 0.1 (sm_100a)"; }

amh_status amh_default_options(amh_options *o)
{
    if (!o) return fail(AMH_ERR_INVALID_ARG, "amh_default_options: opt is NULL");
    o->len_n_ca = 1.458; o->len_ca_c = 1.525; o->len_c_n = 1.329;
    o->ang_n_ca_c = 111.2 * M_PI / 180.0;
    o->ang_ca_c_n = 116.2 * M_PI / 180.0;
    o->ang_c_n_ca = 121.7 * M_PI / 180.0;
    o->omega = M_PI;
    o->cb_len = 1.522; o->cb_ang = 1.927; o->cb_dih = -2.143;
    o->eps = 1e-8;
    o->guard_scale = 1.0;
    o->min_sep = 3;
    o->pad_ = 0;
    return AMH_OK;
}

amh_status amh_default_launch_options(amh_launch_options *o)
{
    if (!o) return fail(AMH_ERR_INVALID_ARG, "amh_default_launch_options: opt is NULL");
    o->warps_per_chain = 0;
    o->spec_local = 0;
    o->lanes_per_step = 0;
    o->spec_global = -1;
    o->chains_per_cta = 0;
    o->ring_cols = 0;
    return AMH_OK;
}

amh_status amh_set_launch_options(amh_ctx *c, const amh_launch_options *o)
{
    if (!c) return fail(AMH_ERR_INVALID_ARG, "amh_set_launch_options: ctx is NULL");
    amh_launch_options d;
    amh_default_launch_options(&d);
    if (o) d = *o;
    amh_status st = check_launch_options(d);
    if (st != AMH_OK) return st;
    c->lopt = d;
    return AMH_OK;
}

amh_status amh_create(amh_ctx **out, int n_res, amh_param param, const float *distogram,
                      const float *bin_edges, int n_bins, const amh_options *opt, void *cuda_stream)
{
    if (!out) return fail(AMH_ERR_INVALID_ARG, "amh_create: out is NULL");
    *out = nullptr;
    if (param == AMH_PARAM_TR5) return fail(AMH_ERR_INVALID_ARG, "amh_create: AMH_PARAM_TR5 contexts are built by amh_create_tr5 (it takes the orientation maps)");
    if (param != AMH_PARAM_PHI_PSI) return fail(AMH_ERR_INVALID_ARG, "amh_create: unknown parameterisation %d", (int)param);
    if (n_res < 1) return fail(AMH_ERR_INVALID_ARG, "amh_create: n_res = %d < 1", n_res);
    if (n_bins < 2) return fail(AMH_ERR_INVALID_ARG, "amh_create: n_bins = %d < 2", n_bins);
    if (!distogram || !bin_edges) return fail(AMH_ERR_INVALID_ARG, "amh_create: distogram / bin_edges is NULL");
    amh_options o;
    amh_default_options(&o);
    if (opt) o = *opt;
    if (o.min_sep < 1) return fail(AMH_ERR_INVALID_ARG, "amh_create: min_sep = %d < 1", o.min_sep);
    if (!(o.eps >= 0.0)) return fail(AMH_ERR_INVALID_ARG, "amh_create: eps < 0");
    if (!(o.guard_scale >= 0.0)) return fail(AMH_ERR_INVALID_ARG, "amh_create: guard_scale < 0");
    for (int b = 0; b <= n_bins; ++b)
        if (!std::isfinite(bin_edges[b])) return fail(AMH_ERR_INVALID_ARG, "amh_create: bin edge %d is not finite", b);
    const double e0 = bin_edges[0], e1 = bin_edges[n_bins];
    const double delta = (e1 - e0) / n_bins;
    if (!(delta > 0.0)) return fail(AMH_ERR_INVALID_ARG, "amh_create: bin edges do not increase");
    for (int b = 0; b < n_bins; ++b) {
        const double w = (double)bin_edges[b + 1] - (double)bin_edges[b];
        if (!(w > 0.0)) return fail(AMH_ERR_INVALID_ARG, "amh_create: bin edges do not increase at %d", b);
        if (std::fabs(w - delta) > 1e-5 * delta)
            return fail(AMH_ERR_UNSUPPORTED, "amh_create: bins are not evenly spaced (bin %d: %g vs %g)", b, w, delta);
    }

    {
        // the local pair loop addresses the packed {E', slope} table with 32-bit byte offsets, row term + column term
        // (LocalTab in amh_sweep.cuh): both terms and their sum must stay below 2^31
        const unsigned long long rows = (unsigned long long)n_res * (n_res > 0 ? n_res - 1 : 0) / 2;
        const unsigned long long reach = (rows + (unsigned long long)n_res + 1) * (unsigned long long)n_bins * 8ull;
        if (reach >= (1ull << 31))
            return fail(AMH_ERR_UNSUPPORTED, "amh_create: L = %d with n_bins = %d makes a pair table of %llu bytes; the sweep kernel "
                        "addresses it with 32-bit offsets (limit 2^31 bytes)", n_res, n_bins, rows * (unsigned long long)n_bins * 8ull);
    }

    amh_ctx *c = new (std::nothrow) amh_ctx;
    if (!c) return fail(AMH_ERR_OOM, "amh_create: host allocation failed");
    c->opt = o;
    amh_default_launch_options(&c->lopt);
    cudaError_t e = cudaGetDevice(&c->device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&c->n_sm, cudaDevAttrMultiProcessorCount, c->device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&c->max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, c->device);
    if (e != cudaSuccess) { delete c; return fail(AMH_ERR_CUDA, "amh_create: no usable CUDA device: %s", cudaGetErrorString(e)); }

    amh::DevModel &m = c->m;
    m.L = n_res; m.nb = n_bins; m.min_sep = o.min_sep; m.n = 2 * n_res;
    m.c0 = (float)(e0 + 0.5 * delta);
    m.inv_delta = (float)(1.0 / delta);
    m.tmax = (float)(n_bins - 1);
    m.thmax = (float)n_bins - 1.75f;
    m.v_far = 0.0;
    m.t0 = (float)(-(e0 + 0.5 * delta) / delta);
    {
        // smallest fp32 d^2 from which pair_energy()'s t is surely clamped to tmax: the last bin centre with a
        // relative margin far above the rounding of sqrtf, the subtraction and the scaling (all monotone in d^2)
        const double c_last = e0 + ((double)n_bins - 0.5) * delta;
        const double lim = c_last * (1.0 + 1e-5) + 1e-5 * delta;
        m.far2 = std::nextafter((float)(lim * lim), INFINITY);
        m.dfar = std::nextafter((float)std::sqrt((double)m.far2), INFINITY);
        m.far2_d = c_last * c_last * (1.0 + 1e-9);
    }
    m.c0_d = e0 + 0.5 * delta; m.delta_d = delta; m.eps_d = o.eps;
    m.A = mplus(o.ang_n_ca_c, 0.0, o.len_ca_c);
    m.W = mplus(o.ang_c_n_ca, o.omega, o.len_n_ca);
    m.c2 = std::cos(o.ang_ca_c_n); m.s2 = std::sin(o.ang_ca_c_n); m.l3 = o.len_c_n;
    // atoms in the residue's bond frame (origin CA, x along N->CA, C at torsion 0)
    m.loc[0][0] = -o.len_n_ca; m.loc[0][1] = 0.0; m.loc[0][2] = 0.0;
    m.loc[1][0] = 0.0; m.loc[1][1] = 0.0; m.loc[1][2] = 0.0;
    m.loc[2][0] = -o.len_ca_c * std::cos(o.ang_n_ca_c); m.loc[2][1] = o.len_ca_c * std::sin(o.ang_n_ca_c); m.loc[2][2] = 0.0;
    m.loc[3][0] = -o.cb_len * std::cos(o.cb_ang);
    m.loc[3][1] = o.cb_len * std::sin(o.cb_ang) * std::cos(o.cb_dih);
    m.loc[3][2] = o.cb_len * std::sin(o.cb_ang) * std::sin(o.cb_dih);
    m.h0x = o.len_n_ca;
    m.inv_len_n_ca = 1.0 / o.len_n_ca; m.inv_len_ca_c = 1.0 / o.len_ca_c;
    // the C-beta as a fixed combination of the residue's own backbone atoms (ideal geometry: C lies at loc[2] in the frame)
    m.cbA = m.loc[3][0] - m.loc[3][1] * m.loc[2][0] / m.loc[2][1];
    m.cbB = m.loc[3][1] / m.loc[2][1];
    m.cbC = m.loc[3][2] / m.loc[2][1];

    if (n_bins > (1 << 20)) { delete c; return fail(AMH_ERR_UNSUPPORTED, "amh_create: n_bins = %d > 2^20", n_bins); }
    if (amh::sweep_smem_bytes(n_res, 1, 1, 0, 0, 0, 0, 1, 1) > (size_t)c->max_smem) {
        delete c;
        return fail(AMH_ERR_UNSUPPORTED, "amh_create: L = %d needs %zu B of shared memory per chain, device allows %d",
                    n_res, amh::sweep_smem_bytes(n_res, 1, 1, 0, 0, 0, 0, 1, 1), c->max_smem);
    }

    cudaStream_t st = (cudaStream_t)cuda_stream;
    const long long count = (long long)n_res * n_res * n_bins;
    float *p_dev = nullptr;
    int *bad_dev = nullptr;
    cudaPointerAttributes at;
    bool on_device = (cudaPointerGetAttributes(&at, distogram) == cudaSuccess) &&
                     (at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged);
    cudaGetLastError();
    auto cleanup = [&]() {
        if (p_dev) cudaFree(p_dev);
        if (bad_dev) cudaFree(bad_dev);
        if (c->Epk) cudaFree(c->Epk);
        if (c->Elast) cudaFree(c->Elast);
        if (c->Ebd) cudaFree(c->Ebd);
        if (c->P) cudaFree(c->P);
        delete c;
    };
#define AMH_CUDA_C(call)                                                                           \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess) {                                                                   \
            cleanup();                                                                             \
            return fail(e_ == cudaErrorMemoryAllocation ? AMH_ERR_OOM : AMH_ERR_CUDA, "%s: %s", #call, \
                        cudaGetErrorString(e_));                                                   \
        }                                                                                          \
    } while (0)
    const size_t n_rows = std::max<size_t>(1, (size_t)n_res * (n_res - 1) / 2);
    AMH_CUDA_C(cudaMalloc(&c->Epk, sizeof(float2) * n_rows * n_bins));
    AMH_CUDA_C(cudaMalloc(&c->Elast, sizeof(float) * n_rows));
    {
        int stride = (n_bins + 3) & ~3;
        while ((stride & 7) != 4) stride += 4;          // 16-byte multiple, bank offset 4 (mod 8) words per row
        m.row_stride = stride;
    }
    // the band of the local phase: pairs up to 64 residues apart (windows up to 32 residues); wider windows gather from L2
    c->band_dmax = std::min(n_res - 1, 64);
    m.band_rows = std::max(0, c->band_dmax - o.min_sep + 1);
    {
        const size_t bb = sizeof(float) * std::max<size_t>(1, (size_t)n_res * m.band_rows) * m.row_stride;
        AMH_CUDA_C(cudaMalloc(&c->Ebd, bb));
        AMH_CUDA_C(cudaMemsetAsync(c->Ebd, 0, bb, st));
    }
    AMH_CUDA_C(cudaMalloc(&c->P, sizeof(float) * n_rows * n_bins));
    AMH_CUDA_C(cudaMalloc(&bad_dev, 3 * sizeof(int)));                // validity flag + the two table statistics
    AMH_CUDA_C(cudaMemsetAsync(bad_dev, 0, 3 * sizeof(int), st));
    const float *src = distogram;
    if (!on_device) {
        AMH_CUDA_C(cudaMalloc(&p_dev, sizeof(float) * (size_t)count));
        AMH_CUDA_C(cudaMemcpyAsync(p_dev, distogram, sizeof(float) * (size_t)count, cudaMemcpyHostToDevice, st));
        src = p_dev;
    }
    {
        const int threads = 256;
        const int blocks = (int)std::min<long long>((count + threads - 1) / threads, (long long)c->n_sm * 16);
        amh::table_kernel<<<blocks, threads, 0, st>>>(src, c->Epk, c->Elast, c->Ebd, m.band_rows, o.min_sep, c->P, m.row_stride, n_res, n_bins, o.eps, bad_dev);
        AMH_CUDA_C(cudaGetLastError());
    }
    double *vfar_dev = nullptr;
    AMH_CUDA_C(cudaMalloc(&vfar_dev, sizeof(double)));
    amh::vfar_kernel<<<1, 1024, 0, st>>>(c->P, n_res, n_bins, o.min_sep, o.eps, vfar_dev);
    {
        cudaError_t e_ = cudaGetLastError();
        if (e_ == cudaSuccess) e_ = cudaMemcpyAsync(&m.v_far, vfar_dev, sizeof(double), cudaMemcpyDeviceToHost, st);
        if (e_ == cudaSuccess) e_ = cudaStreamSynchronize(st);
        cudaFree(vfar_dev);
        if (e_ != cudaSuccess) { cleanup(); return fail(AMH_ERR_CUDA, "amh_create: v_far: %s", cudaGetErrorString(e_)); }
    }
    int bad3[3] = {0, 0, 0};
    AMH_CUDA_C(cudaMemcpyAsync(bad3, bad_dev, sizeof bad3, cudaMemcpyDeviceToHost, st));
    AMH_CUDA_C(cudaStreamSynchronize(st));
    const int bad = bad3[0];
    if (bad) { cleanup(); return fail(AMH_ERR_INVALID_ARG, "amh_create: the distogram holds a negative, NaN or infinite value"); }
    std::memcpy(&c->tab_emax, &bad3[1], sizeof(float));
    std::memcpy(&c->tab_step, &bad3[2], sizeof(float));
    cudaFree(bad_dev); bad_dev = nullptr;
    if (p_dev) { cudaFree(p_dev); p_dev = nullptr; }
    m.Epk = c->Epk; m.Elast = c->Elast; m.Ebd = c->Ebd; m.P = c->P;
#define AMH_SMEM_ATTR(SG_, RING_, CB_) AMH_CUDA_C(cudaFuncSetAttribute(amh::sweep_kernel<SG_, RING_, CB_>, cudaFuncAttributeMaxDynamicSharedMemorySize, c->max_smem))
    AMH_SMEM_ATTR(false, false, false); AMH_SMEM_ATTR(false, false, true); AMH_SMEM_ATTR(false, true, false); AMH_SMEM_ATTR(false, true, true);
    AMH_SMEM_ATTR(true, false, false); AMH_SMEM_ATTR(true, false, true); AMH_SMEM_ATTR(true, true, false); AMH_SMEM_ATTR(true, true, true);
#undef AMH_SMEM_ATTR
#define AMH_SMEM_ATTR_S(SG_, CB_) AMH_CUDA_C(cudaFuncSetAttribute(amh::sweep_kernel<SG_, false, CB_, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, c->max_smem))
    AMH_SMEM_ATTR_S(false, false); AMH_SMEM_ATTR_S(false, true); AMH_SMEM_ATTR_S(true, false); AMH_SMEM_ATTR_S(true, true);
#undef AMH_SMEM_ATTR_S
    AMH_CUDA_C(cudaFuncSetAttribute(amh::energy_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, c->max_smem));
#undef AMH_CUDA_C
    *out = c;
    return AMH_OK;
}

amh_status amh_create_tr5(amh_ctx **out, int n_res, const float *distogram, const float *bin_edges, int n_bins,
                          const amh_orientation_maps *maps, const amh_options *opt, void *cuda_stream)
{
    if (!out) return fail(AMH_ERR_INVALID_ARG, "amh_create_tr5: out is NULL");
    *out = nullptr;
    if (n_res < 1) return fail(AMH_ERR_INVALID_ARG, "amh_create_tr5: n_res = %d < 1", n_res);
    if (n_bins < 2) return fail(AMH_ERR_INVALID_ARG, "amh_create_tr5: n_bins = %d < 2", n_bins);
    if (!distogram || !bin_edges || !maps || !maps->omega || !maps->theta || !maps->phi)
        return fail(AMH_ERR_INVALID_ARG, "amh_create_tr5: distogram / bin_edges / maps is NULL");
    if (maps->nb_omega < 2 || maps->nb_theta < 2 || maps->nb_phi < 2)
        return fail(AMH_ERR_INVALID_ARG, "amh_create_tr5: every orientation map needs at least 2 bins");
    amh_options o;
    amh_default_options(&o);
    if (opt) o = *opt;
    if (o.min_sep < 1) return fail(AMH_ERR_INVALID_ARG, "amh_create_tr5: min_sep = %d < 1", o.min_sep);
    if (!(o.eps >= 0.0)) return fail(AMH_ERR_INVALID_ARG, "amh_create_tr5: eps < 0");
    for (int b = 0; b <= n_bins; ++b)
        if (!std::isfinite(bin_edges[b])) return fail(AMH_ERR_INVALID_ARG, "amh_create_tr5: bin edge %d is not finite", b);
    const double e0 = bin_edges[0], e1 = bin_edges[n_bins];
    const double delta = (e1 - e0) / n_bins;
    if (!(delta > 0.0)) return fail(AMH_ERR_INVALID_ARG, "amh_create_tr5: bin edges do not increase");
    for (int b = 0; b < n_bins; ++b) {
        const double w = (double)bin_edges[b + 1] - (double)bin_edges[b];
        if (!(w > 0.0)) return fail(AMH_ERR_INVALID_ARG, "amh_create_tr5: bin edges do not increase at %d", b);
        if (std::fabs(w - delta) > 1e-5 * delta)
            return fail(AMH_ERR_UNSUPPORTED, "amh_create_tr5: bins are not evenly spaced (bin %d: %g vs %g)", b, w, delta);
    }
    amh_ctx *c = new (std::nothrow) amh_ctx;
    if (!c) return fail(AMH_ERR_OOM, "amh_create_tr5: host allocation failed");
    c->opt = o;
    c->param = AMH_PARAM_TR5;
    amh_default_launch_options(&c->lopt);
    std::memset(&c->m, 0, sizeof c->m);
    cudaError_t e = cudaGetDevice(&c->device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&c->n_sm, cudaDevAttrMultiProcessorCount, c->device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&c->max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, c->device);
    if (e != cudaSuccess) { delete c; return fail(AMH_ERR_CUDA, "amh_create_tr5: no usable CUDA device: %s", cudaGetErrorString(e)); }
    if (amh::tr5_smem_bytes(n_res, true) > (size_t)c->max_smem - 1024) {
        delete c;
        return fail(AMH_ERR_UNSUPPORTED, "amh_create_tr5: L = %d needs %zu B of shared memory per chain, device allows %d", n_res,
                    amh::tr5_smem_bytes(n_res, true), c->max_smem);
    }
    c->m.L = n_res; c->m.n = 5 * n_res; c->m.nb = n_bins; c->m.min_sep = o.min_sep;
    amh::Tr5Model &t = c->tm;
    t.L = n_res; t.n = 5 * n_res; t.nb_d = n_bins; t.nb_o = maps->nb_omega; t.nb_t = maps->nb_theta; t.nb_p = maps->nb_phi;
    t.min_sep = o.min_sep;
    t.c0 = e0 + 0.5 * delta; t.delta = delta;
    t.A = mplus(o.ang_n_ca_c, 0.0, o.len_ca_c);
    t.c2 = std::cos(o.ang_ca_c_n); t.s2 = std::sin(o.ang_ca_c_n); t.l3 = o.len_c_n;
    t.c3 = std::cos(o.ang_c_n_ca); t.s3 = std::sin(o.ang_c_n_ca); t.l1 = o.len_n_ca;
    t.loc[0][0] = -o.len_n_ca; t.loc[0][1] = 0.0; t.loc[0][2] = 0.0;
    t.loc[1][0] = 0.0; t.loc[1][1] = 0.0; t.loc[1][2] = 0.0;
    t.loc[2][0] = -o.len_ca_c * std::cos(o.ang_n_ca_c); t.loc[2][1] = o.len_ca_c * std::sin(o.ang_n_ca_c); t.loc[2][2] = 0.0;
    t.loc[3][0] = -o.cb_len * std::cos(o.cb_ang);
    t.loc[3][1] = o.cb_len * std::sin(o.cb_ang) * std::cos(o.cb_dih);
    t.loc[3][2] = o.cb_len * std::sin(o.cb_ang) * std::sin(o.cb_dih);
    t.h0x = o.len_n_ca;
    t.inv_len_n_ca = 1.0 / o.len_n_ca; t.inv_len_ca_c = 1.0 / o.len_ca_c; t.inv_len_c_n = 1.0 / o.len_c_n;

    cudaStream_t st = (cudaStream_t)cuda_stream;
    int *bad_dev = nullptr;
    float *p_dev = nullptr;
    auto cleanup = [&]() {
        if (bad_dev) cudaFree(bad_dev);
        if (p_dev) cudaFree(p_dev);
        for (double *q : c->tE) if (q) cudaFree(q);
        delete c;
    };
#define AMH_CUDA_T(call)                                                                           \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess) {                                                                   \
            cleanup();                                                                             \
            return fail(e_ == cudaErrorMemoryAllocation ? AMH_ERR_OOM : AMH_ERR_CUDA, "%s: %s", #call, \
                        cudaGetErrorString(e_));                                                   \
        }                                                                                          \
    } while (0)
    AMH_CUDA_T(cudaMalloc(&bad_dev, sizeof(int)));
    AMH_CUDA_T(cudaMemsetAsync(bad_dev, 0, sizeof(int), st));
    const float *src[4] = {distogram, maps->omega, maps->theta, maps->phi};
    const int nbs[4] = {n_bins, maps->nb_omega, maps->nb_theta, maps->nb_phi};
    size_t max_count = 0;
    for (int q = 0; q < 4; ++q) max_count = std::max(max_count, (size_t)n_res * n_res * nbs[q]);
    for (int q = 0; q < 4; ++q) {
        const size_t count = (size_t)n_res * n_res * nbs[q];
        AMH_CUDA_T(cudaMalloc(&c->tE[q], sizeof(double) * count));
        cudaPointerAttributes at;
        const bool on_device = (cudaPointerGetAttributes(&at, src[q]) == cudaSuccess) &&
                               (at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged);
        cudaGetLastError();
        const float *ps = src[q];
        if (!on_device) {
            if (!p_dev) AMH_CUDA_T(cudaMalloc(&p_dev, sizeof(float) * max_count));
            AMH_CUDA_T(cudaMemcpyAsync(p_dev, src[q], sizeof(float) * count, cudaMemcpyHostToDevice, st));
            ps = p_dev;
        }
        const int blocks = (int)std::min<size_t>((count + 255) / 256, (size_t)c->n_sm * 16);
        amh::tr5_table_kernel<<<blocks, 256, 0, st>>>(ps, c->tE[q], (long long)count, o.eps, bad_dev);
        AMH_CUDA_T(cudaGetLastError());
    }
    int bad = 0;
    AMH_CUDA_T(cudaMemcpyAsync(&bad, bad_dev, sizeof(int), cudaMemcpyDeviceToHost, st));
    AMH_CUDA_T(cudaStreamSynchronize(st));
    if (bad) { cleanup(); return fail(AMH_ERR_INVALID_ARG, "amh_create_tr5: a map holds a negative, NaN or infinite value"); }
    cudaFree(bad_dev); bad_dev = nullptr;
    if (p_dev) { cudaFree(p_dev); p_dev = nullptr; }
    t.Ed = c->tE[0]; t.Eo = c->tE[1]; t.Et = c->tE[2]; t.Ep = c->tE[3];
    AMH_CUDA_T(cudaFuncSetAttribute(amh::tr5_sweep_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, c->max_smem - 1024));   // it also has a few static words
    AMH_CUDA_T(cudaFuncSetAttribute(amh::tr5_energy_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, c->max_smem));
    AMH_CUDA_T(cudaFuncSetAttribute(amh::tr5_geometry_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, c->max_smem));
#undef AMH_CUDA_T
    *out = c;
    return AMH_OK;
}

amh_status amh_pair_geometry(amh_ctx *c, const float *states, long long B, double *d_out, double *omega_out,
                             double *theta_out, double *phi_out, void *cuda_stream)
{
    if (!c) return fail(AMH_ERR_INVALID_ARG, "amh_pair_geometry: ctx is NULL");
    if (c->param != AMH_PARAM_TR5) return fail(AMH_ERR_INVALID_ARG, "amh_pair_geometry: needs an AMH_PARAM_TR5 context");
    if (B < 0) return fail(AMH_ERR_INVALID_ARG, "amh_pair_geometry: B = %lld < 0", B);
    if (B == 0) return AMH_OK;
    if (!states) return fail(AMH_ERR_INVALID_ARG, "amh_pair_geometry: states is NULL");
    const int blocks = (int)std::min<long long>(B, (long long)c->n_sm * 16);
    amh::tr5_geometry_kernel<<<blocks, 128, amh::tr5_smem_bytes(c->m.L, false), (cudaStream_t)cuda_stream>>>(
        c->tm, states, B, d_out, omega_out, theta_out, phi_out);
    AMH_CUDA(cudaGetLastError());
    return AMH_OK;
}

amh_status amh_destroy(amh_ctx *c)
{
    if (!c) return AMH_OK;
    // cudaFree waits for the work that still uses the allocation: no device-wide synchronisation of our own
    if (c->Epk) cudaFree(c->Epk);
    if (c->Elast) cudaFree(c->Elast);
    if (c->Ebd) cudaFree(c->Ebd);
    if (c->P) cudaFree(c->P);
    for (double *q : c->tE) if (q) cudaFree(q);
    if (c->stage) cudaFree(c->stage);
    delete c;
    return AMH_OK;
}

static amh_status launch_energy(amh_ctx *c, const float *states, long long B, int k, int window, float *out, cudaStream_t st)
{
    if (B == 0) return AMH_OK;
    if (c->param == AMH_PARAM_TR5) {
        const int blocks = (int)std::min<long long>(B, (long long)c->n_sm * 16);
        amh::tr5_energy_kernel<<<blocks, 128, amh::tr5_smem_bytes(c->m.L, false), st>>>(c->tm, states, B, k, window, out);
        AMH_CUDA(cudaGetLastError());
        return AMH_OK;
    }
    const size_t smem = sizeof(double) * 32 + sizeof(float) * 3 * (size_t)c->m.L;
    const int blocks = (int)std::min<long long>(B, (long long)c->n_sm * 64);
    amh::energy_kernel<<<blocks, 128, smem, st>>>(c->m, states, B, k, window, out);
    AMH_CUDA(cudaGetLastError());
    return AMH_OK;
}

amh_status amh_energy(amh_ctx *c, const float *states, long long B, float *energy_out, void *cuda_stream)
{
    if (!c) return fail(AMH_ERR_INVALID_ARG, "amh_energy: ctx is NULL");
    if (B < 0) return fail(AMH_ERR_INVALID_ARG, "amh_energy: B = %lld < 0", B);
    if (B > 0 && (!states || !energy_out)) return fail(AMH_ERR_INVALID_ARG, "amh_energy: states / energy_out is NULL");
    return launch_energy(c, states, B, -1, 0, energy_out, (cudaStream_t)cuda_stream);
}

amh_status amh_energy_local(amh_ctx *c, const float *states, long long B, int k, int window, float *energy_out,
                            void *cuda_stream)
{
    if (!c) return fail(AMH_ERR_INVALID_ARG, "amh_energy_local: ctx is NULL");
    if (B < 0) return fail(AMH_ERR_INVALID_ARG, "amh_energy_local: B = %lld < 0", B);
    if (k < 0 || k >= c->m.n) return fail(AMH_ERR_INVALID_ARG, "amh_energy_local: k = %d outside [0, %d)", k, c->m.n);
    if (window < 0) return fail(AMH_ERR_INVALID_ARG, "amh_energy_local: window = %d < 0", window);
    if (B > 0 && (!states || !energy_out)) return fail(AMH_ERR_INVALID_ARG, "amh_energy_local: states / energy_out is NULL");
    return launch_energy(c, states, B, k, window, energy_out, (cudaStream_t)cuda_stream);
}

amh_status amh_coords(amh_ctx *c, const float *states, long long B, float *cb_out, double *atoms_out, void *cuda_stream)
{
    if (!c) return fail(AMH_ERR_INVALID_ARG, "amh_coords: ctx is NULL");
    if (B < 0) return fail(AMH_ERR_INVALID_ARG, "amh_coords: B = %lld < 0", B);
    if (B == 0 || (!cb_out && !atoms_out)) return AMH_OK;
    if (!states) return fail(AMH_ERR_INVALID_ARG, "amh_coords: states is NULL");
    const int wpb = 4;
    const long long blocks = (B + wpb - 1) / wpb;
    if (blocks > 0x7fffffffLL) return fail(AMH_ERR_INVALID_ARG, "amh_coords: B too large");
    if (c->param == AMH_PARAM_TR5) {
        amh::tr5_coords_kernel<<<(int)blocks, 32 * wpb, 0, (cudaStream_t)cuda_stream>>>(c->tm, states, B, cb_out, atoms_out);
        AMH_CUDA(cudaGetLastError());
        return AMH_OK;
    }
    amh::coords_kernel<<<(int)blocks, 32 * wpb, 0, (cudaStream_t)cuda_stream>>>(c->m, states, B, cb_out, atoms_out);
    AMH_CUDA(cudaGetLastError());
    return AMH_OK;
}

// Launch shape of amh_run: C chains per CTA, W warps per chain, R ring slots, local proposals
// per pass, lanes per local proposal.
struct SweepShape { int C, W, R, ring_rows, cb64, nspec, gl, wpts; size_t smem; };

static SweepShape choose_shape(const amh_ctx *c, long long B, int window, int strided = 0)
{
    const int L = c->m.L;
    const int w_eff = std::min(window, std::max(L - 1, 0));
    const int span = std::min(2 * window, std::max(L - 1, 0));
    SweepShape sh;
    sh.ring_rows = std::max(0, span - c->m.min_sep + 1);
    sh.wpts = w_eff + 1;
    sh.gl = c->lopt.lanes_per_step > 0 ? c->lopt.lanes_per_step : 8;
    const size_t budget = (size_t)c->max_smem;
    auto spec_for = [&](int W) -> int {                       // local proposals per pass the team's lane groups can hold
        int ns = std::min(W * (32 / sh.gl), amh::kMaxSpec);
        if (c->lopt.spec_local > 0) ns = std::min(ns, c->lopt.spec_local);
        ns = std::min(ns, std::max(1, 8192 / (16 * sh.wpts)));    // the turned C-betas of a pass: 8 KB per chain at most
        return std::max(1, ns);
    };
    auto ring_for = [&](int C, int ns) -> int {               // slots: the window's columns + reach of a pass + drift between teams
        if (strided || c->lopt.ring_cols < 0 || sh.ring_rows == 0 || span > c->band_dmax || c->m.min_sep > amh::kRingPadRows + 1) return 0;
        if (c->lopt.ring_cols > 0) return std::max(c->lopt.ring_cols, w_eff + 3);
        return w_eff + 3 + (ns + 1) / 2 + (C > 1 ? 4 : 0);
    };
    sh.cb64 = 1;
    auto warps_for = [&](int C_) {
        const int W = c->lopt.warps_per_chain;
        return W > 0 ? std::max(1, std::min(W, amh::kMaxTeamWarps / C_)) : std::max(1, std::min(amh::kMaxTeamWarps / C_, 8));
    };
    const int cbn_f = strided ? 2 : 1;                       // strided sweeps keep two sets of columns per proposal
    auto fits = [&](int C, int R, int ns) { return amh::sweep_smem_bytes(L, C, warps_for(C), R, sh.ring_rows, c->m.row_stride, sh.cb64, cbn_f * ns, sh.wpts) <= budget; };
    // chains per CTA: spread the batch over the SMs (one CTA each) and keep as many teams resident as shared memory
    // allows; the ring is added only when it fits beside them (warps in flight are worth more than the ring)
    int C = c->lopt.chains_per_cta;
    const bool auto_c = C <= 0;
    if (auto_c) C = (int)std::min<long long>(7, std::max<long long>(1, (B + c->n_sm - 1) / c->n_sm));    // 7 x 2 warps + producer
    if (auto_c) {
        // the fp64 C-betas (24 L bytes per chain) are dropped before a chain is (they can be rebuilt from N, CA, C)
        if (!fits(C, 0, spec_for(warps_for(C)))) sh.cb64 = 0;
        while (C > 1 && !fits(C, 0, spec_for(warps_for(C)))) --C;
    }
    const int W = warps_for(C);
    int ns = spec_for(W);
    if (sh.cb64 && !fits(C, 0, ns)) sh.cb64 = 0;             // forced shapes
    int R = ring_for(C, ns);
    if (R > 0 && !fits(C, R, ns)) {
        if (sh.cb64) { sh.cb64 = 0; }                        // the ring is worth more than the stored fp64 C-betas
        if (!fits(C, R, ns)) {
            R = ring_for(1, ns);                             // without the slack for drift between teams
            if (!fits(C, R, ns)) { R = 0; sh.cb64 = fits(C, 0, ns) ? sh.cb64 : 0; }   // the ring does not fit: rows are gathered from L2
        }
    }
    if (R == 0 && !sh.cb64) { sh.cb64 = 1; if (!fits(C, 0, ns)) sh.cb64 = 0; }
    // a pass may not reach beyond what the ring can hold next to the window (else the team would wait for a column
    // whose slot it still occupies itself)
    if (R > 0) ns = std::max(1, std::min(ns, 2 * (R - w_eff - 2) - 1));
    sh.C = C; sh.W = W; sh.R = R; sh.nspec = ns;
    if (R == 0) sh.ring_rows = 0;
    sh.smem = amh::sweep_smem_bytes(L, C, W, R, sh.ring_rows, c->m.row_stride, sh.cb64, cbn_f * ns, sh.wpts);
    return sh;
}

amh_status amh_launch_info(amh_ctx *c, long long B, int window, int *threads_per_chain, int *smem_bytes, int *ctas_per_sm, int *n_sm)
{
    if (!c) return fail(AMH_ERR_INVALID_ARG, "amh_launch_info: ctx is NULL");
    if (c->param == AMH_PARAM_TR5) {
        const int threads = 128;
        if (threads_per_chain) *threads_per_chain = threads;
        if (smem_bytes) *smem_bytes = (int)amh::tr5_smem_bytes(c->m.L, true);
        if (n_sm) *n_sm = c->n_sm;
        if (ctas_per_sm) {
            int nb = 0;
            AMH_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, amh::tr5_sweep_kernel, threads, amh::tr5_smem_bytes(c->m.L, true)));
            *ctas_per_sm = nb;
        }
        return AMH_OK;
    }
    const SweepShape sh = choose_shape(c, std::max<long long>(B, 1), window);
    if (threads_per_chain) *threads_per_chain = 32 * sh.W;
    if (smem_bytes) *smem_bytes = (int)sh.smem;
    if (n_sm) *n_sm = c->n_sm;
    if (ctas_per_sm) {
        int nb = 0;
        AMH_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, amh::sweep_kernel<false, false, false>, 32 * (sh.C * sh.W + 1), sh.smem));
        *ctas_per_sm = nb;
    }
    return AMH_OK;
}

amh_status amh_launch_shape(amh_ctx *c, long long B, int window, int *chains_per_cta, int *warps_per_chain, int *ring_cols, int *ring_rows)
{
    if (!c) return fail(AMH_ERR_INVALID_ARG, "amh_launch_shape: ctx is NULL");
    if (c->param == AMH_PARAM_TR5) {
        if (chains_per_cta) *chains_per_cta = 1;
        if (warps_per_chain) *warps_per_chain = 4;
        if (ring_cols) *ring_cols = 0;
        if (ring_rows) *ring_rows = 0;
        return AMH_OK;
    }
    const SweepShape sh = choose_shape(c, std::max<long long>(B, 1), window);
    if (chains_per_cta) *chains_per_cta = sh.C;
    if (warps_per_chain) *warps_per_chain = sh.W;
    if (ring_cols) *ring_cols = sh.R;
    if (ring_rows) *ring_rows = sh.ring_rows;
    return AMH_OK;
}

static amh_status check_run(const amh_ctx *c, const float *states, long long B, long long n_sweeps, long long sweep_offset,
                            const amh_schedule *sc, const amh_temperature *tp, const amh_proposal *pr,
                            const amh_outputs *out)
{
    if (!c) return fail(AMH_ERR_INVALID_ARG, "amh_run: ctx is NULL");
    if (B < 0 || B > 0x7fffffffLL) return fail(AMH_ERR_INVALID_ARG, "amh_run: B = %lld out of range", B);
    if (B > 0 && !states) return fail(AMH_ERR_INVALID_ARG, "amh_run: states is NULL");
    if (n_sweeps < 0 || sweep_offset < 0) return fail(AMH_ERR_INVALID_ARG, "amh_run: n_sweeps / sweep_offset < 0");
    if (!sc || !tp) return fail(AMH_ERR_INVALID_ARG, "amh_run: schedule / temperature is NULL");
    if (sc->n_global < 0 || sc->n_local < 0 || sc->n_global + sc->n_local < 1)
        return fail(AMH_ERR_INVALID_ARG, "amh_run: schedule needs n_global, n_local >= 0 and n_global + n_local >= 1");
    if (sc->window < 0) return fail(AMH_ERR_INVALID_ARG, "amh_run: window = %d < 0", sc->window);
    if (sc->local_stride < 0) return fail(AMH_ERR_INVALID_ARG, "amh_run: local_stride = %d < 0", sc->local_stride);
    if (sc->local_stride > 0 && c->param == AMH_PARAM_TR5)
        return fail(AMH_ERR_UNSUPPORTED, "amh_run: the strided sweep order is built for AMH_PARAM_PHI_PSI only");
    if (!tp->per_chain_T && !(tp->t_start > 0.0 && tp->t_end > 0.0 && std::isfinite(tp->t_start) && std::isfinite(tp->t_end)))
        return fail(AMH_ERR_INVALID_ARG, "amh_run: temperatures must be finite and > 0");
    if (pr) {
        if (pr->mode != AMH_PROP_UNIFORM && pr->mode != AMH_PROP_GRID && pr->mode != AMH_PROP_GAUSSIAN)
            return fail(AMH_ERR_INVALID_ARG, "amh_run: unknown proposal mode %d", pr->mode);
        if (pr->mode == AMH_PROP_GRID && (pr->grid < 1 || pr->grid > (1 << 20))) return fail(AMH_ERR_INVALID_ARG, "amh_run: grid = %d out of range", pr->grid);
        if (pr->mode == AMH_PROP_GAUSSIAN && !(pr->sigma_start > 0.0 && pr->sigma_end > 0.0 && std::isfinite(pr->sigma_start) && std::isfinite(pr->sigma_end)))
            return fail(AMH_ERR_INVALID_ARG, "amh_run: Gaussian proposals need finite sigma_start, sigma_end > 0");
    }
    if (out && out->trace_steps < 0) return fail(AMH_ERR_INVALID_ARG, "amh_run: trace_steps < 0");
    return AMH_OK;
}

amh_status amh_run(amh_ctx *c, float *states, long long B, long long n_sweeps, long long sweep_offset,
                   long long chain_offset, const amh_schedule *sc, const amh_temperature *tp,
                   const amh_proposal *pr, unsigned long long seed, const amh_outputs *out, void *cuda_stream)
{
    amh_status stt = check_run(c, states, B, n_sweeps, sweep_offset, sc, tp, pr, out);
    if (stt != AMH_OK) return stt;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    amh::RunArgs a;
    std::memset(&a, 0, sizeof a);
    a.states = states; a.B = B; a.n_sweeps = n_sweeps; a.sweep_offset = sweep_offset; a.chain_offset = chain_offset;
    a.n_global = sc->n_global; a.n_local = sc->n_local; a.window = sc->window; a.global_first = sc->global_first ? 1 : 0;
    a.local_stride = sc->local_stride;
    a.t_start = tp->t_start; a.t_end = tp->t_end; a.ramp_sweeps = tp->ramp_sweeps; a.per_chain_T = tp->per_chain_T;
    a.prop_mode = pr ? pr->mode : AMH_PROP_UNIFORM; a.grid = pr ? pr->grid : 0;
    a.sigma_start = pr ? pr->sigma_start : 0.0; a.sigma_end = pr ? pr->sigma_end : 0.0; a.ramp_sigma = pr ? pr->ramp_sweeps : 0;
    a.seed = seed;
    {
        // exact-decision guard (R24): bound on |dE_fp32 - dE_fp64| at coordinates up to 32 A, scaled in the kernel by
        // the chain's extent / 32 A.  The constants are measured maxima with a safety factor of
        // about 4 on tables whose excess energies and bin-to-bin steps stay below kGuardTableRef (BASELINE.json's
        // distograms: 7.10 for both).  The fp32 error grows with both - the sums S_new, S_old grow with |E'|, the effect
        // of a coordinate's rounding with the slope - so a sharper table raises the bound by the SQUARE of
        // max(|E'|max, step max) / kGuardTableRef: measured on distograms without a uniform floor down to one-bin
        // peaks (|E'| = step = 18.42, the most eps = 1e-8 allows: factor 6.5) the error grows 4-8.5 fold, and stays
        // below a third of the scaled bound (profiles/r3_guard_sharp_tables.md).
        constexpr double kGuardTableRef = 7.2;
        const double sharp = std::max((double)c->tab_emax, (double)c->tab_step) / kGuardTableRef;
        const double gs = c->opt.guard_scale * (sharp > 1.0 ? sharp * sharp : 1.0);
        const int w_eff = std::min(sc->window, std::max(c->m.L - 1, 0));
        a.guard_global = gs * 2e-3 * std::sqrt(std::max(c->m.L, 64) / 64.0);
        a.guard_local = gs * 1e-3 * std::sqrt((w_eff + 1) / 9.0);
    }
    if (out) {
        a.energy = out->energy; a.best_energy = out->best_energy; a.best_state = out->best_state;
        a.n_accept_local = out->n_accept_local; a.n_accept_global = out->n_accept_global;
        a.first_hit = reinterpret_cast<unsigned long long *>(out->first_hit_sweep);
        a.energy_threshold = out->energy_threshold;
        a.trace_steps = out->trace_steps; a.trace_prop = out->trace_prop; a.trace_dE = out->trace_dE; a.trace_acc = out->trace_acc;
        if (a.first_hit) AMH_CUDA(cudaMemsetAsync(a.first_hit, 0xFF, sizeof(unsigned long long), st));   // -1 = none
    }
    if (B == 0) return AMH_OK;
    if (c->param == AMH_PARAM_TR5) {
        // config 3: one CTA per chain, one proposal at a time (amh_tr5.cuh)
        const int threads = 128;
        // 8 CTAs per SM against AMH_TR5_CTAS = 3 resident: chains differ in run time, and many short CTAs (1-2 rows each
        // at B = 2,048) balance better than one resident wave striding over 4-5 rows (measured on config 3: 7,484 ms
        // per step against 7,606 ms with n_sm * AMH_TR5_CTAS CTAs)
        const long long ctas = std::min<long long>(B, (long long)c->n_sm * 8);
        amh::tr5_sweep_kernel<<<(unsigned)ctas, threads, amh::tr5_smem_bytes(c->m.L, true), st>>>(c->tm, a);
        AMH_CUDA(cudaGetLastError());
        return AMH_OK;
    }
    const SweepShape sh = choose_shape(c, B, sc->window, sc->local_stride > 0);
    if (sh.smem > (size_t)c->max_smem)
        return fail(AMH_ERR_UNSUPPORTED, "amh_run: L = %d, window = %d, %d chains x %d warps need %zu B of shared memory, device allows %d",
                    c->m.L, sc->window, sh.C, sh.W, sh.smem, c->max_smem);
    a.C = sh.C; a.W = sh.W; a.ring_cols = sh.R; a.ring_rows = sh.ring_rows; a.cb64 = sh.cb64;
    a.nspec = sh.nspec; a.lanes_per_step = sh.gl; a.wpts = sh.wpts;
    const long long ctas = (B + sh.C - 1) / sh.C;
    // global proposals: one warp per step, speculatively, when a team has few warps (the whole team on one step when it
    // has many: a speculative pass of W steps wastes the ones after the first accept)
    // (and when the batch leaves most SMs empty: the wasted steps cost nothing there, the shorter critical path helps)
    const bool sg = c->lopt.spec_global >= 0 ? c->lopt.spec_global != 0 : (sh.W <= 2 || 2 * ctas <= c->n_sm);
    const unsigned threads = 32 * (sh.C * sh.W + 1);
    const int variant = (sg ? 4 : 0) | (sh.R > 0 ? 2 : 0) | (sh.cb64 ? 1 : 0);
    if (sc->local_stride > 0) {                              // NEXT-4's own instantiations (no ring)
#define AMH_LAUNCH_S(SG_, CB_) amh::sweep_kernel<SG_, false, CB_, true><<<(unsigned)ctas, threads, sh.smem, st>>>(c->m, a)
        switch (variant & 5) {
        case 0: AMH_LAUNCH_S(false, false); break;
        case 1: AMH_LAUNCH_S(false, true); break;
        case 4: AMH_LAUNCH_S(true, false); break;
        default: AMH_LAUNCH_S(true, true); break;
        }
#undef AMH_LAUNCH_S
        AMH_CUDA(cudaGetLastError());
        return AMH_OK;
    }
#define AMH_LAUNCH(SG_, RING_, CB_) amh::sweep_kernel<SG_, RING_, CB_><<<(unsigned)ctas, threads, sh.smem, st>>>(c->m, a)
    switch (variant) {
    case 0: AMH_LAUNCH(false, false, false); break;
    case 1: AMH_LAUNCH(false, false, true); break;
    case 2: AMH_LAUNCH(false, true, false); break;
    case 3: AMH_LAUNCH(false, true, true); break;
    case 4: AMH_LAUNCH(true, false, false); break;
    case 5: AMH_LAUNCH(true, false, true); break;
    case 6: AMH_LAUNCH(true, true, false); break;
    default: AMH_LAUNCH(true, true, true); break;
    }
#undef AMH_LAUNCH
    AMH_CUDA(cudaGetLastError());
    return AMH_OK;
}

static amh_status ensure_stage(amh_ctx *c, size_t bytes)
{
    if (bytes <= c->stage_bytes) return AMH_OK;
    if (c->stage) { cudaDeviceSynchronize(); cudaFree(c->stage); c->stage = nullptr; c->stage_bytes = 0; }
    AMH_CUDA(cudaMalloc(&c->stage, bytes));
    c->stage_bytes = bytes;
    return AMH_OK;
}

static size_t up256(size_t x) { return (x + 255) & ~(size_t)255; }

amh_status amh_run_host(amh_ctx *c, float *states, long long B, long long n_sweeps, long long sweep_offset,
                        long long chain_offset, const amh_schedule *sc, const amh_temperature *tp,
                        const amh_proposal *pr, unsigned long long seed, const amh_outputs *out, void *cuda_stream)
{
    amh_status stt = check_run(c, states, B, n_sweeps, sweep_offset, sc, tp, pr, out);
    if (stt != AMH_OK) return stt;
    if (tp->per_chain_T)
        for (long long q = 0; q < B; ++q)
            if (!(tp->per_chain_T[q] > 0.0f) || !std::isfinite(tp->per_chain_T[q]))
                return fail(AMH_ERR_INVALID_ARG, "amh_run_host: per_chain_T[%lld] = %g is not a finite temperature > 0", q, (double)tp->per_chain_T[q]);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t n = (size_t)c->m.n, b = (size_t)B;
    const size_t ts = out ? (size_t)out->trace_steps : 0;
    // carve the staging arena
    size_t off = 0;
    auto take = [&](bool want, size_t bytes) { size_t o = off; if (want) off += up256(bytes); return o; };
    const size_t o_states = take(true, b * n * 4);
    const size_t o_T = take(tp->per_chain_T != nullptr, b * 4);
    const size_t o_e = take(out && out->energy, b * 4);
    const size_t o_be = take(out && out->best_energy, b * 4);
    const size_t o_bs = take(out && out->best_state, b * n * 4);
    const size_t o_al = take(out && out->n_accept_local, b * 8);
    const size_t o_ag = take(out && out->n_accept_global, b * 8);
    const size_t o_fh = take(out && out->first_hit_sweep, 8);
    const size_t o_tp = take(out && out->trace_prop && ts, b * ts * 4);
    const size_t o_td = take(out && out->trace_dE && ts, b * ts * 8);
    const size_t o_ta = take(out && out->trace_acc && ts, b * ts);
    stt = ensure_stage(c, off + 256);
    if (stt != AMH_OK) return stt;
    char *base = static_cast<char *>(c->stage);
    AMH_CUDA(cudaMemcpyAsync(base + o_states, states, b * n * 4, cudaMemcpyHostToDevice, st));
    amh_temperature tpd = *tp;
    if (tp->per_chain_T) {
        AMH_CUDA(cudaMemcpyAsync(base + o_T, tp->per_chain_T, b * 4, cudaMemcpyHostToDevice, st));
        tpd.per_chain_T = reinterpret_cast<const float *>(base + o_T);
    }
    amh_outputs od;
    std::memset(&od, 0, sizeof od);
    if (out) {
        od = *out;
        od.energy = out->energy ? reinterpret_cast<float *>(base + o_e) : nullptr;
        od.best_energy = out->best_energy ? reinterpret_cast<float *>(base + o_be) : nullptr;
        od.best_state = out->best_state ? reinterpret_cast<float *>(base + o_bs) : nullptr;
        od.n_accept_local = out->n_accept_local ? reinterpret_cast<unsigned long long *>(base + o_al) : nullptr;
        od.n_accept_global = out->n_accept_global ? reinterpret_cast<unsigned long long *>(base + o_ag) : nullptr;
        od.first_hit_sweep = out->first_hit_sweep ? reinterpret_cast<long long *>(base + o_fh) : nullptr;
        od.trace_prop = (out->trace_prop && ts) ? reinterpret_cast<float *>(base + o_tp) : nullptr;
        od.trace_dE = (out->trace_dE && ts) ? reinterpret_cast<double *>(base + o_td) : nullptr;
        od.trace_acc = (out->trace_acc && ts) ? reinterpret_cast<unsigned char *>(base + o_ta) : nullptr;
    }
    stt = amh_run(c, reinterpret_cast<float *>(base + o_states), B, n_sweeps, sweep_offset, chain_offset, sc, &tpd, pr,
                  seed, out ? &od : nullptr, cuda_stream);
    if (stt != AMH_OK) return stt;
    AMH_CUDA(cudaMemcpyAsync(states, base + o_states, b * n * 4, cudaMemcpyDeviceToHost, st));
    if (out) {
        if (od.energy) AMH_CUDA(cudaMemcpyAsync(out->energy, od.energy, b * 4, cudaMemcpyDeviceToHost, st));
        if (od.best_energy) AMH_CUDA(cudaMemcpyAsync(out->best_energy, od.best_energy, b * 4, cudaMemcpyDeviceToHost, st));
        if (od.best_state) AMH_CUDA(cudaMemcpyAsync(out->best_state, od.best_state, b * n * 4, cudaMemcpyDeviceToHost, st));
        if (od.n_accept_local) AMH_CUDA(cudaMemcpyAsync(out->n_accept_local, od.n_accept_local, b * 8, cudaMemcpyDeviceToHost, st));
        if (od.n_accept_global) AMH_CUDA(cudaMemcpyAsync(out->n_accept_global, od.n_accept_global, b * 8, cudaMemcpyDeviceToHost, st));
        if (od.first_hit_sweep) AMH_CUDA(cudaMemcpyAsync(out->first_hit_sweep, od.first_hit_sweep, 8, cudaMemcpyDeviceToHost, st));
        if (od.trace_prop) AMH_CUDA(cudaMemcpyAsync(out->trace_prop, od.trace_prop, b * ts * 4, cudaMemcpyDeviceToHost, st));
        if (od.trace_dE) AMH_CUDA(cudaMemcpyAsync(out->trace_dE, od.trace_dE, b * ts * 8, cudaMemcpyDeviceToHost, st));
        if (od.trace_acc) AMH_CUDA(cudaMemcpyAsync(out->trace_acc, od.trace_acc, b * ts, cudaMemcpyDeviceToHost, st));
    }
    AMH_CUDA(cudaStreamSynchronize(st));
    return AMH_OK;
}

amh_status amh_energy_host(amh_ctx *c, const float *states, long long B, float *energy_out, void *cuda_stream)
{
    if (!c) return fail(AMH_ERR_INVALID_ARG, "amh_energy_host: ctx is NULL");
    if (B < 0) return fail(AMH_ERR_INVALID_ARG, "amh_energy_host: B = %lld < 0", B);
    if (B == 0) return AMH_OK;
    if (!states || !energy_out) return fail(AMH_ERR_INVALID_ARG, "amh_energy_host: states / energy_out is NULL");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t bytes = (size_t)B * c->m.n * 4;
    amh_status stt = ensure_stage(c, up256(bytes) + up256((size_t)B * 4));
    if (stt != AMH_OK) return stt;
    char *base = static_cast<char *>(c->stage);
    float *e_dev = reinterpret_cast<float *>(base + up256(bytes));
    AMH_CUDA(cudaMemcpyAsync(base, states, bytes, cudaMemcpyHostToDevice, st));
    stt = launch_energy(c, reinterpret_cast<const float *>(base), B, -1, 0, e_dev, st);
    if (stt != AMH_OK) return stt;
    AMH_CUDA(cudaMemcpyAsync(energy_out, e_dev, (size_t)B * 4, cudaMemcpyDeviceToHost, st));
    AMH_CUDA(cudaStreamSynchronize(st));
    return AMH_OK;
}

amh_status amh_exchange(amh_ctx *c, const float *energies, float *per_chain_T, long long B, int replicas, long long cycle,
                        long long chain_offset, unsigned long long seed, unsigned long long *n_tried,
                        unsigned long long *n_accepted, void *cuda_stream)
{
    if (!c) return fail(AMH_ERR_INVALID_ARG, "amh_exchange: ctx is NULL");
    if (B < 0 || replicas < 2 || B % replicas || chain_offset % replicas || cycle < 0)
        return fail(AMH_ERR_INVALID_ARG, "amh_exchange: B = %lld and chain_offset = %lld must be multiples of replicas = %d >= 2, cycle >= 0",
                    B, chain_offset, replicas);
    if (B == 0) return AMH_OK;
    if (!energies || !per_chain_T) return fail(AMH_ERR_INVALID_ARG, "amh_exchange: energies / per_chain_T is NULL");
    const long long pairs = (B / replicas) * (replicas / 2);
    amh::exchange_kernel<<<(unsigned)((pairs + 127) / 128), 128, 0, (cudaStream_t)cuda_stream>>>(
        energies, per_chain_T, B, replicas, cycle, seed, chain_offset, n_tried, n_accepted);
    AMH_CUDA(cudaGetLastError());
    return AMH_OK;
}

amh_status amh_run_pt(amh_ctx *c, float *states, long long B, long long n_cycles, long long cycle_offset,
                      long long chain_offset, const amh_schedule *sc, float *per_chain_T, int replicas,
                      const amh_proposal *pr, unsigned long long seed, float *energy, float *best_energy,
                      unsigned long long *n_tried, unsigned long long *n_accepted, void *cuda_stream)
{
    if (!c) return fail(AMH_ERR_INVALID_ARG, "amh_run_pt: ctx is NULL");
    if (!sc || !per_chain_T || !energy) return fail(AMH_ERR_INVALID_ARG, "amh_run_pt: schedule / per_chain_T / energy is NULL");
    if (n_cycles < 0 || cycle_offset < 0) return fail(AMH_ERR_INVALID_ARG, "amh_run_pt: n_cycles / cycle_offset < 0");
    if (replicas < 2 || B % replicas || chain_offset % replicas)
        return fail(AMH_ERR_INVALID_ARG, "amh_run_pt: B and chain_offset must be multiples of replicas >= 2");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (n_tried) AMH_CUDA(cudaMemsetAsync(n_tried, 0, sizeof(unsigned long long), st));
    if (n_accepted) AMH_CUDA(cudaMemsetAsync(n_accepted, 0, sizeof(unsigned long long), st));
    const long long cyc = (long long)sc->n_global + sc->n_local;
    // the per-cycle best energies land in the staging arena, then fold into best_energy
    float *cycle_best = nullptr;
    if (best_energy && B > 0) {
        amh_status stt = ensure_stage(c, up256((size_t)B * 4));
        if (stt != AMH_OK) return stt;
        cycle_best = static_cast<float *>(c->stage);
    }
    amh_temperature tp;
    tp.t_start = tp.t_end = 1.0; tp.ramp_sweeps = 0; tp.per_chain_T = per_chain_T;
    for (long long y = cycle_offset; y < cycle_offset + n_cycles; ++y) {
        amh_outputs o;
        std::memset(&o, 0, sizeof o);
        o.energy = energy; o.best_energy = cycle_best;
        amh_status stt = amh_run(c, states, B, cyc, y * cyc, chain_offset, sc, &tp, pr, seed, &o, cuda_stream);
        if (stt != AMH_OK) return stt;
        if (cycle_best && B > 0) {
            amh::min_into_kernel<<<(unsigned)((B + 255) / 256), 256, 0, st>>>(best_energy, cycle_best, B, y == cycle_offset);
            AMH_CUDA(cudaGetLastError());
        }
        stt = amh_exchange(c, energy, per_chain_T, B, replicas, y, chain_offset, seed, n_tried, n_accepted, cuda_stream);
        if (stt != AMH_OK) return stt;
    }
    return AMH_OK;
}

// amh_run_pt without the staging arena (include/amh.h says who needs this and why).  The loop below is amh_run_pt's,
// kernel for kernel; the only difference is where the per-cycle best energies live: in amh_pt_static_scratch, reached
// through the address pt_static_scratch() looked up for this device.  Nothing here may call cudaMalloc, cudaFree,
// ensure_stage or anything else that allocates - tests/test_zz_no_alloc.py reads this body and checks that.
amh_status amh_run_pt_static(amh_ctx *c, float *states, long long B, long long n_cycles, long long cycle_offset,
                             long long chain_offset, const amh_schedule *sc, float *per_chain_T, int replicas,
                             const amh_proposal *pr, unsigned long long seed, float *energy, float *best_energy,
                             unsigned long long *n_tried, unsigned long long *n_accepted, void *cuda_stream)
{
    if (!c) return fail(AMH_ERR_INVALID_ARG, "amh_run_pt_static: ctx is NULL");
    if (!sc || !per_chain_T || !energy) return fail(AMH_ERR_INVALID_ARG, "amh_run_pt_static: schedule / per_chain_T / energy is NULL");
    if (n_cycles < 0 || cycle_offset < 0) return fail(AMH_ERR_INVALID_ARG, "amh_run_pt_static: n_cycles / cycle_offset < 0");
    if (replicas < 2 || B % replicas || chain_offset % replicas)
        return fail(AMH_ERR_INVALID_ARG, "amh_run_pt_static: B and chain_offset must be multiples of replicas >= 2");
    if (B > (long long)AMH_RUN_PT_STATIC_MAX_CHAINS)
        return fail(AMH_ERR_UNSUPPORTED, "amh_run_pt_static: B = %lld chains exceed the built-in scratch of AMH_RUN_PT_STATIC_MAX_CHAINS = %d "
                    "(split the batch with chain_offset, or use amh_run_pt, which allocates)", B, (int)AMH_RUN_PT_STATIC_MAX_CHAINS);
    int device = -1;
    AMH_CUDA(cudaGetDevice(&device));
    if (device != c->device)
        return fail(AMH_ERR_INVALID_ARG, "amh_run_pt_static: the context lives on device %d, the current device is %d", c->device, device);
    // first call on this device: the address look-up (and whatever the runtime loads with it) happens here
    float *cycle_best = nullptr;
    amh_status stt = pt_static_scratch(device, &cycle_best);
    if (stt != AMH_OK) return stt;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (n_tried) AMH_CUDA(cudaMemsetAsync(n_tried, 0, sizeof(unsigned long long), st));
    if (n_accepted) AMH_CUDA(cudaMemsetAsync(n_accepted, 0, sizeof(unsigned long long), st));
    const long long cyc = (long long)sc->n_global + sc->n_local;
    const bool want_best = best_energy && B > 0;
    amh_temperature tp;
    tp.t_start = tp.t_end = 1.0; tp.ramp_sweeps = 0; tp.per_chain_T = per_chain_T;
    for (long long y = cycle_offset; y < cycle_offset + n_cycles; ++y) {
        amh_outputs o;
        std::memset(&o, 0, sizeof o);
        // the sweep kernel stores the best energy of every row [0, B) at the end of the cycle: whatever an earlier
        // call (of any batch size) left in the array is overwritten before min_into_kernel reads it - no clearing
        o.energy = energy; o.best_energy = want_best ? cycle_best : nullptr;
        stt = amh_run(c, states, B, cyc, y * cyc, chain_offset, sc, &tp, pr, seed, &o, cuda_stream);
        if (stt != AMH_OK) return stt;
        if (want_best) {
            amh::min_into_kernel<<<(unsigned)((B + 255) / 256), 256, 0, st>>>(best_energy, cycle_best, B, y == cycle_offset);
            AMH_CUDA(cudaGetLastError());
        }
        stt = amh_exchange(c, energy, per_chain_T, B, replicas, y, chain_offset, seed, n_tried, n_accepted, cuda_stream);
        if (stt != AMH_OK) return stt;
    }
    return AMH_OK;
}

amh_status amh_launch_variant(amh_ctx *c, long long B, int window, int *spec_global, int *ring, int *cb64, int *nspec, int *lanes)
{
    if (!c) return fail(AMH_ERR_INVALID_ARG, "amh_launch_variant: ctx is NULL");
    if (c->param == AMH_PARAM_TR5) {
        if (spec_global) *spec_global = 0;
        if (ring) *ring = 0;
        if (cb64) *cb64 = 1;
        if (nspec) *nspec = 1;
        if (lanes) *lanes = 128;
        return AMH_OK;
    }
    const SweepShape sh = choose_shape(c, std::max<long long>(B, 1), window);
    const long long ctas = (std::max<long long>(B, 1) + sh.C - 1) / sh.C;
    if (spec_global) *spec_global = (c->lopt.spec_global >= 0 ? c->lopt.spec_global != 0 : (sh.W <= 2 || 2 * ctas <= c->n_sm)) ? 1 : 0;
    if (ring) *ring = sh.R > 0 ? 1 : 0;
    if (cb64) *cb64 = sh.cb64;
    if (nspec) *nspec = sh.nspec;
    if (lanes) *lanes = sh.gl;
    return AMH_OK;
}

static amh_status probe_common(long long bytes, int reps, void **buf, cudaStream_t st)
{
    if (bytes < (1 << 20) || reps < 1) return fail(AMH_ERR_INVALID_ARG, "amh_probe: bytes >= 1 MiB and reps >= 1 are required");
    AMH_CUDA(cudaMalloc(buf, (size_t)bytes));
    cudaError_t e = cudaMemsetAsync(*buf, 0, (size_t)bytes, st);
    if (e != cudaSuccess) { cudaFree(*buf); return fail(AMH_ERR_CUDA, "amh_probe: %s", cudaGetErrorString(e)); }
    return AMH_OK;
}

amh_status amh_probe_l2_read(long long bytes, int reps, double *gb_per_s, void *cuda_stream)
{
    if (!gb_per_s) return fail(AMH_ERR_INVALID_ARG, "amh_probe_l2_read: output is NULL");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    void *buf = nullptr;
    amh_status stt = probe_common(bytes, reps, &buf, st);
    if (stt != AMH_OK) return stt;
    int dev = 0, n_sm = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    unsigned *out = reinterpret_cast<unsigned *>(buf);
    const size_t n16 = (size_t)bytes / 16;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    amh::l2_read_kernel<<<n_sm * 2, 512, 0, st>>>(reinterpret_cast<const uint4 *>(buf), n16, 1, out);
    cudaEventRecord(e0, st);
    amh::l2_read_kernel<<<n_sm * 2, 512, 0, st>>>(reinterpret_cast<const uint4 *>(buf), n16, reps, out);
    cudaEventRecord(e1, st);
    cudaError_t e = cudaEventSynchronize(e1);
    float ms = 0.0f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(buf);
    if (e != cudaSuccess) return fail(AMH_ERR_CUDA, "amh_probe_l2_read: %s", cudaGetErrorString(e));
    // every CTA reads the whole buffer `reps` times (rounded up to its 4 x blockDim chunks)
    const double chunks = std::ceil((double)n16 / (512.0 * 4.0));
    *gb_per_s = (double)n_sm * 2.0 * reps * chunks * 512.0 * 4.0 * 16.0 / (ms * 1e-3) / 1e9;
    return AMH_OK;
}

amh_status amh_probe_gather(long long bytes, int reps, double *gathers_per_s, void *cuda_stream)
{
    if (!gathers_per_s) return fail(AMH_ERR_INVALID_ARG, "amh_probe_gather: output is NULL");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    size_t n8 = 1;
    while (n8 * 2 * 8 <= (size_t)bytes) n8 *= 2;
    void *buf = nullptr;
    amh_status stt = probe_common((long long)(n8 * 8), reps, &buf, st);
    if (stt != AMH_OK) return stt;
    int dev = 0, n_sm = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    float *out = reinterpret_cast<float *>(buf);
    const int iters = 200;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    amh::gather_kernel<<<n_sm * 4, 256, 0, st>>>(reinterpret_cast<const float2 *>(buf), (unsigned)(n8 - 1), iters, out);
    cudaEventRecord(e0, st);
    for (int r = 0; r < reps; ++r)
        amh::gather_kernel<<<n_sm * 4, 256, 0, st>>>(reinterpret_cast<const float2 *>(buf), (unsigned)(n8 - 1), iters, out);
    cudaEventRecord(e1, st);
    cudaError_t e = cudaEventSynchronize(e1);
    float ms = 0.0f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(buf);
    if (e != cudaSuccess) return fail(AMH_ERR_CUDA, "amh_probe_gather: %s", cudaGetErrorString(e));
    *gathers_per_s = (double)n_sm * 4.0 * 256.0 * iters * 8.0 * reps / (ms * 1e-3);
    return AMH_OK;
}

amh_status amh_check_status(int *code, int *checked)
{
    if (!code || !checked) return fail(AMH_ERR_INVALID_ARG, "amh_check_status: output is NULL");
#ifdef AMH_CHECK
    *checked = 1;
#else
    *checked = 0;
#endif
    int v = 0;
    AMH_CUDA(cudaDeviceSynchronize());
    AMH_CUDA(cudaMemcpyFromSymbol(&v, amh::amh_check_word, sizeof(int)));
    *code = v;
    return AMH_OK;
}

amh_status amh_philox_test(const unsigned int *ctr, const unsigned int *key, unsigned int *out, long long count, void *cuda_stream)
{
    if (count < 0 || (count > 0 && (!ctr || !key || !out))) return fail(AMH_ERR_INVALID_ARG, "amh_philox_test: bad arguments");
    if (count == 0) return AMH_OK;
    amh::philox_test_kernel<<<(unsigned)((count + 127) / 128), 128, 0, (cudaStream_t)cuda_stream>>>(ctr, key, out, count);
    AMH_CUDA(cudaGetLastError());
    return AMH_OK;
}

}  // extern "C"
