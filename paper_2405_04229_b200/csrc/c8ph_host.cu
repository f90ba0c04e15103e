// c8ph_host.cu — host side of libc8ph: context, argument validation, table / detector setup and
// kernel launches behind the C-ABI of include/c8ph.h.  No torch types, no exceptions across the ABI.
#include <cuda_runtime.h>
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>
#include "c8ph_device.cuh"

using namespace c8ph;

static const size_t kSubstepBlockSums = 1u << 17;   // scan scratch: up to 2^27 tracks per sub-stepping call
static const int kMaxChunks = 16;           // host path: pipeline depth (chunks of segments per call)

struct c8ph_ctx {
    int device = 0;
    int n_sm = 0;
    std::string err;
    // atmosphere
    bool have_atm = false;
    DevAtm atm{};
    bool force_brute = false;          // C8PH_FORCE_BRUTE=1: search all telescopes (validation of the grids)
    bool force_generic = false;        // C8PH_FORCE_GENERIC=1: never pick the production-setting kernel variant
    double eta_span = 0.0;             // max |n(h) - n(h_obs)| over the table
    float *d_eta = nullptr, *d_xv = nullptr, *d_dxv = nullptr, *d_ext = nullptr, *d_aexp = nullptr, *d_mom = nullptr;
    // table
    bool have_table = false;
    DevTable tab{};
    c8ph_table_desc tab_desc{};
    float *d_full = nullptr;
    float4 *d_hot = nullptr;
    float4 *d_flat = nullptr;          // flat-plane table (R21): E texels then O texels
    float4 *d_cyl = nullptr;           // cylindrical model's table (R24)
    cudaArray_t tab_arr = nullptr;     // the hot texels as a 2-D array behind a texture object (DevTable::tex)
    cudaTextureObject_t tab_tex = 0;
    // detector
    bool have_det = false;
    DevDet det{};
    float4 *d_tel = nullptr;
    int *d_g_start[2] = {nullptr, nullptr};
    float2 *d_g_items[2] = {nullptr, nullptr};
    float *d_g_kmin[2] = {nullptr, nullptr};
    uint8_t *d_g_kq = nullptr;
    float4 *d_g_first = nullptr;
    int2 *d_g_first_kn = nullptr;
    float4 *d_g_knear = nullptr;
    // run scratch
    unsigned long long *d_cursor = nullptr;
    void *d_slots = nullptr;           // prepared-segment slots of the resident warps
    long long *d_bsums = nullptr;      // sub-stepping: block totals of the piece-count scan
    float *d_lines = nullptr;          // [2][n_lines]: wavelengths, cumulative probabilities (c8ph_set_line_spectrum)
    int n_lines = 0;
    float *d_eff = nullptr;            // detector efficiency table (c8ph_set_efficiency)
    int n_eff = 0;
    float eff_l0 = 0.f, eff_dl = 0.f;
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
    cudaEvent_t ev_done = nullptr;     // end of the context's last launch: a launch on another stream waits for it
    cudaStream_t last_stream = nullptr;
    bool have_launch = false;
    bool timed = false;
    int64_t launches = 0;
    // host-path scratch
    float *d_seg = nullptr; size_t seg_cap = 0;
    uint64_t *d_ids = nullptr; size_t ids_cap = 0;
    void *d_out = nullptr; size_t out_cap = 0;
    cudaStream_t st_h2d = nullptr, st_run = nullptr, st_d2h = nullptr;
    unsigned long long *h_written = nullptr;    // pinned: photon-list cursor after each chunk
    cudaEvent_t ev_in[kMaxChunks] = {}, ev_run[kMaxChunks] = {};
};

static thread_local std::string g_create_err;

static int fail(c8ph_ctx *ctx, int code, const std::string &msg)
{
    if (ctx) ctx->err = msg; else g_create_err = msg;
    return code;
}
static int cuda_fail(c8ph_ctx *ctx, cudaError_t e, const char *what)
{
    return fail(ctx, C8PH_E_CUDA, std::string(what) + ": " + cudaGetErrorString(e));
}
#define CU(call)                                                        \
    do {                                                                \
        cudaError_t e_ = (call);                                        \
        if (e_ != cudaSuccess) return cuda_fail(ctx, e_, #call);        \
    } while (0)

template <typename T>
static void dfree(T *&p)
{
    if (p) cudaFree(p);
    p = nullptr;
}

extern "C" int c8ph_version(void) { return C8PH_VERSION; }

extern "C" const char *c8ph_last_error(const c8ph_ctx *ctx) { return ctx ? ctx->err.c_str() : g_create_err.c_str(); }

extern "C" int c8ph_create(c8ph_ctx **out, int cuda_device)
{
    if (!out) return fail(nullptr, C8PH_E_ARG, "c8ph_create: out is NULL");
    *out = nullptr;
    int n = 0;
    cudaError_t e = cudaGetDeviceCount(&n);
    if (e != cudaSuccess || n <= 0)
        return fail(nullptr, C8PH_E_CUDA, std::string("c8ph_create: no CUDA device: ") + cudaGetErrorString(e));
    if (cuda_device < 0 || cuda_device >= n) return fail(nullptr, C8PH_E_ARG, "c8ph_create: bad device index");
    c8ph_ctx *ctx = new (std::nothrow) c8ph_ctx();
    if (!ctx) return fail(nullptr, C8PH_E_NOMEM, "c8ph_create: out of host memory");
    ctx->device = cuda_device;
    { const char *e = getenv("C8PH_FORCE_BRUTE"); ctx->force_brute = e && e[0] == '1'; }
    { const char *e = getenv("C8PH_FORCE_GENERIC"); ctx->force_generic = e && e[0] == '1'; }
    if ((e = cudaSetDevice(cuda_device)) != cudaSuccess ||
        (e = cudaDeviceGetAttribute(&ctx->n_sm, cudaDevAttrMultiProcessorCount, cuda_device)) != cudaSuccess ||
        (e = cudaMalloc(&ctx->d_cursor, sizeof(unsigned long long))) != cudaSuccess ||
        (e = cudaMalloc(&ctx->d_slots, segment_slot_bytes(ctx->n_sm) + queue_ring_bytes(ctx->n_sm))) != cudaSuccess ||
        (e = cudaMalloc(&ctx->d_bsums, kSubstepBlockSums * sizeof(long long))) != cudaSuccess ||
        (e = cudaEventCreate(&ctx->ev0)) != cudaSuccess || (e = cudaEventCreate(&ctx->ev1)) != cudaSuccess ||
        (e = cudaEventCreateWithFlags(&ctx->ev_done, cudaEventDisableTiming)) != cudaSuccess) {
        g_create_err = std::string("c8ph_create: ") + cudaGetErrorString(e);
        delete ctx;
        return C8PH_E_CUDA;
    }
    *out = ctx;
    return C8PH_OK;
}

extern "C" int c8ph_destroy(c8ph_ctx *ctx)
{
    if (!ctx) return C8PH_E_ARG;
    cudaSetDevice(ctx->device);
    dfree(ctx->d_eta); dfree(ctx->d_xv); dfree(ctx->d_dxv); dfree(ctx->d_ext); dfree(ctx->d_aexp); dfree(ctx->d_mom);
    dfree(ctx->d_full); dfree(ctx->d_hot); dfree(ctx->d_tel); dfree(ctx->d_flat); dfree(ctx->d_cyl);
    if (ctx->tab_tex) cudaDestroyTextureObject(ctx->tab_tex);
    if (ctx->tab_arr) cudaFreeArray(ctx->tab_arr);
    for (int k = 0; k < 2; ++k) { dfree(ctx->d_g_start[k]); dfree(ctx->d_g_items[k]); dfree(ctx->d_g_kmin[k]); }
    dfree(ctx->d_g_kq); dfree(ctx->d_g_first); dfree(ctx->d_g_first_kn);
    dfree(ctx->d_g_knear);
    dfree(ctx->d_cursor); dfree(ctx->d_lines); dfree(ctx->d_eff); dfree(ctx->d_seg); dfree(ctx->d_ids);
    if (ctx->d_slots) { cudaFree(ctx->d_slots); ctx->d_slots = nullptr; }
    dfree(ctx->d_bsums);
    if (ctx->d_out) { cudaFree(ctx->d_out); ctx->d_out = nullptr; }
    if (ctx->st_h2d) {
        cudaStreamDestroy(ctx->st_h2d); cudaStreamDestroy(ctx->st_run); cudaStreamDestroy(ctx->st_d2h);
        if (ctx->h_written) cudaFreeHost(ctx->h_written);
        for (int c = 0; c < kMaxChunks; ++c) { if (ctx->ev_in[c]) cudaEventDestroy(ctx->ev_in[c]); if (ctx->ev_run[c]) cudaEventDestroy(ctx->ev_run[c]); }
    }
    if (ctx->ev0) cudaEventDestroy(ctx->ev0);
    if (ctx->ev1) cudaEventDestroy(ctx->ev1);
    if (ctx->ev_done) cudaEventDestroy(ctx->ev_done);
    delete ctx;
    return C8PH_OK;
}

// ------------------------------------------------------------------------------------ atmosphere
static double lerp_table(const std::vector<float> &t, double h0, double dh, double h)
{
    double f = (h - h0) / dh;
    f = std::min(std::max(f, 0.0), (double)(t.size() - 1));
    int k = std::min((int)f, (int)t.size() - 2);
    double fr = f - k;
    return (1.0 - fr) * t[k] + fr * t[k + 1];
}

extern "C" int c8ph_init_atmosphere(c8ph_ctx *ctx, const c8ph_atmosphere_desc *d)
{
    if (!ctx) return C8PH_E_ARG;
    if (!d || d->size != sizeof(c8ph_atmosphere_desc)) return fail(ctx, C8PH_E_ARG, "init_atmosphere: bad desc/size");
    if (d->model < C8PH_ATM_HOMOGENEOUS || d->model > C8PH_ATM_CYLINDRICAL) return fail(ctx, C8PH_E_ARG, "init_atmosphere: bad model");
    if (d->model == C8PH_ATM_CYLINDRICAL && d->aer_L_m > 0.f) return fail(ctx, C8PH_E_ARG, "init_atmosphere: no aerosol in the cylindrical model");
    CU(cudaSetDevice(ctx->device));
    std::vector<float> eta, xv;
    double h0 = d->h0_m, dh = d->dh_m;
    if (d->model == C8PH_ATM_HOMOGENEOUS) {
        eta.assign(2, d->n_const_minus_1);
        xv.assign(2, 0.f);
        h0 = 0.0; dh = 1.0e6;
    } else {
        if (d->n_nodes < 2 || !d->refractivity || !(d->dh_m > 0.f)) return fail(ctx, C8PH_E_ARG, "init_atmosphere: need n_nodes >= 2, refractivity, dh > 0");
        if (d->n_nodes > 16000) return fail(ctx, C8PH_E_ARG, "init_atmosphere: n_nodes > 16000 does not fit the shared-memory staging");
        eta.assign(d->refractivity, d->refractivity + d->n_nodes);
        if (d->overburden_gcm2) xv.assign(d->overburden_gcm2, d->overburden_gcm2 + d->n_nodes);
        else xv.assign(d->n_nodes, 0.f);
    }
    for (float v : eta) if (!(v > -1.f) || !std::isfinite(v)) return fail(ctx, C8PH_E_ARG, "init_atmosphere: non-finite refractivity");
    if (d->model >= C8PH_ATM_SPHERICAL && !(d->earth_radius_m > 0.f)) return fail(ctx, C8PH_E_ARG, "init_atmosphere: earth_radius");
    const int n = (int)eta.size();
    const int n_pad = (n + 3) & ~3;
    std::vector<float> dxv(n_pad, 0.f), eta_p(n_pad, eta.back()), xv_p(n_pad, xv.back());
    for (int k = 0; k < n; ++k) { eta_p[k] = eta[k]; xv_p[k] = xv[k]; }
    for (int k = 0; k + 1 < n; ++k) {
        dxv[k] = (float)((double)xv[k] - (double)xv[k + 1]);
    }
    dfree(ctx->d_eta); dfree(ctx->d_xv); dfree(ctx->d_dxv);
    const size_t bytes = (size_t)n_pad * sizeof(float);
    CU(cudaMalloc(&ctx->d_eta, bytes)); CU(cudaMalloc(&ctx->d_xv, bytes));
    CU(cudaMalloc(&ctx->d_dxv, bytes));
    CU(cudaMemcpy(ctx->d_eta, eta_p.data(), bytes, cudaMemcpyHostToDevice));
    CU(cudaMemcpy(ctx->d_xv, xv_p.data(), bytes, cudaMemcpyHostToDevice));
    CU(cudaMemcpy(ctx->d_dxv, dxv.data(), bytes, cudaMemcpyHostToDevice));
    DevAtm &a = ctx->atm;
    a.model = d->model; a.n_nodes = n; a.n_pad = n_pad;
    a.h0 = (float)h0; a.dh = (float)dh; a.inv_dh = (float)(1.0 / dh); a.h_top = (float)(h0 + dh * (n - 1)); a.f_max = (float)(n - 1);
    a.eta = ctx->d_eta; a.xv = ctx->d_xv; a.dxv = ctx->d_dxv;
    a.R = d->earth_radius_m; a.h_obs = d->h_obs_m; a.Rg = (double)d->earth_radius_m + (double)d->h_obs_m;
    a.eta_g = (float)lerp_table(eta, h0, dh, d->h_obs_m);
    ctx->eta_span = 0.0;
    for (float v : eta) ctx->eta_span = std::max(ctx->eta_span, std::fabs((double)v - (double)a.eta_g));
    a.ray_inv_X = d->rayleigh_X_gcm2 > 0.f ? 1.0f / d->rayleigh_X_gcm2 : 0.f;
    a.ray_lambda = d->rayleigh_lambda_nm;
    a.aer_L = d->aer_L_m; a.aer_H = d->aer_H_m; a.aer_lambda = d->aer_lambda_nm; a.aer_angstrom = d->aer_angstrom;
    if (a.aer_L > 0.f && !(a.aer_H > 0.f)) return fail(ctx, C8PH_E_ARG, "init_atmosphere: aerosol scale height");
    {
        // aerosol column at the nodes for the per-photon layered sum: A(h) = (H/L) exp(-h/H)
        std::vector<float> aexp(n_pad, 0.f);
        a.aer_HL = a.aer_invH = a.aer_Ag = 0.f;
        if (a.aer_L > 0.f) {
            const double H = a.aer_H, HL = (double)a.aer_H / (double)a.aer_L;
            for (int k = 0; k < n; ++k) aexp[k] = (float)(HL * std::exp(-(h0 + dh * k) / H));
            a.aer_HL = (float)HL; a.aer_invH = (float)(1.0 / H); a.aer_Ag = (float)(HL * std::exp(-(double)d->h_obs_m / H));
        }
        dfree(ctx->d_aexp);
        CU(cudaMalloc(&ctx->d_aexp, bytes));
        CU(cudaMemcpy(ctx->d_aexp, aexp.data(), bytes, cudaMemcpyHostToDevice));
        a.aexp = ctx->d_aexp;
    }
    a.xv_g = (float)lerp_table(xv, h0, dh, d->h_obs_m);
    {
        // The planar layered sum in closed form ("layered sum"): with nu_l = n_l^2 - 1 at the layer's
        // mid height, every term of the sum is a power series in (nu_l - nu_e) / (n_e cos z)^2, so the photon needs only
        // the sums of thickness * nu_l^p (p = 1..4) and of dX_v * n_l * nu_l^p (p = 0..3) over the layers between the
        // observation level and its emission cell.  mom[q][k] holds them for the layers from the observation level up to
        // node k, the same layers, mid-height values and float inputs the per-layer loop uses, accumulated in fp64.
        const float fgf = std::fmin(std::fmax(((float)a.h_obs - a.h0) * a.inv_dh, 0.f), (float)(n - 1));
        const int kg = std::min((int)fgf, n - 2);
        const double frg = (double)(fgf - (float)kg);
        std::vector<float> mom(8 * (size_t)n_pad, 0.f);
        double acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
        double nu_lo = 1e300, nu_hi = -1e300;
        for (int k = 0; k < n; ++k) { const double v = (double)eta[k] * (2.0 + (double)eta[k]); nu_lo = std::min(nu_lo, v); nu_hi = std::max(nu_hi, v); }
        auto add_layer = [&](double eta_l, double thick, double dxv_l) {
            const double nl = 1.0 + eta_l, nu = eta_l * (2.0 + eta_l);
            double pw = nu;
            for (int q = 0; q < 4; ++q) { acc[q] += thick * pw; pw *= nu; }
            pw = 1.0;
            for (int q = 4; q < 8; ++q) { acc[q] += dxv_l * nl * pw; pw *= nu; }
        };
        for (int k = kg + 1; k < n; ++k) {
            if (k == kg + 1) add_layer((double)eta[kg] + 0.5 * (1.0 + frg) * ((double)eta[kg + 1] - (double)eta[kg]), (1.0 - frg) * (double)a.dh, (1.0 - frg) * (double)dxv[kg]);
            else add_layer(0.5 * ((double)eta[k - 1] + (double)eta[k]), (double)a.dh, (double)dxv[k - 1]);
            for (int q = 0; q < 8; ++q) mom[(size_t)q * n_pad + k] = (float)acc[q];
        }
        dfree(ctx->d_mom);
        CU(cudaMalloc(&ctx->d_mom, mom.size() * sizeof(float)));
        CU(cudaMemcpy(ctx->d_mom, mom.data(), mom.size() * sizeof(float), cudaMemcpyHostToDevice));
        a.mom = ctx->d_mom;
        a.nu_span = (float)(nu_hi - nu_lo);
    }
    a.n_ext = 0; a.ext = nullptr; a.ext_l0 = 0.f; a.ext_inv_dl = 0.f;
    dfree(ctx->d_ext);
    if (d->n_ext_lambda > 0) {
        if (d->model == C8PH_ATM_HOMOGENEOUS || !d->ext_tau_v || !d->overburden_gcm2 || (d->n_ext_lambda > 1 && !(d->ext_dlambda_nm > 0.f)) || d->n_ext_lambda > 4096)
            return fail(ctx, C8PH_E_ARG, "init_atmosphere: extinction table needs a height grid, overburden, ext_tau_v and ext_dlambda_nm > 0");
        const size_t ne = (size_t)d->n_ext_lambda * n;
        for (size_t k = 0; k < ne; ++k) if (!(d->ext_tau_v[k] >= 0.f) || !std::isfinite(d->ext_tau_v[k])) return fail(ctx, C8PH_E_ARG, "init_atmosphere: extinction table entry < 0 or not finite");
        CU(cudaMalloc(&ctx->d_ext, ne * sizeof(float)));
        CU(cudaMemcpy(ctx->d_ext, d->ext_tau_v, ne * sizeof(float), cudaMemcpyHostToDevice));
        a.n_ext = d->n_ext_lambda; a.ext = ctx->d_ext; a.ext_l0 = d->ext_lambda0_nm;
        a.ext_inv_dl = d->n_ext_lambda > 1 ? 1.0f / d->ext_dlambda_nm : 0.f;
    }
    ctx->have_atm = true;
    ctx->have_table = false;
    return C8PH_OK;
}

// ------------------------------------------------------------------------------------ trace table
static int alloc_table(c8ph_ctx *ctx, const c8ph_table_desc *t)
{
    if (!t || t->size != sizeof(c8ph_table_desc)) return fail(ctx, C8PH_E_ARG, "trace_table: bad desc/size");
    if (t->n_h < 2 || t->n_zen < 2 || (int64_t)t->n_h * t->n_zen > (1 << 26) || !(t->h_max_m > 0.f) ||
        !(t->zen_max_deg > 0.f) || !(t->zen_max_deg < 90.f))
        return fail(ctx, C8PH_E_ARG, "trace_table: need n_h,n_zen >= 2, h_max > 0, 0 < zen_max < 90");
    if (!ctx->have_atm) return fail(ctx, C8PH_E_STATE, "trace_table: atmosphere not initialised");
    if (t->n_rho < 0 || t->n_rho == 1 || t->n_rho > 4096 || (t->n_rho >= 2 && (!(t->rho_max_m > 0.f) || ctx->atm.model != C8PH_ATM_SPHERICAL)))
        return fail(ctx, C8PH_E_ARG, "trace_table: the flat-plane table needs n_rho >= 2, rho_max_m > 0 and the spherical model");
    if (t->n_c < 0 || t->n_c == 1 || t->n_c > 1024 || (t->n_c >= 2 && ctx->atm.model != C8PH_ATM_CYLINDRICAL))
        return fail(ctx, C8PH_E_ARG, "trace_table: n_c >= 2 needs the cylindrical model");
    CU(cudaSetDevice(ctx->device));
    dfree(ctx->d_full); dfree(ctx->d_hot); dfree(ctx->d_flat); dfree(ctx->d_cyl);
    const size_t n = (size_t)t->n_h * t->n_zen;
    CU(cudaMalloc(&ctx->d_full, n * C8PH_TABLE_CHANNELS * sizeof(float)));
    CU(cudaMalloc(&ctx->d_hot, n * sizeof(float4)));
    ctx->tab_desc = *t;
    DevTable &d = ctx->tab;
    d.n_h = t->n_h; d.n_zen = t->n_zen; d.h_max = t->h_max_m;
    const double zmax = (double)t->zen_max_deg * (3.14159265358979323846 / 180.0);
    d.zen_max = (float)zmax;
    d.inv_dh = (float)((t->n_h - 1) / (double)t->h_max_m);
    d.inv_dz = (float)((t->n_zen - 1) / zmax);
    d.f_max = (float)(t->n_h - 1); d.g_max = (float)(t->n_zen - 1);
    d.hot = ctx->d_hot; d.full = ctx->d_full;
    d.n_rho = 0; d.rho_max = 0.f; d.inv_drho = 0.f; d.e_max = 0.f; d.flatE = d.flatO = nullptr;
    if (t->n_rho >= 2) {
        CU(cudaMalloc(&ctx->d_flat, 2 * (size_t)t->n_rho * n * sizeof(float4)));
        d.n_rho = t->n_rho; d.rho_max = t->rho_max_m; d.inv_drho = (float)((t->n_rho - 1) / (double)t->rho_max_m);
        d.e_max = (float)(t->n_rho - 1);
        d.flatE = ctx->d_flat; d.flatO = ctx->d_flat + (size_t)t->n_rho * n;
    }
    d.n_c = 0; d.c_max = 0.f; d.cyl = nullptr;
    if (t->n_c >= 2) {
        CU(cudaMalloc(&ctx->d_cyl, (size_t)t->n_c * n * sizeof(float4)));
        d.n_c = t->n_c; d.c_max = (float)(t->n_c - 1); d.cyl = ctx->d_cyl;
    }
    // texture view of the hot texels: x = zenith node, y = height node, unnormalised coordinates, clamped, bilinear
    if (ctx->tab_tex) { cudaDestroyTextureObject(ctx->tab_tex); ctx->tab_tex = 0; }
    if (ctx->tab_arr) { cudaFreeArray(ctx->tab_arr); ctx->tab_arr = nullptr; }
    d.tex = 0;
    if (t->n_zen <= 65536 && t->n_h <= 65536) {
        const cudaChannelFormatDesc fmt = cudaCreateChannelDesc<float4>();
        CU(cudaMallocArray(&ctx->tab_arr, &fmt, (size_t)t->n_zen, (size_t)t->n_h));
        cudaResourceDesc res{};
        res.resType = cudaResourceTypeArray;
        res.res.array.array = ctx->tab_arr;
        cudaTextureDesc td{};
        td.addressMode[0] = td.addressMode[1] = cudaAddressModeClamp;
        td.filterMode = cudaFilterModeLinear;
        td.readMode = cudaReadModeElementType;
        td.normalizedCoords = 0;
        CU(cudaCreateTextureObject(&ctx->tab_tex, &res, &td, nullptr));
        d.tex = ctx->tab_tex;
    }
    return C8PH_OK;
}

// copy the hot texels into the texture's array (device to device, on `st`)
static int fill_table_texture(c8ph_ctx *ctx, cudaStream_t st)
{
    if (!ctx->tab_arr) return C8PH_OK;
    const size_t row = (size_t)ctx->tab.n_zen * sizeof(float4);
    CU(cudaMemcpy2DToArrayAsync(ctx->tab_arr, 0, 0, ctx->d_hot, row, row, (size_t)ctx->tab.n_h, cudaMemcpyDeviceToDevice, st));
    return C8PH_OK;
}

extern "C" int c8ph_build_trace_table(c8ph_ctx *ctx, const c8ph_table_desc *t, void *stream)
{
    if (!ctx) return C8PH_E_ARG;
    int rc = alloc_table(ctx, t);
    if (rc) return rc;
    TableBuildArgs a{};
    a.atm = ctx->atm;
    a.n_h = t->n_h; a.n_zen = t->n_zen; a.substeps = std::max(1, t->substeps);
    a.h_max = t->h_max_m;
    a.zen_max = (double)t->zen_max_deg * (3.14159265358979323846 / 180.0);
    a.full = ctx->d_full; a.hot = ctx->d_hot;
    a.n_rho = ctx->tab.n_rho; a.rho_max = ctx->tab.rho_max;
    a.flatE = const_cast<float4 *>(ctx->tab.flatE); a.flatO = const_cast<float4 *>(ctx->tab.flatO);
    a.n_c = ctx->tab.n_c; a.cyl = ctx->d_cyl;
    cudaError_t e = launch_build_table(a, (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "build_trace_table launch");
    rc = fill_table_texture(ctx, (cudaStream_t)stream);
    if (rc) return rc;
    ctx->launches += 1 + (ctx->tab.n_rho >= 2 ? 1 : 0) + (ctx->tab.n_c >= 2 ? 1 : 0);
    ctx->have_table = true;
    return C8PH_OK;
}

extern "C" int c8ph_get_trace_table_flat(c8ph_ctx *ctx, float *host_out, int64_t n_floats)
{
    if (!ctx) return C8PH_E_ARG;
    if (!ctx->have_table || ctx->tab.n_rho < 2) return fail(ctx, C8PH_E_STATE, "get_trace_table_flat: no flat-plane table");
    const int64_t need = 2ll * ctx->tab.n_rho * ctx->tab.n_h * ctx->tab.n_zen * 4;
    if (!host_out || n_floats < need) return fail(ctx, C8PH_E_ARG, "get_trace_table_flat: buffer too small");
    CU(cudaSetDevice(ctx->device));
    CU(cudaDeviceSynchronize());
    CU(cudaMemcpy(host_out, ctx->d_flat, need * sizeof(float), cudaMemcpyDeviceToHost));
    return C8PH_OK;
}

extern "C" int c8ph_get_trace_table_cyl(c8ph_ctx *ctx, float *host_out, int64_t n_floats)
{
    if (!ctx) return C8PH_E_ARG;
    if (!ctx->have_table || ctx->tab.n_c < 2) return fail(ctx, C8PH_E_STATE, "get_trace_table_cyl: no cylindrical table");
    const int64_t need = (int64_t)ctx->tab.n_c * ctx->tab.n_h * ctx->tab.n_zen * 4;
    if (!host_out || n_floats < need) return fail(ctx, C8PH_E_ARG, "get_trace_table_cyl: buffer too small");
    CU(cudaSetDevice(ctx->device));
    CU(cudaDeviceSynchronize());
    CU(cudaMemcpy(host_out, ctx->d_cyl, need * sizeof(float), cudaMemcpyDeviceToHost));
    return C8PH_OK;
}

extern "C" int c8ph_get_trace_table(c8ph_ctx *ctx, float *host_out, int64_t n_floats)
{
    if (!ctx) return C8PH_E_ARG;
    if (!ctx->have_table) return fail(ctx, C8PH_E_STATE, "get_trace_table: no table");
    const int64_t need = (int64_t)ctx->tab.n_h * ctx->tab.n_zen * C8PH_TABLE_CHANNELS;
    if (!host_out || n_floats < need) return fail(ctx, C8PH_E_ARG, "get_trace_table: buffer too small");
    CU(cudaSetDevice(ctx->device));
    CU(cudaDeviceSynchronize());
    CU(cudaMemcpy(host_out, ctx->d_full, need * sizeof(float), cudaMemcpyDeviceToHost));
    return C8PH_OK;
}

extern "C" int c8ph_set_trace_table(c8ph_ctx *ctx, const c8ph_table_desc *t, const float *host_in)
{
    if (!ctx) return C8PH_E_ARG;
    if (!host_in) return fail(ctx, C8PH_E_ARG, "set_trace_table: host_in is NULL");
    if (t && t->size == sizeof(c8ph_table_desc) && (t->n_rho != 0 || t->n_c != 0)) return fail(ctx, C8PH_E_ARG, "set_trace_table: n_rho and n_c must be 0 (those tables are built, not injected)");
    int rc = alloc_table(ctx, t);
    if (rc) return rc;
    const size_t n = (size_t)t->n_h * t->n_zen;
    std::vector<float4> hot(n);
    for (size_t i = 0; i < n; ++i) {
        const float *v = host_in + i * C8PH_TABLE_CHANNELS;
        hot[i] = make_float4(v[0], v[2], v[3], v[4]);
    }
    CU(cudaMemcpy(ctx->d_full, host_in, n * C8PH_TABLE_CHANNELS * sizeof(float), cudaMemcpyHostToDevice));
    CU(cudaMemcpy(ctx->d_hot, hot.data(), n * sizeof(float4), cudaMemcpyHostToDevice));
    rc = fill_table_texture(ctx, nullptr);
    if (rc) return rc;
    CU(cudaStreamSynchronize(nullptr));
    ctx->have_table = true;
    return C8PH_OK;
}

// ------------------------------------------------------------------------------------ detector
// Uniform grid over the telescope footprints (see DevGrid).  mode 0 (hit): key = dist(cell, centre)
// / (r + |z|), listed while key <= key_max = 1/min_cos.  mode 1 (LV2): key = dist(cell, centre) in
// metres, listed while key <= r_max/min_cos + margin_max.  Cell rectangles are padded so that the
// fp32 cell index of a point can be off by rounding without losing a candidate; keys are rounded
// DOWN to fp32 so a device-side "key > threshold" never rejects a reachable telescope.
static const double kLv2MarginMax = 64.0;   // the LV2 grid lists telescopes up to this margin
static const double kGridMinCos = 0.2588190451;   // grids valid up to 75 deg zenith
static const double kHitListSlack = 0.02;    // hit lists reach 2 % beyond 1/min_cos (refraction rotation)

static float f32_down(double v)
{
    float f = (float)v;
    if ((double)f > v) f = std::nextafterf(f, -INFINITY);
    return f;
}

static int build_grid(c8ph_ctx *ctx, int which, const std::vector<float> &tel, int mode, double min_cos,
                      double margin_max, DevGrid &g)
{
    const int n = (int)tel.size() / 4;
    double r_max = 0.0, rz_min = 1e300, coord_max = 0.0;
    for (int k = 0; k < n; ++k) {
        r_max = std::max(r_max, (double)tel[4 * k + 3]);
        rz_min = std::min(rz_min, (double)tel[4 * k + 3] + std::fabs((double)tel[4 * k + 2]));
        coord_max = std::max(coord_max, std::max(std::fabs((double)tel[4 * k]), std::fabs((double)tel[4 * k + 1])));
    }
    auto reach = [&](int k) {            // horizontal distance up to which telescope k is listed
        const double rz = (double)tel[4 * k + 3] + std::fabs((double)tel[4 * k + 2]);
        return mode == 0 ? rz / min_cos * (1.0 + kHitListSlack) : r_max / min_cos + margin_max;
    };
    double x0 = 1e300, y0 = 1e300, x1 = -1e300, y1 = -1e300;
    for (int k = 0; k < n; ++k) {
        const double rc = reach(k) * 1.001 + 1e-2;
        x0 = std::min(x0, tel[4 * k] - rc); x1 = std::max(x1, tel[4 * k] + rc);
        y0 = std::min(y0, tel[4 * k + 1] - rc); y1 = std::max(y1, tel[4 * k + 1] + rc);
    }
    const double ext = std::max(x1 - x0, y1 - y0);
    // cell size: about one telescope radius, but no more than ~4e6 list entries and 1536^2 cells
    double cs = mode == 0 ? 0.5 * rz_min : r_max;       // hit grid: half a radius (fewer false candidates; measured)
    {
        double area = 0.0;
        for (int k = 0; k < n; ++k) area += 3.14159265358979 * reach(k) * reach(k);
        cs = std::max(cs, std::sqrt(area / 4.0e6));
    }
    cs = std::max(cs, ext / 1536.0);
    if (!(cs > 0.0)) cs = 1.0;
    // fp32 rounding of (x - x0) * inv_cs on the device: a few ulp of the largest coordinate
    const double pad = 1e-3 * cs + 8.0 * (coord_max + ext + 8.0 * cs) * 1.2e-7 + 1e-4;
    if (mode == 0) {
        // hit grid: a ring of cells no telescope reaches around the footprint, so that the device may CLAMP the cell
        // coordinates of a point outside the grid instead of testing them (the ring cells are empty: checked below)
        const double ring = (1.0 + std::ceil(2.0 * pad / cs)) * cs;
        x0 -= ring; y0 -= ring; x1 += ring; y1 += ring;
    }
    const int nx = std::max(1, (int)std::ceil((x1 - x0) / cs)), ny = std::max(1, (int)std::ceil((y1 - y0) / cs));
    const size_t ncell = (size_t)nx * ny;
    struct Entry { uint32_t cell; float key; int k; };
    std::vector<Entry> ent;
    std::vector<float> near_d(mode == 1 ? ncell : 0, INFINITY);      // LV2: least dist(cell centre, centre_k) - r_k so far
    std::vector<int> near_k(mode == 1 ? ncell : 0, -1);
    ent.reserve((size_t)n * 64);
    for (int k = 0; k < n; ++k) {
        const double cx_ = tel[4 * k], cy_ = tel[4 * k + 1], rc = reach(k);
        const double rz = (double)tel[4 * k + 3] + std::fabs((double)tel[4 * k + 2]);
        const int a = std::max(0, (int)std::floor((cx_ - rc - pad - x0) / cs)), b = std::min(nx - 1, (int)std::floor((cx_ + rc + pad - x0) / cs));
        const int c = std::max(0, (int)std::floor((cy_ - rc - pad - y0) / cs)), d = std::min(ny - 1, (int)std::floor((cy_ + rc + pad - y0) / cs));
        for (int iy = c; iy <= d; ++iy)
            for (int ix = a; ix <= b; ++ix) {
                const double bx0 = x0 + ix * cs - pad, bx1 = x0 + (ix + 1) * cs + pad;
                const double by0 = y0 + iy * cs - pad, by1 = y0 + (iy + 1) * cs + pad;
                const double px = std::min(std::max(cx_, bx0), bx1), py = std::min(std::max(cy_, by0), by1);
                const double dist = std::sqrt((px - cx_) * (px - cx_) + (py - cy_) * (py - cy_));
                if (dist > rc) continue;
                if (mode == 1) {
                    // the telescope nearest to the cell: the device tests it in line before walking the list
                    const double mx_ = x0 + (ix + 0.5) * cs - cx_, my_ = y0 + (iy + 0.5) * cs - cy_;
                    const float dn = (float)(std::sqrt(mx_ * mx_ + my_ * my_) - (double)tel[4 * k + 3]);
                    const size_t ci = (size_t)iy * nx + ix;
                    if (dn < near_d[ci]) { near_d[ci] = dn; near_k[ci] = k; }
                }
                const double key = mode == 0 ? dist / rz : dist;
                ent.push_back({(uint32_t)((size_t)iy * nx + ix), f32_down(key * (1.0 - 1e-6)), k});
            }
    }
    std::sort(ent.begin(), ent.end(), [](const Entry &l, const Entry &r) {
        if (l.cell != r.cell) return l.cell < r.cell;
        if (l.key != r.key) return l.key < r.key;
        return l.k < r.k;
    });
    std::vector<int> start(ncell + 1, 0);
    std::vector<float> kmin(ncell, INFINITY);
    std::vector<float2> items(std::max<size_t>(1, ent.size()));
    for (const Entry &e : ent) start[e.cell + 1]++;
    for (size_t i = 1; i <= ncell; ++i) start[i] += start[i - 1];
    for (size_t i = 0; i < ent.size(); ++i) {
        float kb;
        memcpy(&kb, &ent[i].k, sizeof kb);
        items[i] = make_float2(ent[i].key, kb);
        if (ent[i].key < kmin[ent[i].cell]) kmin[ent[i].cell] = ent[i].key;
    }
    if (mode == 0 && n > 0) {
        bool ring_empty = nx >= 3 && ny >= 3;
        for (int ix = 0; ix < nx && ring_empty; ++ix)
            ring_empty = start[(size_t)ix + 1] == start[(size_t)ix] && start[(size_t)(ny - 1) * nx + ix + 1] == start[(size_t)(ny - 1) * nx + ix];
        for (int iy = 0; iy < ny && ring_empty; ++iy)
            ring_empty = start[(size_t)iy * nx + 1] == start[(size_t)iy * nx] && start[(size_t)iy * nx + nx] == start[(size_t)iy * nx + nx - 1];
        if (!ring_empty) return fail(ctx, C8PH_E_STATE, "set_detector: internal error, the border ring of the hit grid is not empty");
    }
    dfree(ctx->d_g_start[which]); dfree(ctx->d_g_items[which]); dfree(ctx->d_g_kmin[which]);
    CU(cudaMalloc(&ctx->d_g_start[which], start.size() * sizeof(int)));
    CU(cudaMalloc(&ctx->d_g_items[which], items.size() * sizeof(float2)));
    CU(cudaMalloc(&ctx->d_g_kmin[which], kmin.size() * sizeof(float)));
    CU(cudaMemcpy(ctx->d_g_start[which], start.data(), start.size() * sizeof(int), cudaMemcpyHostToDevice));
    CU(cudaMemcpy(ctx->d_g_items[which], items.data(), items.size() * sizeof(float2), cudaMemcpyHostToDevice));
    CU(cudaMemcpy(ctx->d_g_kmin[which], kmin.data(), kmin.size() * sizeof(float), cudaMemcpyHostToDevice));
    g.x0 = (float)x0; g.y0 = (float)y0; g.inv_cs = (float)(1.0 / cs); g.nx = nx; g.ny = ny;
    g.kmin = ctx->d_g_kmin[which]; g.start = ctx->d_g_start[which]; g.items = ctx->d_g_items[which];
    g.knear = nullptr;
    g.kq = nullptr;
    g.first = nullptr; g.first_kn = nullptr;
    if (mode == 0) {
        // hit pre-test: the smallest key of a cell in 1/64 steps, rounded down (conservative: a false candidate is
        // rejected by the exact search), one byte per cell so that the cells under the shower stay in L1
        std::vector<uint8_t> kq(ncell);
        for (size_t i = 0; i < ncell; ++i)
            kq[i] = std::isinf(kmin[i]) ? 255 : (uint8_t)std::min(254.0, std::floor((double)kmin[i] * kHitKeyScale));
        dfree(ctx->d_g_kq);
        CU(cudaMalloc(&ctx->d_g_kq, ncell));
        CU(cudaMemcpy(ctx->d_g_kq, kq.data(), ncell, cudaMemcpyHostToDevice));
        g.kq = ctx->d_g_kq;
        // the first listed telescope of every cell, in line (finish() tests it without walking the list)
        std::vector<float4> first(ncell, make_float4(0.f, 0.f, 0.f, 0.f));
        std::vector<int2> first_kn(ncell, make_int2(-1, 0));
        for (size_t i = 0; i < ncell; ++i)
            if (start[i + 1] > start[i]) {
                const int k = ent[start[i]].k;
                first[i] = make_float4(tel[4 * k], tel[4 * k + 1], tel[4 * k + 2], tel[4 * k + 3]);
                first_kn[i] = make_int2(k, start[i + 1] - start[i]);
            }
        dfree(ctx->d_g_first); dfree(ctx->d_g_first_kn);
        CU(cudaMalloc(&ctx->d_g_first, ncell * sizeof(float4)));
        CU(cudaMalloc(&ctx->d_g_first_kn, ncell * sizeof(int2)));
        CU(cudaMemcpy(ctx->d_g_first, first.data(), ncell * sizeof(float4), cudaMemcpyHostToDevice));
        CU(cudaMemcpy(ctx->d_g_first_kn, first_kn.data(), ncell * sizeof(int2), cudaMemcpyHostToDevice));
        g.first = ctx->d_g_first; g.first_kn = ctx->d_g_first_kn;
    }
    if (mode == 1) {
        std::vector<float4> kn(ncell);
        for (size_t i = 0; i < ncell; ++i) {
            const int k = near_k[i];
            kn[i] = k >= 0 ? make_float4(kmin[i], tel[4 * k], tel[4 * k + 1], tel[4 * k + 3]) : make_float4(INFINITY, 3.0e18f, 3.0e18f, 0.f);
        }
        dfree(ctx->d_g_knear);
        CU(cudaMalloc(&ctx->d_g_knear, ncell * sizeof(float4)));
        CU(cudaMemcpy(ctx->d_g_knear, kn.data(), ncell * sizeof(float4), cudaMemcpyHostToDevice));
        g.knear = ctx->d_g_knear;
    }
    return C8PH_OK;
}


static int setup_detector(c8ph_ctx *ctx, const c8ph_detector *d)
{
    DevDet &o = ctx->det;
    const int n = d->n_tel;
    std::vector<float> tel(d->tel_xyzr ? d->tel_xyzr : nullptr, d->tel_xyzr ? d->tel_xyzr + 4 * (size_t)n : nullptr);
    o.r_max = 0.f;
    for (int k = 0; k < n; ++k) o.r_max = std::max(o.r_max, tel[4 * k + 3]);
    if (n > 0) {
        const double min_cos = kGridMinCos;
        o.grid_min_cos = (float)(min_cos * (1.0 + 1e-4));
        o.use_grid = n > 8 ? 1 : 0;
        if (o.use_grid) {
            int rc = build_grid(ctx, 0, tel, 0, min_cos, 0.0, o.hit);
            if (rc) return rc;
            rc = build_grid(ctx, 1, tel, 1, min_cos, kLv2MarginMax, o.lv2);
            if (rc) return rc;
        }
    }
    return C8PH_OK;
}

extern "C" int c8ph_set_detector(c8ph_ctx *ctx, const c8ph_detector *d)
{
    if (!ctx) return C8PH_E_ARG;
    if (!d || d->size != sizeof(c8ph_detector)) return fail(ctx, C8PH_E_ARG, "set_detector: bad desc/size");
    if (d->hist_nx < 0 || d->hist_ny < 0 || (int64_t)d->hist_nx * d->hist_ny > (1ll << 30)) return fail(ctx, C8PH_E_ARG, "set_detector: hist size");
    if ((d->hist_nx > 0) != (d->hist_ny > 0) || (d->hist_nx > 0 && !(d->hist_cell > 0.f))) return fail(ctx, C8PH_E_ARG, "set_detector: hist grid");
    if (d->n_tel < 0 || d->n_tel >= (int)C8PH_TEL_NONE || (d->n_tel > 0 && !d->tel_xyzr)) return fail(ctx, C8PH_E_ARG, "set_detector: telescopes");
    if (d->cam_enabled && (d->n_tel != 1 || d->cam_rows < 1 || d->cam_cols < 1 || d->n_tbins < 1 || !(d->cam_pix_deg > 0.f) || !(d->t_bin_ns > 0.f)))
        return fail(ctx, C8PH_E_ARG, "set_detector: camera needs exactly one telescope, rows, cols, time bins");
    if (d->opt_enabled) {
        if (d->cam_enabled || d->n_tel < 1 || !(d->opt_focal_m > 0.f) || !(d->opt_mirror_radius_m > 0.f) || !(d->opt_camera_radius_m > 0.f))
            return fail(ctx, C8PH_E_ARG, "set_detector: optics need telescopes, focal length, mirror and camera radius; not with cam_enabled");
        if (d->opt_kind < 0 || d->opt_kind > 1 || d->opt_n_abs < 0 || d->opt_n_abs > 8)
            return fail(ctx, C8PH_E_ARG, "set_detector: opt_kind must be 0 or 1 and opt_n_abs in [0, 8]");
        for (int k = 0; k < d->opt_n_abs; ++k) {
            for (int j = 0; j < 7; ++j) if (!std::isfinite(d->opt_abs[k][j])) return fail(ctx, C8PH_E_ARG, "set_detector: absorber not finite");
            if (!(d->opt_abs[k][6] > 0.f)) return fail(ctx, C8PH_E_ARG, "set_detector: absorber radius <= 0");
        }
        if (d->opt_kind == 1) {
            const double Rl = d->opt_lens_roc_m, t = d->opt_lens_thickness_m, nl = d->opt_lens_index, rmv = d->opt_mirror_radius_m;
            if (!(Rl > 0.0) || !(t > 0.0) || !(t <= Rl) || !(nl > 1.0) || !(rmv * rmv <= Rl * Rl - (Rl - t) * (Rl - t) + 1e-9))
                return fail(ctx, C8PH_E_ARG, "set_detector: lens needs roc > 0, 0 < thickness <= roc, index > 1 and an aperture inside the cap");
        }
        const double f = d->opt_focal_m, rm = d->opt_mirror_radius_m, rc = d->opt_camera_radius_m;
        // lens: apex on the axis, rim of the plane face and rim of the camera must be inside the sphere
        const double need = d->opt_kind == 1 ? std::max(0.5 * f + (double)d->opt_lens_thickness_m, std::max(std::sqrt(0.25 * f * f + rm * rm), std::sqrt(0.25 * f * f + rc * rc))) : std::max(std::sqrt(0.25 * f * f + rc * rc), std::sqrt(std::pow(0.5 * f - rm * rm / (4.0 * f), 2) + rm * rm));
        for (int k = 0; k < d->n_tel; ++k)
            if (d->tel_xyzr[4 * k + 3] < need) return fail(ctx, C8PH_E_ARG, "set_detector: a bounding sphere does not contain the mirror and the camera");
    }
    CU(cudaSetDevice(ctx->device));
    DevDet o{};
    o.hist_nx = d->hist_nx; o.hist_ny = d->hist_ny;
    o.hist_x0 = d->hist_x0; o.hist_y0 = d->hist_y0; o.hist_cell = d->hist_nx > 0 ? d->hist_cell : 1.f;
    o.hist_inv_cell = 1.0f / o.hist_cell;
    o.n_tel = d->n_tel;
    double r_arr = 0.0;
    for (int k = 0; k < d->n_tel; ++k) {
        const float *t = d->tel_xyzr + 4 * k;
        if (!(t[3] > 0.f)) return fail(ctx, C8PH_E_ARG, "set_detector: telescope radius <= 0");
        r_arr = std::max(r_arr, std::sqrt((double)t[0] * t[0] + (double)t[1] * t[1] + (double)t[2] * t[2]) + t[3]);
    }
    if (d->hist_nx > 0 && !d->cam_enabled) {
        const double xs[2] = {d->hist_x0, (double)d->hist_x0 + d->hist_nx * (double)d->hist_cell};
        const double ys[2] = {d->hist_y0, (double)d->hist_y0 + d->hist_ny * (double)d->hist_cell};
        for (double x : xs) for (double y : ys) r_arr = std::max(r_arr, std::sqrt(x * x + y * y));
    }
    o.r_array = r_arr;
    o.cam_enabled = d->cam_enabled ? 1 : 0;
    o.cam_rows = d->cam_rows; o.cam_cols = d->cam_cols; o.n_tbins = d->n_tbins;
    {
        const double d2r = 3.14159265358979323846 / 180.0;
        const double az = d->cam_axis_az_deg * d2r, el = d->cam_axis_el_deg * d2r;
        const double w[3] = {std::cos(el) * std::cos(az), std::cos(el) * std::sin(az), std::sin(el)};
        const double r[3] = {-std::sin(az), std::cos(az), 0.0};
        const double u[3] = {w[1] * r[2] - w[2] * r[1], w[2] * r[0] - w[0] * r[2], w[0] * r[1] - w[1] * r[0]};
        for (int k = 0; k < 3; ++k) { o.cam_w[k] = (float)w[k]; o.cam_r[k] = (float)r[k]; o.cam_u[k] = (float)u[k]; }
        o.cam_pitch = (float)(d->cam_pix_deg * d2r);
        o.cam_inv_pitch = d->cam_pix_deg > 0.f ? (float)(1.0 / (d->cam_pix_deg * d2r)) : 0.f;
    }
    o.opt_enabled = d->opt_enabled ? 1 : 0;
    {
        const double d2r = 3.14159265358979323846 / 180.0;
        const double az = d->opt_az_deg * d2r, el = d->opt_el_deg * d2r;
        const double w[3] = {std::cos(el) * std::cos(az), std::cos(el) * std::sin(az), std::sin(el)};
        const double r[3] = {-std::sin(az), std::cos(az), 0.0};
        const double u[3] = {w[1] * r[2] - w[2] * r[1], w[2] * r[0] - w[0] * r[2], w[0] * r[1] - w[1] * r[0]};
        for (int k = 0; k < 3; ++k) { o.opt_w[k] = (float)w[k]; o.opt_r[k] = (float)r[k]; o.opt_u[k] = (float)u[k]; }
        o.opt_f = d->opt_focal_m; o.opt_rm2 = d->opt_mirror_radius_m * d->opt_mirror_radius_m;
        o.opt_rc2 = d->opt_camera_radius_m * d->opt_camera_radius_m;
        o.opt_kind = d->opt_kind; o.opt_n_abs = d->opt_enabled ? d->opt_n_abs : 0;
        o.opt_lens_roc = d->opt_lens_roc_m; o.opt_lens_t = d->opt_lens_thickness_m; o.opt_lens_n = d->opt_lens_index;
        for (int k = 0; k < 8; ++k) for (int j = 0; j < 7; ++j) o.opt_abs[k][j] = k < o.opt_n_abs ? d->opt_abs[k][j] : 0.f;
    }
    o.t_ref = d->t_ref_ns; o.t_bin = d->t_bin_ns; o.inv_t_bin = d->t_bin_ns > 0.f ? 1.0f / d->t_bin_ns : 0.f;
    dfree(ctx->d_tel);
    if (d->n_tel > 0) {
        CU(cudaMalloc(&ctx->d_tel, (size_t)d->n_tel * sizeof(float4)));
        CU(cudaMemcpy(ctx->d_tel, d->tel_xyzr, (size_t)d->n_tel * sizeof(float4), cudaMemcpyHostToDevice));
    }
    o.tel = ctx->d_tel;
    ctx->det = o;
    // the LV2 grid lists telescopes for margins up to kLv2MarginMax (checked in emit_propagate)
    int rc = setup_detector(ctx, d);
    if (rc) return rc;
    ctx->have_det = true;
    return C8PH_OK;
}

// ------------------------------------------------------------------------------------ wavelength tables
extern "C" int c8ph_set_line_spectrum(c8ph_ctx *ctx, int32_t n_lines, const float *line_nm, const float *line_cdf)
{
    if (!ctx) return C8PH_E_ARG;
    if (n_lines < 0 || n_lines > (1 << 20) || (n_lines > 0 && (!line_nm || !line_cdf))) return fail(ctx, C8PH_E_ARG, "set_line_spectrum: n_lines / NULL array");
    for (int k = 0; k < n_lines; ++k) {
        if (!(line_nm[k] > 0.f) || !std::isfinite(line_nm[k])) return fail(ctx, C8PH_E_ARG, "set_line_spectrum: wavelength <= 0 or not finite");
        if (!(line_cdf[k] >= 0.f && line_cdf[k] <= 1.f) || (k > 0 && line_cdf[k] < line_cdf[k - 1])) return fail(ctx, C8PH_E_ARG, "set_line_spectrum: cdf must rise from >= 0 to 1");
    }
    CU(cudaSetDevice(ctx->device));
    CU(cudaDeviceSynchronize());                               // nothing in flight may still read the old table
    dfree(ctx->d_lines);
    ctx->n_lines = 0;
    if (n_lines > 0) {
        CU(cudaMalloc(&ctx->d_lines, 2 * (size_t)n_lines * sizeof(float)));
        CU(cudaMemcpy(ctx->d_lines, line_nm, n_lines * sizeof(float), cudaMemcpyHostToDevice));
        CU(cudaMemcpy(ctx->d_lines + n_lines, line_cdf, n_lines * sizeof(float), cudaMemcpyHostToDevice));
        ctx->n_lines = n_lines;
    }
    return C8PH_OK;
}

extern "C" int c8ph_set_efficiency(c8ph_ctx *ctx, int32_t n_eff, float lambda0_nm, float dlambda_nm, const float *eff)
{
    if (!ctx) return C8PH_E_ARG;
    if (n_eff < 0 || n_eff > (1 << 20) || (n_eff > 0 && !eff) || (n_eff > 1 && !(dlambda_nm > 0.f)))
        return fail(ctx, C8PH_E_ARG, "set_efficiency: needs eff and dlambda_nm > 0");
    for (int k = 0; k < n_eff; ++k)
        if (!(eff[k] >= 0.f && eff[k] <= 1.f)) return fail(ctx, C8PH_E_ARG, "set_efficiency: efficiency outside [0,1]");
    CU(cudaSetDevice(ctx->device));
    CU(cudaDeviceSynchronize());
    dfree(ctx->d_eff);
    ctx->n_eff = 0;
    if (n_eff > 0) {
        CU(cudaMalloc(&ctx->d_eff, (size_t)n_eff * sizeof(float)));
        CU(cudaMemcpy(ctx->d_eff, eff, (size_t)n_eff * sizeof(float), cudaMemcpyHostToDevice));
        ctx->n_eff = n_eff; ctx->eff_l0 = lambda0_nm; ctx->eff_dl = dlambda_nm;
    }
    return C8PH_OK;
}

// ------------------------------------------------------------------------------------ the hot call
static int make_args(c8ph_ctx *ctx, const c8ph_segments *s, int64_t n_seg, int64_t base, const c8ph_params *p,
                     uint64_t seed, const c8ph_outputs *o, KArgs &a)
{
    if (!s || s->size != sizeof(c8ph_segments) || !p || p->size != sizeof(c8ph_params) || !o || o->size != sizeof(c8ph_outputs))
        return fail(ctx, C8PH_E_ARG, "emit_propagate: NULL struct or size mismatch");
    if (n_seg < 0 || base < 0) return fail(ctx, C8PH_E_ARG, "emit_propagate: negative n_segments / seg_id_base");
    if (n_seg > 0x7FFFFFFFll) return fail(ctx, C8PH_E_ARG, "emit_propagate: more than 2^31-1 segments per call (photon records carry a 32-bit segment index); split the call");
    if (!ctx->have_atm) return fail(ctx, C8PH_E_STATE, "emit_propagate: atmosphere not initialised");
    if (!ctx->have_det) return fail(ctx, C8PH_E_STATE, "emit_propagate: detector not set");
    if (n_seg > 0 && (!s->x || !s->y || !s->z || !s->dx || !s->dy || !s->dz || !s->len || !s->beta || !s->t0 || !s->charge))
        return fail(ctx, C8PH_E_ARG, "emit_propagate: NULL segment array");
    if (p->emit != C8PH_EMIT_CHERENKOV && p->emit != C8PH_EMIT_FLUORESCENCE) return fail(ctx, C8PH_E_ARG, "emit_propagate: emit");
    if (p->trace < C8PH_TRACE_STRAIGHT || p->trace > C8PH_TRACE_TABLE) return fail(ctx, C8PH_E_ARG, "emit_propagate: trace");
    if (p->trans < C8PH_TRANS_OFF || p->trans > C8PH_TRANS_ROULETTE) return fail(ctx, C8PH_E_ARG, "emit_propagate: trans");
    if (p->write < C8PH_WRITE_NONE || p->write > C8PH_WRITE_TEL) return fail(ctx, C8PH_E_ARG, "emit_propagate: write");
    if (!(p->bunch_weight > 0.f)) return fail(ctx, C8PH_E_ARG, "emit_propagate: bunch_weight <= 0");
    if (!o->counters) return fail(ctx, C8PH_E_ARG, "emit_propagate: counters is NULL");
    if (o->photons && o->photon_capacity < 0) return fail(ctx, C8PH_E_ARG, "emit_propagate: photon_capacity");
    if (p->trace == C8PH_TRACE_TABLE && !ctx->have_table) return fail(ctx, C8PH_E_STATE, "emit_propagate: trace table not built");
    if (p->trace == C8PH_TRACE_NUMERIC && ctx->atm.model >= C8PH_ATM_SPHERICAL)
        return fail(ctx, C8PH_E_ARG, "emit_propagate: per-photon numeric tracing is planar only; use the table in the spherical / cylindrical model");
    if (ctx->atm.model == C8PH_ATM_CYLINDRICAL && p->trace == C8PH_TRACE_TABLE && ctx->have_table && ctx->tab.n_c < 2)
        return fail(ctx, C8PH_E_STATE, "emit_propagate: the cylindrical model needs a trace table built with n_c >= 2");
    if (ctx->atm.model == C8PH_ATM_CYLINDRICAL && p->emit == C8PH_EMIT_FLUORESCENCE)
        return fail(ctx, C8PH_E_ARG, "emit_propagate: fluorescence is not available in the cylindrical model");
    if (p->trace == C8PH_TRACE_NUMERIC && p->emit == C8PH_EMIT_FLUORESCENCE) return fail(ctx, C8PH_E_ARG, "emit_propagate: fluorescence + numeric tracing");
    if (p->emit == C8PH_EMIT_CHERENKOV && !(p->lambda_min_nm > 0.f && p->lambda_max_nm > p->lambda_min_nm))
        return fail(ctx, C8PH_E_ARG, "emit_propagate: wavelength band");
    if (ctx->det.opt_enabled && p->write == C8PH_WRITE_ALL)
        return fail(ctx, C8PH_E_ARG, "emit_propagate: WRITE_ALL is not defined with last-mile optics (records are camera hits)");
    if (!(p->disp_b_nm2 >= 0.f) || (p->disp_b_nm2 > 0.f && !(p->disp_lambda0_nm > 0.f)))
        return fail(ctx, C8PH_E_ARG, "emit_propagate: dispersion needs disp_b_nm2 >= 0 and disp_lambda0_nm > 0");
    if (p->use_efficiency && ctx->n_eff < 1) return fail(ctx, C8PH_E_STATE, "emit_propagate: use_efficiency without c8ph_set_efficiency");
    if (p->use_efficiency && p->trans == C8PH_TRANS_OFF) return fail(ctx, C8PH_E_ARG, "emit_propagate: the efficiency table needs a transmission mode");
    if (p->emit == C8PH_EMIT_FLUORESCENCE) {
        if (ctx->det.n_tel < 1) return fail(ctx, C8PH_E_STATE, "emit_propagate: fluorescence needs a telescope to aim at");
        if (ctx->n_lines < 1) return fail(ctx, C8PH_E_STATE, "emit_propagate: fluorescence needs c8ph_set_line_spectrum");
        if (n_seg > 0 && !s->edep) return fail(ctx, C8PH_E_ARG, "emit_propagate: edep is NULL");
    }
    if (p->filter_lv2 && (!(p->lv2_margin_m >= 0.f) || (p->lv2_margin_m > (float)kLv2MarginMax && ctx->det.use_grid)))
        return fail(ctx, C8PH_E_ARG, "emit_propagate: lv2_margin_m must be in [0, 64] m (range covered by the LV2 grid)");
    a.atm = ctx->atm;
    a.tab = ctx->tab;
    a.det = ctx->det;
    if (ctx->force_brute) a.det.use_grid = 0;
    DevRun &r = a.run;
    r.emit = p->emit; r.trace = p->trace; r.trans = p->trans; r.write = p->write;
    r.lv1 = p->filter_lv1 ? 1 : 0; r.lv2 = p->filter_lv2 ? 1 : 0;
    r.il1 = p->emit == C8PH_EMIT_CHERENKOV ? 1.0f / p->lambda_min_nm : 0.f;
    r.il2 = p->emit == C8PH_EMIT_CHERENKOV ? 1.0f / p->lambda_max_nm : 0.f;
    r.w = p->bunch_weight;
    r.yield_k = p->emit == C8PH_EMIT_CHERENKOV
                    ? 2.0 * 3.14159265358979323846 / 137.035999 * (1.0 / ((double)p->lambda_min_nm * 1e-9) - 1.0 / ((double)p->lambda_max_nm * 1e-9))
                    : 0.0;
    r.lv1_margin = p->lv1_margin_rad; r.lv2_margin = p->lv2_margin_m;
    {
        // LV2 keep-box: the histogram extent widened by the margin, in the fp32 arithmetic of the test
        const DevDet &dd = ctx->det;
        const bool geom = dd.hist_nx > 0 && !dd.cam_enabled;
        const float m = p->lv2_margin_m;
        const float hx1 = dd.hist_x0 + (float)dd.hist_nx * dd.hist_cell, hy1 = dd.hist_y0 + (float)dd.hist_ny * dd.hist_cell;
        r.box_x0 = geom ? dd.hist_x0 - m : INFINITY; r.box_x1 = geom ? hx1 + m : -INFINITY;
        r.box_y0 = geom ? dd.hist_y0 - m : INFINITY; r.box_y1 = geom ? hy1 + m : -INFINITY;
    }
    r.fluor_yield = p->fluor_yield_per_MeV; r.aim_factor = p->aim_factor;
    r.inv_Rg = (float)(1.0 / ctx->atm.Rg);
    {
        // relative change of 1/|u_z| by the refraction rotation: <= (n_e - n_g)/n_g tan^2(zenith) plus
        // the spherical term, at the grid's zenith limit; the hit lists are built for 2 % (kHitListSlack)
        const double tan2 = 1.0 / (kGridMinCos * kGridMinCos) - 1.0;
        const double infl = 1.0 + 2.0 * ctx->eta_span * tan2 + 1e-3;
        r.hit_infl = (float)infl;
        r.hit_brute = (p->trace != C8PH_TRACE_STRAIGHT && infl > 1.0 + 0.9 * kHitListSlack) ? 1 : 0;
        if (p->trace == C8PH_TRACE_STRAIGHT) r.hit_infl = 1.0f + 1e-5f;
    }
    r.n_lines = 0; r.line_nm = nullptr; r.line_cdf = nullptr;
    r.force_generic = ctx->force_generic ? 1 : 0;
    if (p->flat_plane < 0 || p->flat_plane > 2) return fail(ctx, C8PH_E_ARG, "emit_propagate: flat_plane must be 0, 1 or 2");
    r.flat_plane = (p->flat_plane && ctx->atm.model == C8PH_ATM_SPHERICAL && p->trace != C8PH_TRACE_STRAIGHT) ? p->flat_plane : 0;
    if (r.flat_plane == 2 && (p->trace != C8PH_TRACE_TABLE || ctx->tab.n_rho < 2))
        return fail(ctx, C8PH_E_STATE, "emit_propagate: flat_plane = 2 needs table tracing and a trace table built with n_rho >= 2");
    r.n_eff = p->use_efficiency ? ctx->n_eff : 0; r.eff = p->use_efficiency ? ctx->d_eff : nullptr;
    r.eff_l0 = ctx->eff_l0; r.eff_inv_dl = ctx->n_eff > 1 ? 1.0f / ctx->eff_dl : 0.f;
    r.disp_b = p->emit == C8PH_EMIT_CHERENKOV ? p->disp_b_nm2 : 0.f;
    r.disp_k0sq = r.disp_b > 0.f ? 1.0 / ((double)p->disp_lambda0_nm * (double)p->disp_lambda0_nm) : 0.0;
    r.disp_c0 = (float)(1.0 - (double)r.disp_b * r.disp_k0sq);
    r.il1_d = p->emit == C8PH_EMIT_CHERENKOV ? 1.0 / (double)p->lambda_min_nm : 0.0;
    r.il2_d = p->emit == C8PH_EMIT_CHERENKOV ? 1.0 / (double)p->lambda_max_nm : 0.0;
    if (p->emit == C8PH_EMIT_FLUORESCENCE) { r.n_lines = ctx->n_lines; r.line_nm = ctx->d_lines; r.line_cdf = ctx->d_lines + ctx->n_lines; }
    for (int k = 0; k < 10; ++k) {
        r.key0[k] = (uint32_t)seed + (uint32_t)k * 0x9E3779B9u;
        r.key1[k] = (uint32_t)(seed >> 32) + (uint32_t)k * 0xBB67AE85u;
    }
    r.n_seg = n_seg; r.seg_id_base = base; r.local_base = 0;
    r.seg = *s; r.out = *o;
    r.cursor = ctx->d_cursor;
    r.slots = ctx->d_slots;
    r.qring = static_cast<unsigned char *>(ctx->d_slots) + segment_slot_bytes(ctx->n_sm);
    const long long warps = (long long)ctx->n_sm * 2 * 8;
    long long g = n_seg / (warps * 4);
    r.segs_per_grab = (int)std::min<long long>(32, std::max<long long>(1, g));
    {
        HotConst &h = a.hc;
        for (int k = 0; k < 10; ++k) h.key[k] = make_uint2(r.key0[k], r.key1[k]);
        h.eta_h0 = a.atm.h0; h.eta_inv_dh = a.atm.inv_dh; h.eta_fmax = a.atm.f_max; h.eta_kmax = a.atm.n_nodes - 2;
        h.eta = a.atm.eta; h.il1 = r.il1; h.dil = r.il1 - r.il2;
        h.box_x0 = r.box_x0; h.box_x1 = r.box_x1; h.box_y0 = r.box_y0; h.box_y1 = r.box_y1;
        h.lv2_margin = r.lv2_margin; h.r_max = a.det.r_max; h.grid_min_cos = a.det.grid_min_cos; h.hit_infl_q = r.hit_infl * kHitKeyScale;
        h.ray_lambda = a.atm.ray_lambda; h.ray_k = (float)(1.4426950408889634 * (double)a.atm.ray_inv_X); h.w = r.w; h.pad0 = 0.f;
        h.hit_x0 = a.det.hit.x0; h.hit_y0 = a.det.hit.y0; h.hit_inv_cs = a.det.hit.inv_cs; h.hit_nx = a.det.hit.nx;
        h.hit_ny = a.det.hit.ny; h.hist_inv_cell = a.det.hist_inv_cell; h.hist_nx = a.det.hist_nx; h.hist_ny = a.det.hist_ny;
        h.hit_kq = a.det.hit.kq; h.hist = r.out.hist;
    }
    if (emit_smem_bytes(a) > 200 * 1024) return fail(ctx, C8PH_E_ARG, "emit_propagate: atmosphere table too large for shared memory");
    return C8PH_OK;
}

// Launches of one context share the work cursor and the prepared-segment slots: a launch on another stream than the
// previous one first waits for that one's end event (a capturing stream is left alone: see c8ph.h).
static int order_after_last_launch(c8ph_ctx *ctx, cudaStream_t st)
{
    if (ctx->have_launch && st != ctx->last_stream) {
        cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
        if (cudaStreamIsCapturing(st, &cs) != cudaSuccess) { cudaGetLastError(); cs = cudaStreamCaptureStatusNone; }
        if (cs == cudaStreamCaptureStatusNone) CU(cudaStreamWaitEvent(st, ctx->ev_done, 0));
    }
    return C8PH_OK;
}
static int mark_launch_end(c8ph_ctx *ctx, cudaStream_t st)
{
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(st, &cs) != cudaSuccess) { cudaGetLastError(); cs = cudaStreamCaptureStatusNone; }
    if (cs == cudaStreamCaptureStatusNone) {
        CU(cudaEventRecord(ctx->ev_done, st));
        ctx->last_stream = st; ctx->have_launch = true;
    }
    return C8PH_OK;
}

static int launch(c8ph_ctx *ctx, const KArgs &a, cudaStream_t st)
{
    int rc = order_after_last_launch(ctx, st);
    if (rc) return rc;
    CU(cudaMemsetAsync(ctx->d_cursor, 0, sizeof(unsigned long long), st));
    CU(cudaEventRecord(ctx->ev0, st));
    cudaError_t e = launch_emit_propagate(a, ctx->n_sm, st);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "emit_propagate launch");
    CU(cudaEventRecord(ctx->ev1, st));
    ctx->timed = true;
    ctx->launches++;
    return mark_launch_end(ctx, st);
}

extern "C" int c8ph_emit_propagate(c8ph_ctx *ctx, const c8ph_segments *s, int64_t n_seg, int64_t base,
                                   const c8ph_params *p, uint64_t seed, const c8ph_outputs *o, void *stream)
{
    if (!ctx) return C8PH_E_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    CU(cudaSetDevice(ctx->device));
    KArgs a{};
    int rc = make_args(ctx, s, n_seg, base, p, seed, o, a);
    if (rc) return rc;
    if (n_seg == 0) return C8PH_OK;
    return launch(ctx, a, st);
}

// HOST-buffer path.  The call is split into chunks of segments and pipelined over three streams:
// H2D of chunk c+1 | kernel of chunk c | D2H of the photons chunk c-1 wrote, so the PCIe transfer of
// the photon list (the dominant cost) overlaps the kernel.  Chunks run in order on one
// stream, each with seg_id_base = base + offset: the photons are those of a single call.
extern "C" int c8ph_emit_propagate_host(c8ph_ctx *ctx, const c8ph_segments *hs, int64_t n_seg, int64_t base,
                                        const c8ph_params *p, uint64_t seed, const c8ph_outputs *ho)
{
    if (!ctx) return C8PH_E_ARG;
    if (!hs || hs->size != sizeof(c8ph_segments) || !ho || ho->size != sizeof(c8ph_outputs) || n_seg < 0)
        return fail(ctx, C8PH_E_ARG, "emit_propagate_host: NULL struct or size mismatch");
    if (!ctx->have_det) return fail(ctx, C8PH_E_STATE, "emit_propagate_host: detector not set");
    CU(cudaSetDevice(ctx->device));
    if (!ctx->st_h2d) {
        CU(cudaStreamCreateWithFlags(&ctx->st_h2d, cudaStreamNonBlocking));
        CU(cudaStreamCreateWithFlags(&ctx->st_run, cudaStreamNonBlocking));
        CU(cudaStreamCreateWithFlags(&ctx->st_d2h, cudaStreamNonBlocking));
        CU(cudaHostAlloc(&ctx->h_written, (kMaxChunks + C8PH_N_COUNTERS) * sizeof(unsigned long long), cudaHostAllocDefault));
        for (int c = 0; c < kMaxChunks; ++c) {
            CU(cudaEventCreateWithFlags(&ctx->ev_in[c], cudaEventDisableTiming));
            CU(cudaEventCreateWithFlags(&ctx->ev_run[c], cudaEventDisableTiming));
        }
    }
    const float *src[11] = {hs->x, hs->y, hs->z, hs->dx, hs->dy, hs->dz, hs->len, hs->beta, hs->t0, hs->charge, hs->edep};
    const size_t n = (size_t)n_seg, npad = (n + 63) & ~(size_t)63;
    if (11 * npad > ctx->seg_cap) {
        dfree(ctx->d_seg);
        CU(cudaMalloc(&ctx->d_seg, std::max<size_t>(1, 11 * npad) * sizeof(float)));
        ctx->seg_cap = 11 * npad;
    }
    if (hs->id && n > ctx->ids_cap) {
        dfree(ctx->d_ids);
        CU(cudaMalloc(&ctx->d_ids, n * sizeof(uint64_t)));
        ctx->ids_cap = n;
    }
    // device outputs in one arena: counters | hist | tel_counts | photon_weight | photons
    const DevDet &det = ctx->det;
    const size_t n_hist = ho->hist ? (det.cam_enabled ? (size_t)det.cam_rows * det.cam_cols * det.n_tbins : (size_t)det.hist_nx * det.hist_ny) : 0;
    const size_t n_tel = ho->tel_counts ? (size_t)det.n_tel : 0;
    const size_t cap = ho->photons ? (size_t)std::max<int64_t>(0, ho->photon_capacity) : 0;
    auto up = [](size_t v) { return (v + 255) & ~(size_t)255; };
    const size_t off_hist = up(C8PH_N_COUNTERS * sizeof(uint64_t));
    const size_t off_tel = off_hist + up(n_hist * sizeof(float));
    const size_t off_w = off_tel + up(n_tel * sizeof(float));
    const size_t off_ph = off_w + up((ho->photon_weight ? cap : 0) * sizeof(float));
    const size_t total = off_ph + up(cap * sizeof(c8ph_photon));
    if (total > ctx->out_cap) {
        if (ctx->d_out) cudaFree(ctx->d_out);
        ctx->d_out = nullptr;
        CU(cudaMalloc(&ctx->d_out, total));
        ctx->out_cap = total;
    }
    char *b = (char *)ctx->d_out;
    cudaStream_t s_in = ctx->st_h2d, s_run = ctx->st_run, s_out = ctx->st_d2h;
    CU(cudaMemsetAsync(b, 0, off_w, s_run));                // counters, hist, tel_counts
    c8ph_outputs dout{};
    dout.size = sizeof(dout);
    dout.counters = (uint64_t *)b;
    dout.hist = n_hist ? (float *)(b + off_hist) : nullptr;
    dout.tel_counts = n_tel ? (float *)(b + off_tel) : nullptr;
    dout.photon_weight = (ho->photon_weight && cap) ? (float *)(b + off_w) : nullptr;
    dout.photons = cap ? (c8ph_photon *)(b + off_ph) : nullptr;
    dout.photon_capacity = (int64_t)cap;

    // chunk plan: at most kMaxChunks, at least 2^18 segments each (keeps the persistent grid busy)
    int n_chunks = (int)std::min<size_t>(kMaxChunks, std::max<size_t>(1, n / (1u << 18)));
    if (!cap) n_chunks = 1;                                 // nothing to overlap without a photon list
    const size_t chunk = ((n + n_chunks - 1) / n_chunks + 63) & ~(size_t)63;
    bool first = true;
    for (int c = 0; c < n_chunks; ++c) {
        const size_t lo = std::min(n, (size_t)c * chunk), hi = std::min(n, lo + chunk);
        for (int k = 0; k < 11; ++k)
            if (src[k] && hi > lo)
                CU(cudaMemcpyAsync(ctx->d_seg + k * npad + lo, src[k] + lo, (hi - lo) * sizeof(float), cudaMemcpyHostToDevice, s_in));
        if (hs->id && hi > lo) CU(cudaMemcpyAsync(ctx->d_ids + lo, hs->id + lo, (hi - lo) * sizeof(uint64_t), cudaMemcpyHostToDevice, s_in));
        CU(cudaEventRecord(ctx->ev_in[c], s_in));
        CU(cudaStreamWaitEvent(s_run, ctx->ev_in[c], 0));
        c8ph_segments ds{};
        ds.size = sizeof(ds);
        const float **dp[11] = {&ds.x, &ds.y, &ds.z, &ds.dx, &ds.dy, &ds.dz, &ds.len, &ds.beta, &ds.t0, &ds.charge, &ds.edep};
        for (int k = 0; k < 11; ++k) *dp[k] = src[k] ? ctx->d_seg + k * npad + lo : nullptr;
        ds.id = hs->id ? ctx->d_ids + lo : nullptr;
        KArgs a{};
        int rc = make_args(ctx, &ds, (int64_t)(hi - lo), base + (int64_t)lo, p, seed, &dout, a);
        if (rc) { cudaDeviceSynchronize(); return rc; }
        a.run.local_base = (uint32_t)lo;
        if (hi > lo) {
            if (first) { rc = order_after_last_launch(ctx, s_run); if (rc) { cudaDeviceSynchronize(); return rc; } }
            CU(cudaMemsetAsync(ctx->d_cursor, 0, sizeof(unsigned long long), s_run));
            if (first) CU(cudaEventRecord(ctx->ev0, s_run));
            first = false;
            cudaError_t e = launch_emit_propagate(a, ctx->n_sm, s_run);
            if (e != cudaSuccess) { cudaDeviceSynchronize(); return cuda_fail(ctx, e, "emit_propagate launch"); }
            ctx->launches++;
        }
        CU(cudaMemcpyAsync(&ctx->h_written[c], &dout.counters[C8PH_CNT_WRITTEN], sizeof(unsigned long long), cudaMemcpyDeviceToHost, s_run));
        CU(cudaEventRecord(ctx->ev_run[c], s_run));
    }
    if (!first) { CU(cudaEventRecord(ctx->ev1, s_run)); ctx->timed = true; int rc2 = mark_launch_end(ctx, s_run); if (rc2) return rc2; }
    // photons: as soon as a chunk's kernel is done its records [written before, written after) go home
    size_t done = 0;
    for (int c = 0; c < n_chunks && cap; ++c) {
        CU(cudaEventSynchronize(ctx->ev_run[c]));
        const size_t w = (size_t)std::min<unsigned long long>(ctx->h_written[c], cap);
        if (w > done) {
            CU(cudaMemcpyAsync(ho->photons + done, dout.photons + done, (w - done) * sizeof(c8ph_photon), cudaMemcpyDeviceToHost, s_out));
            if (dout.photon_weight) CU(cudaMemcpyAsync(ho->photon_weight + done, dout.photon_weight + done, (w - done) * sizeof(float), cudaMemcpyDeviceToHost, s_out));
            done = w;
        }
    }
    // the small results follow the last kernel on the run stream (counters through pinned memory)
    uint64_t *cnt = reinterpret_cast<uint64_t *>(ctx->h_written + kMaxChunks);
    CU(cudaMemcpyAsync(cnt, dout.counters, C8PH_N_COUNTERS * sizeof(uint64_t), cudaMemcpyDeviceToHost, s_run));
    if (n_hist) CU(cudaMemcpyAsync(ho->hist, dout.hist, n_hist * sizeof(float), cudaMemcpyDeviceToHost, s_run));
    if (n_tel) CU(cudaMemcpyAsync(ho->tel_counts, dout.tel_counts, n_tel * sizeof(float), cudaMemcpyDeviceToHost, s_run));
    CU(cudaStreamSynchronize(s_run));
    CU(cudaStreamSynchronize(s_out));
    if (ho->counters) memcpy(ho->counters, cnt, C8PH_N_COUNTERS * sizeof(uint64_t));
    return C8PH_OK;
}

// ------------------------------------------------------------------------------------ sub-stepping
static int substep_args(c8ph_ctx *ctx, const c8ph_segments *t, const float *p_GeV, int64_t n, const c8ph_substep_desc *d,
                        SubstepArgs &a)
{
    if (!t || t->size != sizeof(c8ph_segments) || !d || d->size != sizeof(c8ph_substep_desc))
        return fail(ctx, C8PH_E_ARG, "substep: NULL struct or size mismatch");
    if (n < 0 || substep_scratch_elems(n) > kSubstepBlockSums) return fail(ctx, C8PH_E_ARG, "substep: n_tracks out of range (<= 2^27 per call)");
    if (n > 0 && (!t->x || !t->y || !t->z || !t->dx || !t->dy || !t->dz || !t->len || !t->beta || !t->t0 || !t->charge || !p_GeV))
        return fail(ctx, C8PH_E_ARG, "substep: NULL track array");
    if (!(d->tol_m > 0.f) || d->max_sub < 1 || d->max_sub > (1 << 20)) return fail(ctx, C8PH_E_ARG, "substep: tol_m > 0 and 1 <= max_sub <= 2^20 required");
    if (d->ms_enabled) {
        if (!ctx->have_atm) return fail(ctx, C8PH_E_STATE, "substep: multiple scattering needs the atmosphere (overburden) of the context");
        if (!(d->ms_X0_gcm2 > 0.f) || !(d->ms_max_step_m >= 0.f) || d->track_id_base < 0)
            return fail(ctx, C8PH_E_ARG, "substep: ms_X0_gcm2 > 0, ms_max_step_m >= 0 and track_id_base >= 0 required");
    }
    a.trk = *t; a.p_GeV = p_GeV; a.n = n;
    for (int k = 0; k < 3; ++k) a.B[k] = d->B_tesla[k];
    a.Bn = std::sqrt(a.B[0] * a.B[0] + a.B[1] * a.B[1] + a.B[2] * a.B[2]);
    a.tol = d->tol_m; a.max_sub = d->max_sub;
    a.ms_enabled = d->ms_enabled ? 1 : 0; a.ms_max_step = d->ms_max_step_m; a.ms_X0 = d->ms_X0_gcm2;
    a.id_base = d->track_id_base;
    a.clipped = reinterpret_cast<unsigned long long *>(d->clipped);
    for (int k = 0; k < 10; ++k)
        a.key[k] = make_uint2((uint32_t)d->seed + (uint32_t)k * 0x9E3779B9u, (uint32_t)(d->seed >> 32) + (uint32_t)k * 0xBB67AE85u);
    if (ctx->have_atm) a.atm = ctx->atm;
    return C8PH_OK;
}

extern "C" int c8ph_substep_plan(c8ph_ctx *ctx, const c8ph_segments *t, const float *p_GeV, int64_t n,
                                 const c8ph_substep_desc *d, int64_t *offsets, void *stream)
{
    if (!ctx) return C8PH_E_ARG;
    SubstepArgs a{};
    int rc = substep_args(ctx, t, p_GeV, n, d, a);
    if (rc) return rc;
    if (!offsets) return fail(ctx, C8PH_E_ARG, "substep_plan: offsets is NULL");
    CU(cudaSetDevice(ctx->device));
    a.offsets = reinterpret_cast<long long *>(offsets);
    if (n == 0) { CU(cudaMemsetAsync(offsets, 0, sizeof(int64_t), (cudaStream_t)stream)); return C8PH_OK; }
    cudaError_t e = launch_substep_plan(a, ctx->d_bsums, (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "substep_plan launch");
    ctx->launches += 3;
    return C8PH_OK;
}

extern "C" int c8ph_substep_fill(c8ph_ctx *ctx, const c8ph_segments *t, const float *p_GeV, int64_t n,
                                 const c8ph_substep_desc *d, const int64_t *offsets, const c8ph_segments_out *out, void *stream)
{
    if (!ctx) return C8PH_E_ARG;
    SubstepArgs a{};
    int rc = substep_args(ctx, t, p_GeV, n, d, a);
    if (rc) return rc;
    if (!offsets || !out || out->size != sizeof(c8ph_segments_out) || !out->x || !out->y || !out->z || !out->dx || !out->dy ||
        !out->dz || !out->len || !out->beta || !out->t0 || !out->charge)
        return fail(ctx, C8PH_E_ARG, "substep_fill: NULL offsets / output array or size mismatch");
    if (n == 0) return C8PH_OK;
    CU(cudaSetDevice(ctx->device));
    a.offsets = const_cast<long long *>(reinterpret_cast<const long long *>(offsets));
    a.out = *out;
    cudaError_t e = launch_substep_fill(a, ctx->n_sm, (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "substep_fill launch");
    ctx->launches++;
    return C8PH_OK;
}

extern "C" float c8ph_last_kernel_ms(c8ph_ctx *ctx)
{
    if (!ctx || !ctx->timed) return -1.f;
    if (cudaEventSynchronize(ctx->ev1) != cudaSuccess) return -1.f;
    float ms = -1.f;
    if (cudaEventElapsedTime(&ms, ctx->ev0, ctx->ev1) != cudaSuccess) return -1.f;
    return ms;
}

extern "C" int64_t c8ph_launch_count(const c8ph_ctx *ctx) { return ctx ? ctx->launches : 0; }

extern "C" const char *c8ph_counter_name(int i)
{
    static const char *names[C8PH_N_COUNTERS] = {
        "segments", "seg_below_threshold", "seg_lv1", "seg_emitting", "emitted", "upgoing", "lv2", "table_range",
        "roulette", "landed", "in_grid", "tel_hit", "cam_hit", "written", "overflow", "clipped", "nonfinite"};
    return (i >= 0 && i < C8PH_N_COUNTERS) ? names[i] : "";
}
