// mm_api.cu -- the C ABI of libmm (include/mm.h): context, validation, buffer ownership, kernel dispatch.
// All arithmetic of the hot path lives in the kernels (mm_coef.cuh = default; mm_stream.cuh, mm_tile.cuh,
// mm_generic.cuh = variants / fallback for other grids; mm_rk2.cuh, mm_local.cuh = SURVEY.md 8(f) NEXT-1, NEXT-3);
// this file only validates, marshals arguments and launches.  There is no CPU fallback.
#include "mm_ctx.cuh"

#include "mm_generic.cuh"
#include "mm_local.cuh"
#include "mm_spread.cuh"
#include "mm_free.cuh"
#include "mm_peak.cuh"

thread_local std::string g_create_err;

// what MM_OPT_KERNEL = 0 picks where the grid and flags allow a fast kernel (measured)
#ifndef MM_AUTO_KERNEL
#define MM_AUTO_KERNEL 5
#endif

// ---- S8 positivity bound (only with MM_FLAG_CHECK_DT) -----------------------------------------
template <typename real>
__global__ void check_dt_kernel(const __grid_constant__ KParams<real> kp, unsigned int *flag)
{
    const int plane = kp.nxi * kp.neta;
    const int64_t total = kp.nc * (int64_t)kp.ns * plane;
    for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total;
         idx += (int64_t)gridDim.x * blockDim.x) {
        const int64_t c = idx / ((int64_t)kp.ns * plane);
        int rem = (int)(idx - c * (int64_t)kp.ns * plane);
        const int j = rem / plane; rem -= j * plane;
        const int a = rem / kp.neta, b = rem - a * kp.neta;
        const int kth = (int)(c % kp.ntheta);
        const double ct = kp.cos_t[kth], st = kp.sin_t[kth], U = kp.U[c], V = kp.V[c], Om = kp.Om[c];
        const double R = kp.R, dxi = kp.dxi, deta = kp.deta;
        const double sj = (double)kp.s_lo + (j + 0.5) * (double)kp.ds;
        const double xi = -R + (a + 0.5) * dxi, eta = -R + (b + 0.5) * deta;
        auto w = [&](double x, double e) { return walk_speed<double>(kp.v0, kp.kload, ct, st, x, e); };
        const double Axh = U + w(xi + 0.5 * dxi, eta) * ct - sj * Om * st, Axl = U + w(xi - 0.5 * dxi, eta) * ct - sj * Om * st;
        const double Aeh = V + w(xi, eta + 0.5 * deta) * st + sj * Om * ct, Ael = V + w(xi, eta - 0.5 * deta) * st + sj * Om * ct;
        const bool endc = (j < kp.n_end) || (j >= kp.ns - kp.n_end);
        const double kap = (double)kp.kappa[rem] * (endc ? 1.0 + (double)kp.dt_endx / (double)kp.dt : 1.0);
        const double rate = w(xi, eta) / (double)kp.ds + (fmax(Axh, 0.0) - fmin(Axl, 0.0)) / dxi +
                            (fmax(Aeh, 0.0) - fmin(Ael, 0.0)) / deta + kap;
        if (!(1.0 - (double)kp.dt * rate >= 0.0)) *flag = 1u;
    }
}

template <typename real>
static mm_status launch_generic(mm_ctx *c, double dt, const void *in, void *out)
{
    KParams<real> kp = make_kparams<real>(c, dt);
    int64_t blocks = (c->cells + 255) / 256;
    const int64_t cap = (int64_t)c->sm_count * 64;
    if (blocks > cap) blocks = cap;
    substep_generic_kernel<real><<<(unsigned)blocks, 256, 0, c->stream>>>(kp, (const real *)in, (real *)out);
    CUDA_TRY(c, cudaGetLastError());
    c->launches++;
    snprintf(c->kname, sizeof c->kname, "generic<%s>", sizeof(real) == 8 ? "f64" : "f32");
    return MM_OK;
}

template <typename real>
static mm_status launch_moments(mm_ctx *c)
{
    KParams<real> kp = make_kparams<real>(c, 1.0);
    const int plane = c->g.nxi * c->g.neta;
    constexpr int VWF = 16 / sizeof(real);
    const real *dens = (const real *)c->buf[c->cur];
    // planes that tile a warp: one warp per configuration with vector loads; otherwise one block per configuration
    const int vw = plane % (32 * VWF) == 0 ? VWF : (VWF > 2 && plane % (32 * 2) == 0 ? 2 : 0);
    if (vw && plane <= 32 * vw * 4) {
        int64_t blocks = (c->nc + 7) / 8;
        const int64_t cap = (int64_t)c->sm_count * 8;
        if (blocks > cap) blocks = cap;
        if (vw == VWF)
            moments_warp_kernel<real, VWF><<<(unsigned)blocks, 256, 0, c->stream>>>(kp, dens, c->mom_force, c->mom_torque);
        else
            moments_warp_kernel<real, 2><<<(unsigned)blocks, 256, 0, c->stream>>>(kp, dens, c->mom_force, c->mom_torque);
    } else {
        int64_t blocks = c->nc;
        const int64_t cap = (int64_t)c->sm_count * 16;
        if (blocks > cap) blocks = cap;
        moments_generic_kernel<real><<<(unsigned)blocks, 256, 0, c->stream>>>(kp, dens, c->mom_force, c->mom_torque);
    }
    CUDA_TRY(c, cudaGetLastError());
    c->launches++;
    return MM_OK;
}

// ---- C ABI -----------------------------------------------------------------------------------
static bool finite_nonneg(double x) { return std::isfinite(x) && x >= 0.0; }

extern "C" mm_status mm_create(const mm_grid *grid, const mm_params *params, mm_dtype dtype, void *b0, void *b1,
                               void *cuda_stream, mm_ctx **out)
{
    if (out) *out = nullptr;
    if (!grid || !params || !out) return fail(nullptr, MM_ERR_INVALID_ARG, "NULL argument");
    const mm_grid &g = *grid;
    const mm_params &p = *params;
    if (g.nx < 1 || g.ny < 1 || g.ntheta < 1 || g.ns < 1 || g.nxi < 1 || g.neta < 1)
        return fail(nullptr, MM_ERR_INVALID_ARG, "grid dimensions must be >= 1");
    if (dtype != MM_F32 && dtype != MM_F64) return fail(nullptr, MM_ERR_INVALID_ARG, "bad dtype");
    if (!(std::isfinite(p.R) && p.R > 0) || !(std::isfinite(p.f_stall) && p.f_stall > 0) ||
        !(std::isfinite(p.f_detach) && p.f_detach > 0) || !finite_nonneg(p.v0) || !finite_nonneg(p.k_spring) ||
        !finite_nonneg(p.k_on) || !finite_nonneg(p.k_off0) || !finite_nonneg(p.end_detach_mult) ||
        !finite_nonneg(p.m_free) || !std::isfinite(p.s_lo) || !std::isfinite(p.s_hi) || !(p.s_hi > p.s_lo))
        return fail(nullptr, MM_ERR_INVALID_ARG, "parameter out of range or not finite");
    if (p.n_end_cells < 0 || 2 * (int64_t)p.n_end_cells > g.ns)
        return fail(nullptr, MM_ERR_INVALID_ARG, "need 0 <= 2*n_end_cells <= ns");
    if (p.flags & ~(MM_FLAG_S_PERIODIC | MM_FLAG_OFFSET_PERIODIC_NOMASK | MM_FLAG_CHECK_DT | MM_FLAG_RK2_SUPERBEE))
        return fail(nullptr, MM_ERR_INVALID_ARG, "unknown flag");
    if (b0 == nullptr && b1 != nullptr) return fail(nullptr, MM_ERR_INVALID_ARG, "pass dens_buf0, both density buffers, or neither");
    if (b0 && (b0 == b1 || ((uintptr_t)b0 & 15) || ((uintptr_t)b1 & 15)))
        return fail(nullptr, MM_ERR_INVALID_ARG, "density buffers must be distinct and 16-byte aligned");
    const int64_t nc = (int64_t)g.nx * g.ny * g.ntheta;
    const int64_t inner = (int64_t)g.ns * g.nxi * g.neta;
    if (nc > (int64_t)1 << 40 || inner > (int64_t)1 << 30) return fail(nullptr, MM_ERR_INVALID_ARG, "grid too large");

    int dev = 0;
    CUDA_TRY(nullptr, cudaGetDevice(&dev));
    mm_ctx *c = new (std::nothrow) mm_ctx();
    if (!c) return fail(nullptr, MM_ERR_NOMEM, "host allocation failed");
    c->g = g; c->p = p; c->dtype = dtype; c->esize = dtype == MM_F64 ? 8 : 4;
    c->nc = nc; c->inner = inner; c->cells = nc * inner;
    c->stream = (cudaStream_t)cuda_stream;
    c->device = dev;
    c->buf[0] = b0; c->buf[1] = b1; c->owns = (b0 == nullptr); c->cur = 0;
    c->U = c->V = c->Om = c->kappa = c->cos_t = c->sin_t = nullptr;
    c->inside = nullptr; c->mom_force = c->mom_torque = nullptr; c->flag_dev = nullptr;
    c->loc_lambda = nullptr; c->loc_n = c->loc_nmax = c->loc_list = c->loc_count = nullptr; c->loc_dt = nullptr;
    c->loc_valid = false;
    c->psi = c->fline = c->F2 = c->spread_G = c->spread_part = nullptr; c->psi_set = false; c->opt_spread_atomic = 0;
    c->Mf_f32 = nullptr; c->node_tab_x = c->node_tab_y = nullptr;
    c->Mf = c->Mbc = c->free_raw = c->free_factor = nullptr; c->free_fx = nullptr; c->free_any = nullptr; c->coupled = false;
    c->mom_valid = c->vel_set = false; c->tile_ok = false; c->fline_valid = false;
    c->dens_cov_count = 0;
    // measured defaults: the upwind-sparse tensor-memory kernel, at most MM_MAX_FUSE_T
    // substeps per pass (with MM_AUTO_KERNEL = 4: the coefficient-form kernel at depth 10 / 5)
    c->opt_kernel = 0; c->opt_fuse_t = MM_AUTO_KERNEL == 5 ? MM_MAX_FUSE_T : (dtype == MM_F64 ? 5 : 10); c->opt_fuse_mom = 1;
    c->opt_free_refresh = 0;
    c->single = (b0 != nullptr && b1 == nullptr);
    c->opt_inplace = c->single ? 1 : 0;
    c->checked_dt = NAN; c->launches = 0; c->kname[0] = 0;
    try { c->dens_cov.assign((size_t)nc, 0); } catch (...) { delete c; return fail(nullptr, MM_ERR_NOMEM, "host allocation failed"); }

    auto bail = [&](mm_status s, const std::string &m) { std::string mm_ = m; mm_destroy(c); return fail(nullptr, s, mm_); };
#define CR(expr)                                                                                              \
    do {                                                                                                      \
        cudaError_t e_ = (expr);                                                                              \
        if (e_ != cudaSuccess)                                                                                \
            return bail(e_ == cudaErrorMemoryAllocation ? MM_ERR_NOMEM : MM_ERR_CUDA,                         \
                        std::string(#expr) + ": " + cudaGetErrorString(e_));                                  \
    } while (0)
    CR(cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, dev));
    if (c->owns) {
        CR(cudaMalloc(&c->buf[0], (size_t)c->cells * c->esize));
        CR(cudaMalloc(&c->buf[1], (size_t)c->cells * c->esize));
    }
    const size_t plane = (size_t)g.nxi * g.neta;
    CR(cudaMalloc(&c->U, (size_t)nc * c->esize));
    CR(cudaMalloc(&c->V, (size_t)nc * c->esize));
    CR(cudaMalloc(&c->Om, (size_t)nc * c->esize));
    CR(cudaMalloc(&c->kappa, plane * c->esize));
    CR(cudaMalloc(&c->cos_t, (size_t)g.ntheta * c->esize));
    CR(cudaMalloc(&c->sin_t, (size_t)g.ntheta * c->esize));
    CR(cudaMalloc(&c->inside, plane));
    CR(cudaMalloc(&c->mom_force, (size_t)nc * 2 * sizeof(double)));
    CR(cudaMalloc(&c->mom_torque, (size_t)nc * sizeof(double)));
    CR(cudaMalloc(&c->flag_dev, sizeof(unsigned int)));
    const int nomask = (p.flags & MM_FLAG_OFFSET_PERIODIC_NOMASK) ? 1 : 0;
    if (dtype == MM_F64)
        setup_tables_kernel<double><<<8, 128, 0, c->stream>>>(g.nxi, g.neta, g.ntheta, p.R, p.k_spring, p.k_off0,
                                                              p.f_detach, nomask, (double *)c->kappa, c->inside,
                                                              (double *)c->cos_t, (double *)c->sin_t);
    else
        setup_tables_kernel<float><<<8, 128, 0, c->stream>>>(g.nxi, g.neta, g.ntheta, p.R, p.k_spring, p.k_off0,
                                                             p.f_detach, nomask, (float *)c->kappa, c->inside,
                                                             (float *)c->cos_t, (float *)c->sin_t);
    CR(cudaGetLastError());
    c->launches++;
#undef CR
    {
        mm_status ts = build_tensor_maps(c);
        if (ts != MM_OK) { std::string m = c->err; mm_destroy(c); return fail(nullptr, ts, m); }
    }
    *out = c;
    return MM_OK;
}

extern "C" mm_status mm_destroy(mm_ctx *c)
{
    if (!c) return MM_OK;
    cudaStreamSynchronize(c->stream);
    if (c->owns) { cudaFree(c->buf[0]); cudaFree(c->buf[1]); }
    cudaFree(c->U); cudaFree(c->V); cudaFree(c->Om);
    cudaFree(c->kappa); cudaFree(c->cos_t); cudaFree(c->sin_t); cudaFree(c->inside);
    cudaFree(c->mom_force); cudaFree(c->mom_torque); cudaFree(c->flag_dev);
    cudaFree(c->loc_lambda); cudaFree(c->loc_n); cudaFree(c->loc_nmax); cudaFree(c->loc_dt);
    cudaFree(c->loc_list); cudaFree(c->loc_count);
    cudaFree(c->psi); cudaFree(c->fline); cudaFree(c->F2); cudaFree(c->spread_G); cudaFree(c->spread_part);
    cudaFree(c->node_tab_x); cudaFree(c->Mf_f32); cudaFree(c->Mf); cudaFree(c->Mbc); cudaFree(c->free_raw); cudaFree(c->free_factor); cudaFree(c->free_fx); cudaFree(c->free_any);
    delete c;
    return MM_OK;
}

static mm_status copy_in(mm_ctx *c, void *dst, const void *src, size_t bytes, int src_on_device)
{
    CUDA_TRY(c, cudaMemcpyAsync(dst, src, bytes, src_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice,
                                c->stream));
    if (!src_on_device) CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    return MM_OK;
}
static mm_status copy_out(mm_ctx *c, void *dst, const void *src, size_t bytes, int dst_on_device)
{
    CUDA_TRY(c, cudaMemcpyAsync(dst, src, bytes, dst_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost,
                                c->stream));
    if (!dst_on_device) CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    return MM_OK;
}

extern "C" mm_status mm_set_density_range(mm_ctx *c, int64_t c_begin, int64_t n, const void *src, int on_device)
{
    if (!c) return MM_ERR_INVALID_ARG;
    if (!src || c_begin < 0 || n < 0 || c_begin + n > c->nc) return fail(c, MM_ERR_INVALID_ARG, "bad range or NULL source");
    if (n == 0) return MM_OK;
    char *dst = (char *)c->buf[c->cur] + (size_t)c_begin * c->inner * c->esize;
    mm_status s = copy_in(c, dst, src, (size_t)n * c->inner * c->esize, on_device);
    if (s != MM_OK) return s;
    for (int64_t i = c_begin; i < c_begin + n; ++i)
        if (!c->dens_cov[(size_t)i]) { c->dens_cov[(size_t)i] = 1; c->dens_cov_count++; }
    c->mom_valid = false; c->fline_valid = false;
    return MM_OK;
}
extern "C" mm_status mm_set_density(mm_ctx *c, const void *src, int on_device)
{
    if (!c) return MM_ERR_INVALID_ARG;
    return mm_set_density_range(c, 0, c->nc, src, on_device);
}
extern "C" mm_status mm_get_density_range(mm_ctx *c, int64_t c_begin, int64_t n, void *dst, int on_device)
{
    if (!c) return MM_ERR_INVALID_ARG;
    if (!dst || c_begin < 0 || n < 0 || c_begin + n > c->nc) return fail(c, MM_ERR_INVALID_ARG, "bad range or NULL destination");
    if (c->dens_cov_count != c->nc) return fail(c, MM_ERR_STATE, "density not set");
    if (n == 0) return MM_OK;
    const char *src = (const char *)c->buf[c->cur] + (size_t)c_begin * c->inner * c->esize;
    return copy_out(c, dst, src, (size_t)n * c->inner * c->esize, on_device);
}
extern "C" mm_status mm_get_density(mm_ctx *c, void *dst, int on_device)
{
    if (!c) return MM_ERR_INVALID_ARG;
    return mm_get_density_range(c, 0, c->nc, dst, on_device);
}

extern "C" mm_status mm_set_filament_velocity(mm_ctx *c, const void *U, const void *V, const void *Om, int on_device)
{
    if (!c) return MM_ERR_INVALID_ARG;
    if (!U || !V || !Om) return fail(c, MM_ERR_INVALID_ARG, "NULL velocity array");
    const size_t bytes = (size_t)c->nc * c->esize;
    const cudaMemcpyKind kind = on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
    CUDA_TRY(c, cudaMemcpyAsync(c->U, U, bytes, kind, c->stream));
    CUDA_TRY(c, cudaMemcpyAsync(c->V, V, bytes, kind, c->stream));
    CUDA_TRY(c, cudaMemcpyAsync(c->Om, Om, bytes, kind, c->stream));
    if (!on_device) CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    c->vel_set = true;
    c->checked_dt = NAN;
    c->loc_valid = false;
    return MM_OK;
}

static mm_status refresh_free_motors(mm_ctx *c);   // NEXT-2, below

extern "C" mm_status mm_substep(mm_ctx *c, int32_t n_sub, double dt)
{
    if (!c) return MM_ERR_INVALID_ARG;
    if (n_sub < 0) return fail(c, MM_ERR_INVALID_ARG, "n_sub < 0");
    if (n_sub == 0) return MM_OK;
    if (!(std::isfinite(dt) && dt > 0)) return fail(c, MM_ERR_INVALID_ARG, "dt must be finite and > 0");
    if (c->dens_cov_count != c->nc || !c->vel_set) return fail(c, MM_ERR_STATE, "set density and filament velocity first");
    if ((c->p.flags & MM_FLAG_CHECK_DT) && !(c->checked_dt == dt)) {
        CUDA_TRY(c, cudaMemsetAsync(c->flag_dev, 0, sizeof(unsigned int), c->stream));
        const int blocks = c->sm_count * 16;
        if (c->dtype == MM_F64) check_dt_kernel<double><<<blocks, 256, 0, c->stream>>>(make_kparams<double>(c, dt), c->flag_dev);
        else check_dt_kernel<float><<<blocks, 256, 0, c->stream>>>(make_kparams<float>(c, dt), c->flag_dev);
        CUDA_TRY(c, cudaGetLastError());
        c->launches++;
        unsigned int flag = 0;
        CUDA_TRY(c, cudaMemcpyAsync(&flag, c->flag_dev, sizeof flag, cudaMemcpyDeviceToHost, c->stream));
        CUDA_TRY(c, cudaStreamSynchronize(c->stream));
        if (flag) return fail(c, MM_ERR_UNSTABLE, "dt violates the positivity bound S8");
        c->checked_dt = dt;
    }
    // kernel choice: 0 auto (the upwind-sparse tensor-memory kernel when the grid/flags are supported; else generic),
    // 1 generic, 2 warp-streamed (1-D TMA), 3 tile, 4 coefficient form, 5 upwind-sparse / tensor memory (same
    // grids/flags as 2)
    int kind = c->opt_kernel;
    if (kind == 0) kind = (stream_supported(c) && !(c->coupled && (c->g.nx > 32767 || c->g.ny > 32767))) ? MM_AUTO_KERNEL : 1;
    const bool fast = kind == 4 || kind == 5;   // the two coefficient-form families: coupled source, in-place passes
    if (c->coupled && fast && (c->g.nx > 32767 || c->g.ny > 32767))
        return fail(c, MM_ERR_INVALID_ARG, "the coupled coefficient-form kernels need nx, ny <= 32767");
    if (c->coupled && kind != 1 && !fast)
        return fail(c, MM_ERR_INVALID_ARG, "the free-motor coupled source runs on the coefficient-form or generic kernels (MM_OPT_KERNEL 0, 1, 4 or 5)");
    if (c->single && !(fast && stream_supported(c)))
        return fail(c, MM_ERR_INVALID_ARG, "a single-buffer context runs only the in-place coefficient-form / fused RK2 kernels (16x16 or 8x8 offset planes, no test flags)");
    if (kind == 2 && !stream_supported(c)) return fail(c, MM_ERR_INVALID_ARG, "streamed kernel does not support this grid/flags");
    if (fast && !stream_supported(c)) return fail(c, MM_ERR_INVALID_ARG, "coefficient-form kernels do not support this grid/flags");
    if (kind == 3 && !c->tile_ok) return fail(c, MM_ERR_INVALID_ARG, "tile kernel does not support this grid/flags");
    c->mom_valid = false; c->fline_valid = false;
    const int refresh = c->coupled ? c->opt_free_refresh : 0;
    if (refresh > 0 && !c->psi_set) return fail(c, MM_ERR_STATE, "MM_OPT_FREE_REFRESH needs mm_set_psi");
    if (c->p.flags & MM_FLAG_RK2_SUPERBEE) {
        // kernel 0 (auto): the fused one-pass kernel where the grid is supported, else the generic stages; 1: generic
        if (c->opt_kernel != 0 && c->opt_kernel != 1)
            return fail(c, MM_ERR_INVALID_ARG, "RK2 + Superbee runs on kernel 0 (auto) or 1 (generic)");
        const bool fused = c->opt_kernel == 0 && stream_supported(c) && !c->coupled;
        // the generic stages write m* into the spare buffer: a single-buffer context has none
        if (c->single && !fused)
            return fail(c, MM_ERR_INVALID_ARG, "a single-buffer context runs RK2 + Superbee only on the fused in-place kernel (no coupled source, 16x16 or 8x8 offset planes)");
        for (int n = 0; n < n_sub; ++n) {
            if (refresh > 0 && n % refresh == 0) { mm_status fs = refresh_free_motors(c); if (fs != MM_OK) return fs; }
            const bool mom = fused && c->opt_fuse_mom && n == n_sub - 1;   // moments fused into the last pass
            mm_status s = fused ? launch_rk2_fused_any(c, dt, mom)
                                : launch_rk2_generic(c, dt);
            if (s != MM_OK) return s;
            if (mom) c->mom_valid = true;
        }
        return MM_OK;
    }
    // Alg. 2's cadence (MM_OPT_FREE_REFRESH = k > 0): the coarse reduction, cap and M_f are redone before every k-th
    // substep, so a chunk of at most k substeps is fused between two updates
    for (int n0 = 0; n0 < n_sub; n0 += (refresh > 0 ? refresh : n_sub)) {
    int remaining = refresh > 0 ? (n_sub - n0 < refresh ? n_sub - n0 : refresh) : n_sub;
    if (refresh > 0) { mm_status fs = refresh_free_motors(c); if (fs != MM_OK) return fs; c->mom_valid = false; c->fline_valid = false; }
    const bool last_chunk = refresh <= 0 || n0 + remaining == n_sub;   // moments are fused into the call's last pass only
    while (remaining > 0) {
        mm_status s;
        int t = 1;
        if (kind == 1) {
            s = c->dtype == MM_F64 ? launch_generic<double>(c, dt, c->buf[c->cur], c->buf[c->cur ^ 1])
                                   : launch_generic<float>(c, dt, c->buf[c->cur], c->buf[c->cur ^ 1]);
        } else {
            // balanced passes: as few as the fuse depth allows, of equal depth (10 substeps at depth 6 = 5 + 5)
            int tmax = c->opt_fuse_t;
            if (!fast && tmax > 4) tmax = 4;   // the streamed / tiled variants are instantiated up to 4
            if (kind == 4 && tmax > 10) tmax = 10;
            if (kind == 4 && tmax > 6 && !(c->dtype == MM_F32 && c->g.nxi == 16)) tmax = 6;   // depth 7-10: fp32 16x16 only
            if (kind == 5 && tmax > tm_max_levels(c)) tmax = tm_max_levels(c);               // tensor-memory budget
            const int passes_left = (remaining + tmax - 1) / tmax;
            t = (remaining + passes_left - 1) / passes_left;
            const bool mom = c->opt_fuse_mom && remaining == t && last_chunk;
            const bool inpl = c->opt_inplace != 0;
            // auto: shallow passes run faster on the coefficient-form kernel, whose per-plane set-up is leaner (measured
            // crossover, profiles/r02a_README.md: depth 8 in fp32, 6 in fp64); forced kernels are taken as asked
            int pk = kind;
            if (c->opt_kernel == 0 && kind == 5) {
                const int coef_max = (c->dtype == MM_F32 && c->g.nxi == 16) ? 10 : 6;
                if (t < (c->dtype == MM_F64 ? 6 : 8) && t <= coef_max) pk = 4;
            }
            s = kind == 2   ? launch_stream(c, t, mom, dt, c->buf[c->cur], c->buf[c->cur ^ 1])
                : pk == 4 ? launch_coef(c, t, mom, dt, c->buf[c->cur], c->buf[inpl ? c->cur : c->cur ^ 1])
                : pk == 5 ? launch_tm(c, t, mom, dt, c->buf[c->cur], c->buf[inpl ? c->cur : c->cur ^ 1], false, 0, false)
                            : launch_tile(c, t, mom, dt, c->cur, c->buf[c->cur ^ 1]);
            if (s == MM_OK && mom) { c->mom_valid = true; c->fline_valid = (pk == 5 && c->fline != nullptr); }
        }
        if (s != MM_OK) return s;
        if (!(fast && c->opt_inplace)) c->cur ^= 1;
        remaining -= t;
    }
    }
    return MM_OK;
}

// ---- NEXT-3: local adaptive time step per configuration (mm_local.cuh) ------------------------------------
template <typename real>
static mm_status advance_local_impl(mm_ctx *c, double dt, double cfl)
{
    const mm_grid &g = c->g;
    const mm_params &p = c->p;
    LocalParams lp;
    lp.v0 = p.v0; lp.f_stall = p.f_stall; lp.R = p.R;
    lp.dxi = 2.0 * p.R / g.nxi; lp.deta = 2.0 * p.R / g.neta; lp.ds = (p.s_hi - p.s_lo) / g.ns; lp.s_lo = p.s_lo;
    lp.k_spring = p.k_spring; lp.k_off0 = p.k_off0; lp.f_detach = p.f_detach; lp.end_mult = p.end_detach_mult;
    lp.dt = dt; lp.cfl = cfl;
    lp.ns = g.ns; lp.nxi = g.nxi; lp.neta = g.neta; lp.ntheta = g.ntheta; lp.n_end = p.n_end_cells;
    {
        const int32_t init[2] = {0, INT32_MIN};   // running max of n_c and of -n_c
        CUDA_TRY(c, cudaMemcpyAsync(c->loc_nmax, init, sizeof init, cudaMemcpyHostToDevice, c->stream));
    }
    int64_t blocks = (c->nc + 7) / 8;
    const int64_t cap = (int64_t)c->sm_count * 16;
    if (blocks > cap) blocks = cap;
    local_rate_kernel<real><<<(unsigned)blocks, 256, 0, c->stream>>>(lp, c->nc, (const real *)c->U, (const real *)c->V,
                                                                     (const real *)c->Om, c->inside, c->loc_lambda,
                                                                     c->loc_n, (real *)c->loc_dt, c->loc_nmax);
    CUDA_TRY(c, cudaGetLastError());
    c->launches++;
    int32_t nmm[2] = {0, 0};   // the number of passes is a host decision: one small read at the macro cadence
    CUDA_TRY(c, cudaMemcpyAsync(nmm, c->loc_nmax, sizeof nmm, cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    const int32_t nmax = nmm[0], nmin = -nmm[1];
    c->loc_valid = true;
    c->mom_valid = false; c->fline_valid = false;
    if (c->p.flags & MM_FLAG_RK2_SUPERBEE) {
        // Alg. 2 as one loop with the paper's scheme (l.5 driving l.9-10), any grid, coupled source or not: the generic
        // stage kernels, one local step of every unfinished unit per pair of launches
        for (int32_t step = 0; step < nmax; ++step) {
            mm_status s = launch_rk2_local_generic(c, step);
            if (s != MM_OK) return s;
        }
        return MM_OK;
    }
    // kernel choice: 0 auto = the coefficient-form local-step kernel where the grid is supported, else (or 1) generic
    if (c->opt_kernel != 0 && c->opt_kernel != 1 && c->opt_kernel != 4 && c->opt_kernel != 5)
        return fail(c, MM_ERR_INVALID_ARG, "mm_advance_local runs on kernel 0 (auto), 1 (generic), 4 (coefficient form) or 5 (upwind-sparse)");
    if ((c->opt_kernel == 4 || c->opt_kernel == 5) && !stream_supported(c))
        return fail(c, MM_ERR_INVALID_ARG, "coefficient-form kernels do not support this grid/flags");
    if (c->opt_kernel != 1 && stream_supported(c)) {
        // kernel 5 (and auto): the tensor-memory kernel takes the level count of a configuration at run time, so a pass
        // fuses up to MM_OPT_FUSE_T local steps; kernel 4: the coefficient-form instances, MM_LOCAL_FUSE_T per pass
        const bool tm = c->opt_kernel == 5 || (c->opt_kernel == 0 && MM_AUTO_KERNEL == 5);
        int FT = MM_LOCAL_FUSE_T;
        if (tm) { FT = c->opt_fuse_t; if (FT > tm_max_levels(c)) FT = tm_max_levels(c); }
        auto launch_pass = [&](bool mom, const void *in, void *out, int32_t done, bool use_list) {
            return tm ? launch_tm(c, FT, mom, 1.0, in, out, true, done, use_list) : launch_coef_local(c, mom, in, out, done, use_list);
        };
        // fp32: passes run IN PLACE on the current buffer and, from the second pass on, visit only the unfinished
        // configurations (compact list built on the device); a configuration writes its moments when it finishes.
        // fp64 (measured: in-place is slower there): ping-pong passes over all configurations,
        // finished ones copied through, moments in the last pass.
        const int32_t passes = (nmax + FT - 1) / FT;
        const bool inplace = sizeof(real) == 4 || c->opt_inplace;
        for (int32_t ps = 0; ps < passes; ++ps) {
            const int32_t done = ps * FT;
            mm_status s;
            if (inplace) {
                // moments are only compiled into the passes in which some configuration can finish
                const bool mom = c->opt_fuse_mom != 0 && nmin <= done + FT;
                if (ps > 0) {
                    CUDA_TRY(c, cudaMemsetAsync(c->loc_count, 0, sizeof(int32_t), c->stream));
                    int64_t lb = (c->nc + 255) / 256;
                    if (lb > (int64_t)c->sm_count * 8) lb = (int64_t)c->sm_count * 8;
                    local_list_kernel<<<(unsigned)lb, 256, 0, c->stream>>>(c->nc, c->loc_n, done, c->loc_list, c->loc_count);
                    CUDA_TRY(c, cudaGetLastError());
                    c->launches++;
                }
                s = launch_pass(mom, c->buf[c->cur], c->buf[c->cur], done, ps > 0);
            } else {
                s = launch_pass(c->opt_fuse_mom != 0 && ps == passes - 1, c->buf[c->cur], c->buf[c->cur ^ 1], done, false);
                if (s == MM_OK) c->cur ^= 1;
            }
            if (s != MM_OK) return s;
        }
        if (c->opt_fuse_mom) { c->mom_valid = true; c->fline_valid = tm && c->fline != nullptr; }
        return MM_OK;
    }
    if (c->single) return fail(c, MM_ERR_INVALID_ARG, "a single-buffer context runs only the in-place kernels");
    KParams<real> kp = make_kparams<real>(c, 1.0);   // per unit dt; the kernels scale by dt_c
    int64_t gblocks = (c->cells + 255) / 256;
    const int64_t gcap = (int64_t)c->sm_count * 64;
    if (gblocks > gcap) gblocks = gcap;
    for (int32_t step = 0; step < nmax; ++step) {
        substep_generic_local_kernel<real><<<(unsigned)gblocks, 256, 0, c->stream>>>(
            kp, (const real *)c->buf[c->cur], (real *)c->buf[c->cur ^ 1], c->loc_n, (const real *)c->loc_dt, step);
        CUDA_TRY(c, cudaGetLastError());
        c->launches++;
        c->cur ^= 1;
    }
    snprintf(c->kname, sizeof c->kname, "local_generic<%s>", sizeof(real) == 8 ? "f64" : "f32");
    return MM_OK;
}

extern "C" mm_status mm_advance_local(mm_ctx *c, double dt, double cfl)
{
    if (!c) return MM_ERR_INVALID_ARG;
    if (!(std::isfinite(dt) && dt > 0) || !(std::isfinite(cfl) && cfl > 0))
        return fail(c, MM_ERR_INVALID_ARG, "dt and cfl must be finite and > 0");
    const bool rk2 = (c->p.flags & MM_FLAG_RK2_SUPERBEE) != 0;
    if (rk2 && c->single) return fail(c, MM_ERR_INVALID_ARG, "local RK2 + Superbee steps run on the generic stages: two density buffers");
    if (!rk2 && c->coupled && !((c->opt_kernel == 0 || c->opt_kernel == 5) && MM_AUTO_KERNEL == 5 && stream_supported(c)))
        return fail(c, MM_ERR_INVALID_ARG, "with the free-motor coupled source mm_advance_local runs on kernel 0 / 5 only (16x16 or 8x8 offset planes)");
    if (!rk2 && c->coupled && (c->g.nx > 32767 || c->g.ny > 32767))
        return fail(c, MM_ERR_INVALID_ARG, "the coupled coefficient-form kernels need nx, ny <= 32767");
    if (c->dens_cov_count != c->nc || !c->vel_set) return fail(c, MM_ERR_STATE, "set density and filament velocity first");
    if (c->nc > INT32_MAX) return fail(c, MM_ERR_INVALID_ARG, "mm_advance_local keeps 32-bit configuration lists: nx*ny*ntheta must be < 2^31");
    if (!c->loc_count) {   // the group counts as allocated when its LAST member is (a failed call leaves no half group behind)
        void *g[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
        const size_t bytes[6] = {(size_t)c->nc * sizeof(double), (size_t)c->nc * sizeof(int32_t), (size_t)c->nc * c->esize,
                                 2 * sizeof(int32_t), (size_t)c->nc * sizeof(int32_t), sizeof(int32_t)};
        for (int i = 0; i < 6; ++i)
            if (cudaMalloc(&g[i], bytes[i]) != cudaSuccess) {
                cudaGetLastError();
                for (int k = 0; k < i; ++k) cudaFree(g[k]);
                return fail(c, MM_ERR_NOMEM, "device allocation failed (local-step buffers)");
            }
        c->loc_lambda = (double *)g[0]; c->loc_n = (int32_t *)g[1]; c->loc_dt = g[2];
        c->loc_nmax = (int32_t *)g[3]; c->loc_list = (int32_t *)g[4]; c->loc_count = (int32_t *)g[5];
    }
    return c->dtype == MM_F64 ? advance_local_impl<double>(c, dt, cfl) : advance_local_impl<float>(c, dt, cfl);
}

extern "C" mm_status mm_local_steps(mm_ctx *c, int32_t *n_steps, double *lambda, int on_device)
{
    if (!c) return MM_ERR_INVALID_ARG;
    if (!c->loc_valid) return fail(c, MM_ERR_STATE, "no mm_advance_local call yet");
    const cudaMemcpyKind kind = on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
    if (n_steps) CUDA_TRY(c, cudaMemcpyAsync(n_steps, c->loc_n, (size_t)c->nc * sizeof(int32_t), kind, c->stream));
    if (lambda) CUDA_TRY(c, cudaMemcpyAsync(lambda, c->loc_lambda, (size_t)c->nc * sizeof(double), kind, c->stream));
    if (!on_device) CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    return MM_OK;
}

// ---- NEXT-4: motor-force spreading onto the fluid grid (mm_spread.cuh) -----------------------------------------
extern "C" mm_status mm_set_psi(mm_ctx *c, const double *psi, int on_device)
{
    if (!c) return MM_ERR_INVALID_ARG;
    if (!psi) return fail(c, MM_ERR_INVALID_ARG, "NULL psi");
    if (!c->psi) CUDA_TRY(c, cudaMalloc(&c->psi, (size_t)c->nc * sizeof(double)));
    CUDA_TRY(c, cudaMemcpyAsync(c->psi, psi, (size_t)c->nc * sizeof(double),
                                on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, c->stream));
    if (!on_device) CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    c->psi_set = true;
    return MM_OK;
}

template <typename real>
static mm_status spread_impl(mm_ctx *c)
{
    KParams<real> kp = make_kparams<real>(c, 1.0);
    const int plane = c->g.nxi * c->g.neta;
    constexpr int VWF = 16 / sizeof(real);
    const real *dens = (const real *)c->buf[c->cur];
    int64_t blocks = (c->nc + 7) / 8;
    const int64_t cap = (int64_t)c->sm_count * 8;
    if (blocks > cap) blocks = cap;
    if (!c->fline_valid) {   // else: the last pass of mm_substep / mm_advance_local already wrote the plane forces
        if (plane % VWF == 0)
            plane_force_kernel<real, VWF><<<(unsigned)blocks, 256, 0, c->stream>>>(kp, dens, c->fline);
        else
            plane_force_kernel<real, 1><<<(unsigned)blocks, 256, 0, c->stream>>>(kp, dens, c->fline);
        CUDA_TRY(c, cudaGetLastError());
        c->launches++;
        c->fline_valid = true;
    }
    const double ds = (c->p.s_hi - c->p.s_lo) / c->g.ns;
    const int nn = c->g.nx * c->g.ny, nt = c->g.ntheta * c->g.ns;
    if (c->opt_spread_atomic) {   // the first version: one thread per point force and stencil column, fp64 atomic adds
        CUDA_TRY(c, cudaMemsetAsync(c->F2, 0, (size_t)nn * 2 * sizeof(double), c->stream));
        const int64_t total = c->nc * c->g.ns * 4;
        int64_t sb = (total + 255) / 256;
        const int64_t scap = (int64_t)c->sm_count * 32;
        if (sb > scap) sb = scap;
        spread_kernel<<<(unsigned)sb, 256, 0, c->stream>>>(c->nc, c->g.ns, c->g.nx, c->g.ny, c->g.ntheta, c->p.s_lo, ds, c->psi,
                                                           c->fline, c->F2);
        CUDA_TRY(c, cudaGetLastError());
        c->launches += 1;
        return MM_OK;
    }
    // gather: scale + transpose the plane forces, one thread per target node and chunk of (theta, j) pairs, chunks summed
    const int nchunks = (nt + SPREAD_CH - 1) / SPREAD_CH;
    const double w0 = 2.0 * 3.14159265358979323846264338327950288 / (double)c->g.ntheta * ds;
    spread_transpose_kernel<<<dim3((unsigned)((nn + 31) / 32), (unsigned)((nt + 31) / 32)), dim3(32, 8), 0, c->stream>>>(
        nn, c->g.ntheta, c->g.ns, w0, c->psi, (const double2 *)c->fline, (double2 *)c->spread_G);
    CUDA_TRY(c, cudaGetLastError());
    spread_gather_kernel<<<dim3((unsigned)((nn + 255) / 256), (unsigned)nchunks), 256, 0, c->stream>>>(
        c->g.nx, c->g.ny, c->g.ntheta, c->g.ns, c->p.s_lo, ds, (const double2 *)c->spread_G, (double2 *)c->spread_part);
    CUDA_TRY(c, cudaGetLastError());
    spread_sum_kernel<<<(unsigned)((nn + 255) / 256), 256, 0, c->stream>>>(nn, nchunks, (const double2 *)c->spread_part, (double2 *)c->F2);
    CUDA_TRY(c, cudaGetLastError());
    c->launches += 3;
    return MM_OK;
}

extern "C" mm_status mm_spread_force(mm_ctx *c, double *F2, int on_device)
{
    if (!c) return MM_ERR_INVALID_ARG;
    if (!F2) return fail(c, MM_ERR_INVALID_ARG, "NULL destination");
    if (c->dens_cov_count != c->nc || !c->psi_set) return fail(c, MM_ERR_STATE, "set density and psi first");
    if ((int64_t)c->g.ntheta * c->g.ns > 65535LL * 32)
        return fail(c, MM_ERR_INVALID_ARG, "mm_spread_force: ntheta * ns must be <= 2097120");
    if (!c->F2) {   // allocated as a group, committed together
        void *a = nullptr, *b = nullptr, *g = nullptr, *pt = nullptr;
        const size_t nchunks = ((size_t)c->g.ntheta * c->g.ns + SPREAD_CH - 1) / SPREAD_CH;
        if (cudaMalloc(&a, (size_t)c->nc * c->g.ns * 2 * sizeof(double)) != cudaSuccess ||
            cudaMalloc(&b, (size_t)c->g.nx * c->g.ny * 2 * sizeof(double)) != cudaSuccess ||
            cudaMalloc(&g, (size_t)c->nc * c->g.ns * 2 * sizeof(double)) != cudaSuccess ||
            cudaMalloc(&pt, nchunks * c->g.nx * c->g.ny * 2 * sizeof(double)) != cudaSuccess) {
            cudaGetLastError();
            cudaFree(a); cudaFree(b); cudaFree(g);
            return fail(c, MM_ERR_NOMEM, "device allocation failed (spreading buffers)");
        }
        c->fline = (double *)a; c->F2 = (double *)b; c->spread_G = (double *)g; c->spread_part = (double *)pt;
    }
    mm_status s = c->dtype == MM_F64 ? spread_impl<double>(c) : spread_impl<float>(c);
    if (s != MM_OK) return s;
    CUDA_TRY(c, cudaMemcpyAsync(F2, c->F2, (size_t)c->g.nx * c->g.ny * 2 * sizeof(double),
                                on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, c->stream));
    if (!on_device) CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    return MM_OK;
}

// ---- NEXT-2: free-motor coupling (mm_free.cuh) -------------------------------------------------------------------
template <typename real>
static mm_status free_impl(mm_ctx *c)
{
    const mm_grid &g = c->g;
    const mm_params &p = c->p;
    FreeGeom q;
    q.R = p.R; q.dxi = 2.0 * p.R / g.nxi; q.deta = 2.0 * p.R / g.neta; q.ds = (p.s_hi - p.s_lo) / g.ns; q.s_lo = p.s_lo;
    q.ns = g.ns; q.nxi = g.nxi; q.neta = g.neta; q.ntheta = g.ntheta; q.nx = g.nx; q.ny = g.ny;
    q.tabx = c->node_tab_x; q.taby = c->node_tab_y;
    const int nn = g.nx * g.ny;
    const double w = 2.0 * 3.14159265358979323846264338327950288 / (double)g.ntheta * q.ds * q.dxi * q.deta;
    CUDA_TRY(c, cudaMemsetAsync(c->free_raw, 0, (size_t)nn * sizeof(double), c->stream));
    CUDA_TRY(c, cudaMemsetAsync(c->free_any, 0, sizeof(int), c->stream));
    int64_t blocks = (c->nc + 7) / 8;
    const int64_t cap = (int64_t)c->sm_count * 8;
    if (blocks > cap) blocks = cap;
    real *dens = (real *)c->buf[c->cur];
    // the BASELINE offset planes run the vector kernels
    const int vw = (g.nxi == 16 && g.neta == 16) || (g.nxi == 8 && g.neta == 8) ? 1 : 0;
    // a private copy of the table per CTA in shared memory where it fits: 96-bit fixed point (12 bytes per node) in the
    // vector kernels, fp64 in the generic one
    const size_t tab_bytes = vw ? (size_t)g.nx * (g.ny | 1) * 12 : (size_t)nn * sizeof(double);
    const bool priv = tab_bytes <= 200 * 1024;
    const bool fx = priv && vw;
    double unit = 1.0;   // power of two >= M_total
    if (p.m_free > 0) { int e = 0; std::frexp(p.m_free, &e); unit = std::ldexp(1.0, e); }
    if (fx) CUDA_TRY(c, cudaMemsetAsync(c->free_fx, 0, (size_t)nn * 16, c->stream));
    auto run = [&](auto kern0, auto kern1, int threads, size_t smem) -> mm_status {
        int bps = 0;
        mm_status ks = kernel_shape(c, (const void *)kern0, threads, smem, "free-motor deposit kernel", &bps);
        if (ks != MM_OK) return ks;
        const int wpb = threads / 32;
        int64_t pb = (int64_t)c->sm_count * bps;
        if (pb > (c->nc + wpb - 1) / wpb) pb = (c->nc + wpb - 1) / wpb;
        kern0<<<(unsigned)pb, threads, smem, c->stream>>>(q, c->nc, dens, c->psi, w, c->free_raw, nullptr, nullptr, c->free_fx, 1.0 / unit);
        CUDA_TRY(c, cudaGetLastError());
        free_cap_kernel<<<(nn + 255) / 256, 256, 0, c->stream>>>(nn, p.m_free, c->free_raw, c->free_factor, c->Mbc, c->Mf, c->free_any,
                                                                  fx ? c->free_fx : nullptr, unit, c->Mf_f32);
        CUDA_TRY(c, cudaGetLastError());
        kern1<<<(unsigned)blocks, 256, 0, c->stream>>>(q, c->nc, dens, nullptr, 0.0, nullptr, c->free_factor, c->free_any, nullptr, 1.0);
        CUDA_TRY(c, cudaGetLastError());
        return MM_OK;
    };
    mm_status rs;
#define MM_FREE_VEC(N_) (priv ? run(free_cells_vec_kernel<real, 0, true, N_, N_, MM_FREE_PRIV_PL>, free_cells_vec_kernel<real, 1, false, N_, N_, 4>, sizeof(real) == 4 ? MM_FREE_PRIV_THREADS_F32 : 512, tab_bytes) \
                             : run(free_cells_vec_kernel<real, 0, false, N_, N_, 4>, free_cells_vec_kernel<real, 1, false, N_, N_, 4>, 256, 0))
    if (vw && g.nxi == 16) rs = MM_FREE_VEC(16);
    else if (vw) rs = MM_FREE_VEC(8);
    else rs = priv ? run(free_cells_kernel<real, 0, true>, free_cells_kernel<real, 1, false>, 1024, tab_bytes)
                   : run(free_cells_kernel<real, 0, false>, free_cells_kernel<real, 1, false>, 256, 0);
#undef MM_FREE_VEC
    if (rs != MM_OK) return rs;
    c->launches += 3;
    return MM_OK;
}

static mm_status refresh_free_motors(mm_ctx *c)
{
    return c->dtype == MM_F64 ? free_impl<double>(c) : free_impl<float>(c);
}

extern "C" mm_status mm_update_free_motors(mm_ctx *c, double *Mb_coarse, double *M_free, int on_device)
{
    if (!c) return MM_ERR_INVALID_ARG;
    if (c->dens_cov_count != c->nc || !c->psi_set) return fail(c, MM_ERR_STATE, "set density and psi first");
    const size_t nn = (size_t)c->g.nx * c->g.ny;
    if (!c->free_any) {   // allocated as a group, committed together
        void *g[8] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
        // the anchor-node tables of the vector / tensor-memory kernels (16-bit entries; the BASELINE offset planes)
        const mm_grid &gr = c->g;
        const bool tabs = ((gr.nxi == 16 && gr.neta == 16) || (gr.nxi == 8 && gr.neta == 8)) && gr.nx <= 65535 && gr.ny <= 65535;
        const size_t tabx_bytes = (((size_t)gr.nx * gr.ntheta * gr.ns * gr.nxi * 2 + 255) / 256) * 256;
        const size_t taby_bytes = (size_t)gr.ny * gr.ntheta * gr.ns * gr.neta * 2;
        const size_t bytes[8] = {nn * sizeof(double), nn * sizeof(double), nn * sizeof(double), nn * sizeof(double), nn * 16,
                                 nn * sizeof(float), sizeof(int), tabs ? tabx_bytes + taby_bytes : 256};
        for (int i = 0; i < 8; ++i)
            if (cudaMalloc(&g[i], bytes[i]) != cudaSuccess) {
                cudaGetLastError();
                for (int k = 0; k < i; ++k) cudaFree(g[k]);
                return fail(c, MM_ERR_NOMEM, "device allocation failed (free-motor tables)");
            }
        c->Mf = (double *)g[0]; c->Mbc = (double *)g[1]; c->free_raw = (double *)g[2]; c->free_factor = (double *)g[3];
        c->free_fx = (unsigned long long *)g[4]; c->Mf_f32 = (float *)g[5]; c->free_any = (int *)g[6];
        if (tabs) {
            unsigned short *tx = (unsigned short *)g[7], *ty = (unsigned short *)((char *)g[7] + tabx_bytes);
            FreeGeom q;
            const mm_params &p = c->p;
            q.R = p.R; q.dxi = 2.0 * p.R / gr.nxi; q.deta = 2.0 * p.R / gr.neta; q.ds = (p.s_hi - p.s_lo) / gr.ns; q.s_lo = p.s_lo;
            q.ns = gr.ns; q.nxi = gr.nxi; q.neta = gr.neta; q.ntheta = gr.ntheta; q.nx = gr.nx; q.ny = gr.ny;
            q.tabx = q.taby = nullptr;
            node_table_kernel<<<c->sm_count * 8, 256, 0, c->stream>>>(q, tx, ty);
            if (cudaGetLastError() != cudaSuccess) {
                for (int k = 0; k < 8; ++k) cudaFree(g[k]);
                c->Mf = c->Mbc = c->free_raw = c->free_factor = nullptr; c->free_fx = nullptr; c->Mf_f32 = nullptr; c->free_any = nullptr;
                return fail(c, MM_ERR_CUDA, "anchor-node table kernel failed to launch");
            }
            c->launches++;
            c->node_tab_x = tx; c->node_tab_y = ty;
        } else {
            cudaFree(g[7]);
        }
    }
    mm_status s = c->dtype == MM_F64 ? free_impl<double>(c) : free_impl<float>(c);
    if (s != MM_OK) return s;
    c->coupled = true;
    c->mom_valid = false; c->fline_valid = false;     // the cap may have rescaled the density
    const cudaMemcpyKind kind = on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
    if (Mb_coarse) CUDA_TRY(c, cudaMemcpyAsync(Mb_coarse, c->Mbc, nn * sizeof(double), kind, c->stream));
    if (M_free) CUDA_TRY(c, cudaMemcpyAsync(M_free, c->Mf, nn * sizeof(double), kind, c->stream));
    if (!on_device) CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    return MM_OK;
}

extern "C" mm_status mm_moments(mm_ctx *c, double *force, double *torque, int on_device)
{
    if (!c) return MM_ERR_INVALID_ARG;
    if (c->dens_cov_count != c->nc) return fail(c, MM_ERR_STATE, "density not set");
    if (!c->mom_valid) {
        mm_status s = c->dtype == MM_F64 ? launch_moments<double>(c) : launch_moments<float>(c);
        if (s != MM_OK) return s;
        c->mom_valid = true;
    }
    const cudaMemcpyKind kind = on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
    if (force) CUDA_TRY(c, cudaMemcpyAsync(force, c->mom_force, (size_t)c->nc * 2 * sizeof(double), kind, c->stream));
    if (torque) CUDA_TRY(c, cudaMemcpyAsync(torque, c->mom_torque, (size_t)c->nc * sizeof(double), kind, c->stream));
    if (!on_device) CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    return MM_OK;
}

extern "C" mm_status mm_set_option(mm_ctx *c, mm_option opt, int64_t v)
{
    if (!c) return MM_ERR_INVALID_ARG;
    switch (opt) {
    case MM_OPT_KERNEL:
        if (v < 0 || v > 5) return fail(c, MM_ERR_INVALID_ARG, "MM_OPT_KERNEL in 0..5");
        c->opt_kernel = (int)v; return MM_OK;
    case MM_OPT_FUSE_T:
        if (v < 1 || v > MM_MAX_FUSE_T) return fail(c, MM_ERR_INVALID_ARG, "MM_OPT_FUSE_T in 1..MM_MAX_FUSE_T");
        c->opt_fuse_t = (int)v; return MM_OK;
    case MM_OPT_FUSE_MOMENTS:
        c->opt_fuse_mom = v ? 1 : 0; return MM_OK;
    case MM_OPT_FREE_COUPLING:
        if (v && !c->Mf) return fail(c, MM_ERR_STATE, "no free-motor table yet: call mm_update_free_motors first");
        c->coupled = v != 0; return MM_OK;
    case MM_OPT_FREE_REFRESH:
        if (v < 0 || v > INT32_MAX) return fail(c, MM_ERR_INVALID_ARG, "MM_OPT_FREE_REFRESH >= 0");
        c->opt_free_refresh = (int)v; return MM_OK;
    case MM_OPT_INPLACE:
        if (c->single && !v) return fail(c, MM_ERR_INVALID_ARG, "a single-buffer context is always in place");
        c->opt_inplace = v ? 1 : 0; return MM_OK;
    case MM_OPT_SPREAD_ATOMIC: c->opt_spread_atomic = v ? 1 : 0; return MM_OK;
    }
    return fail(c, MM_ERR_INVALID_ARG, "unknown option");
}

extern "C" mm_status mm_get_option(const mm_ctx *c, mm_option opt, int64_t *v)
{
    if (!c || !v) return MM_ERR_INVALID_ARG;
    switch (opt) {
    case MM_OPT_KERNEL: *v = c->opt_kernel; return MM_OK;
    case MM_OPT_FUSE_T: *v = c->opt_fuse_t; return MM_OK;
    case MM_OPT_FUSE_MOMENTS: *v = c->opt_fuse_mom; return MM_OK;
    case MM_OPT_INPLACE: *v = c->opt_inplace; return MM_OK;
    case MM_OPT_FREE_COUPLING: *v = c->coupled ? 1 : 0; return MM_OK;
    case MM_OPT_FREE_REFRESH: *v = c->opt_free_refresh; return MM_OK;
    case MM_OPT_SPREAD_ATOMIC: *v = c->opt_spread_atomic; return MM_OK;
    }
    return MM_ERR_INVALID_ARG;
}

// ---- the second roof: FMA issue peak of this device, measured (SURVEY.md 8(d) "measure and record the box's fp64 and
// fp32 FMA peaks with a small register-only microbenchmark") ------------------------------------------------------------
template <typename real>
static mm_status fma_peak_impl(cudaStream_t stream, double *tflops)
{
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return fail(nullptr, MM_ERR_CUDA, "no CUDA device");
    real *out = nullptr;
    if (cudaMalloc(&out, (size_t)sms * 1024 * sizeof(real)) != cudaSuccess) { cudaGetLastError(); return fail(nullptr, MM_ERR_NOMEM, "device allocation failed"); }
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int iters = sizeof(real) == 8 ? 2048 : 4096;
    double best = 0.0;
    for (int rep = 0; rep < 4; ++rep) {   // the first repetition is the warm-up
        cudaEventRecord(e0, stream);
        fma_peak_kernel<real><<<sms, 1024, 0, stream>>>(out, (real)0.999, (real)1e-3, iters);
        cudaEventRecord(e1, stream);
        if (cudaEventSynchronize(e1) != cudaSuccess) break;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double flops = 2.0 * (double)FMA_PEAK_PER_ITER * iters * 1024.0 * sms;
        if (rep > 0 && ms > 0.f && flops / (ms * 1e-3) / 1e12 > best) best = flops / (ms * 1e-3) / 1e12;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(out);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess || best <= 0.0) return fail(nullptr, MM_ERR_CUDA, std::string("FMA peak probe failed: ") + cudaGetErrorString(e));
    *tflops = best;
    return MM_OK;
}

template <typename real>
static mm_status fma_fresh_impl(cudaStream_t stream, double *tflops)
{
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return fail(nullptr, MM_ERR_CUDA, "no CUDA device");
    real *out = nullptr, *in = nullptr;
    if (cudaMalloc(&out, (size_t)sms * 512 * sizeof(real)) != cudaSuccess || cudaMalloc(&in, 24 * sizeof(real)) != cudaSuccess) {
        cudaGetLastError();
        cudaFree(out);
        return fail(nullptr, MM_ERR_NOMEM, "device allocation failed");
    }
    real h[24];
    for (int i = 0; i < 24; ++i) h[i] = i < 8 ? (real)(0.5 + 0.01 * i) : (i < 16 ? (real)(0.25 + 0.01 * i) : (real)(1e-3 * i));
    cudaMemcpyAsync(in, h, sizeof h, cudaMemcpyHostToDevice, stream);
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int iters = sizeof(real) == 8 ? 2048 : 4096;
    double best = 0.0;
    for (int rep = 0; rep < 4; ++rep) {   // the first repetition is the warm-up
        cudaEventRecord(e0, stream);
        fma_fresh_kernel<real><<<sms, 512, 0, stream>>>(out, in, iters);
        cudaEventRecord(e1, stream);
        if (cudaEventSynchronize(e1) != cudaSuccess) break;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double flops = 2.0 * 64.0 * iters * 512.0 * sms;
        if (rep > 0 && ms > 0.f && flops / (ms * 1e-3) / 1e12 > best) best = flops / (ms * 1e-3) / 1e12;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(out); cudaFree(in);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess || best <= 0.0) return fail(nullptr, MM_ERR_CUDA, std::string("FMA operand probe failed: ") + cudaGetErrorString(e));
    *tflops = best;
    return MM_OK;
}

extern "C" mm_status mm_measure_fma_rate(mm_dtype dtype, int32_t fresh_operands, void *cuda_stream, double *tflops)
{
    if (!tflops) return fail(nullptr, MM_ERR_INVALID_ARG, "NULL argument");
    if (dtype != MM_F32 && dtype != MM_F64) return fail(nullptr, MM_ERR_INVALID_ARG, "bad dtype");
    if (fresh_operands == 1) return mm_measure_fma_peak(dtype, cuda_stream, tflops);
    if (fresh_operands != 3) return fail(nullptr, MM_ERR_INVALID_ARG, "fresh_operands must be 1 (mm_measure_fma_peak) or 3");
    return dtype == MM_F64 ? fma_fresh_impl<double>((cudaStream_t)cuda_stream, tflops) : fma_fresh_impl<float>((cudaStream_t)cuda_stream, tflops);
}

extern "C" mm_status mm_measure_fma_peak(mm_dtype dtype, void *cuda_stream, double *tflops)
{
    if (!tflops) return fail(nullptr, MM_ERR_INVALID_ARG, "NULL argument");
    if (dtype != MM_F32 && dtype != MM_F64) return fail(nullptr, MM_ERR_INVALID_ARG, "bad dtype");
    return dtype == MM_F64 ? fma_peak_impl<double>((cudaStream_t)cuda_stream, tflops) : fma_peak_impl<float>((cudaStream_t)cuda_stream, tflops);
}

extern "C" int64_t mm_launch_count(const mm_ctx *c) { return c ? c->launches : 0; }
extern "C" const char *mm_kernel_name(const mm_ctx *c) { return c ? c->kname : ""; }

extern "C" const char *mm_status_string(mm_status s)
{
    switch (s) {
    case MM_OK: return "MM_OK";
    case MM_ERR_INVALID_ARG: return "MM_ERR_INVALID_ARG";
    case MM_ERR_CUDA: return "MM_ERR_CUDA";
    case MM_ERR_NOMEM: return "MM_ERR_NOMEM";
    case MM_ERR_STATE: return "MM_ERR_STATE";
    case MM_ERR_UNSTABLE: return "MM_ERR_UNSTABLE";
    }
    return "MM_ERR_?";
}
extern "C" const char *mm_last_error(const mm_ctx *c) { return c ? c->err.c_str() : g_create_err.c_str(); }
