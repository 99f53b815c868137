// mm_ctx.cuh -- the context behind the opaque handle of include/mm.h, error helpers, the kernel parameter block and
// the launch-shape cache, shared by the translation units of libmm.  Product code (sm_100a); shares nothing with oracle/.
#pragma once
#include "../../include/mm.h"

#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <type_traits>
#include <vector>

#include <cuda.h>
#include "mm_common.cuh"

using namespace mm;

struct mm_ctx {
    mm_grid g;
    mm_params p;
    mm_dtype dtype;
    size_t esize;
    int64_t nc, inner, cells;
    cudaStream_t stream;
    void *buf[2];
    bool owns;
    int cur;
    void *U, *V, *Om;               // [nc] real
    void *kappa, *cos_t, *sin_t;    // tables (real)
    uint8_t *inside;
    double *mom_force, *mom_torque; // [nc][2], [nc]
    unsigned int *flag_dev;         // stability-check flag
    bool mom_valid, vel_set;
    std::vector<uint8_t> dens_cov;  // per configuration: density uploaded
    int64_t dens_cov_count;
    int opt_kernel, opt_fuse_t, opt_fuse_mom, opt_inplace, opt_free_refresh;
    bool single;                    // created with ONE density buffer: only the in-place kernels can run
    double checked_dt;              // dt the S8 check last passed with (NaN = none)
    int64_t launches;
    int sm_count;
    double *loc_lambda;             // NEXT-3: per-configuration rate bound, step count, local dt, max step count
    int32_t *loc_n, *loc_nmax, *loc_list, *loc_count;
    void *loc_dt;
    bool loc_valid;
    double *psi, *fline, *F2;       // NEXT-4: filament density weights [nc], plane forces [nc][ns][2], fluid-grid force
    double *spread_G, *spread_part; // ... scaled plane forces transposed to [theta][j][node][2], per-chunk partial sums
    int opt_spread_atomic;
    bool psi_set, fline_valid;      // fline_valid: fline holds the plane forces of the CURRENT density
    unsigned short *node_tab_x, *node_tab_y;     // anchor-node tables (one allocation; NULL when nx or ny > 65535)
    float *Mf_f32;                               // fp32 contexts: M_f rounded to fp32 (written with the table)
    double *Mf, *Mbc, *free_raw, *free_factor;   // NEXT-2: free / coarse bound motor tables [nx][ny], scratch
    unsigned long long *free_fx;   // [nx][ny][2]: the coarse sums in 128-bit fixed point (mm_free.cuh)
    int *free_any;
    bool coupled;                   // the substep source is k_on M_f(r0) instead of k_on m_free
    CUtensorMap tmap[2];            // tiled-TMA views of buf[0], buf[1] (tile kernel)
    bool tile_ok;                   // tensor maps built and grid/flags supported by the tile kernel
    std::string err;
    char kname[64];
    int device;                     // the device the context was created on
    // launch shape per kernel instantiation, per CONTEXT (the shared-memory attribute is per device and the handles
    // are independent: no process-wide statics)
    struct KShape { const void *fn; size_t smem; int blocks_per_sm; };
    std::vector<KShape> kshapes;
};

extern thread_local std::string g_create_err;   // defined in mm_api.cu

inline mm_status fail(mm_ctx *ctx, mm_status s, const std::string &msg)
{
    if (ctx) ctx->err = msg; else g_create_err = msg;
    return s;
}
#define CUDA_TRY(ctx, expr)                                                                          \
    do {                                                                                             \
        cudaError_t e_ = (expr);                                                                     \
        if (e_ != cudaSuccess)                                                                       \
            return fail(ctx, e_ == cudaErrorMemoryAllocation ? MM_ERR_NOMEM : MM_ERR_CUDA,           \
                        std::string(#expr) + ": " + cudaGetErrorString(e_));                         \
    } while (0)

template <typename real>
inline KParams<real> make_kparams(const mm_ctx *c, double dt)
{
    KParams<real> k;
    const mm_grid &g = c->g;
    const mm_params &p = c->p;
    k.nc = c->nc; k.ns = g.ns; k.nxi = g.nxi; k.neta = g.neta; k.ntheta = g.ntheta;
    k.n_end = p.n_end_cells; k.flags = p.flags;
    const double ds = (p.s_hi - p.s_lo) / g.ns, dxi = 2.0 * p.R / g.nxi, deta = 2.0 * p.R / g.neta;
    k.v0 = (real)p.v0; k.kload = (real)(p.k_spring / p.f_stall);
    k.R = (real)p.R; k.dxi = (real)dxi; k.deta = (real)deta; k.ds = (real)ds; k.s_lo = (real)p.s_lo;
    k.dt = (real)dt; k.dt_ds = (real)(dt / ds); k.dt_dxi = (real)(dt / dxi); k.dt_deta = (real)(dt / deta);
    k.dt_src = (real)(dt * p.k_on * p.m_free);
    k.dt_kon = (real)(dt * p.k_on);
    k.Mf = (c->coupled && c->Mf) ? c->Mf : nullptr;
    k.Mf_r = !k.Mf ? nullptr : (sizeof(real) == 8 ? (const real *)c->Mf : (const real *)c->Mf_f32);
    k.node_x = k.Mf ? c->node_tab_x : nullptr; k.node_y = k.Mf ? c->node_tab_y : nullptr;
    k.nx = g.nx; k.ny = g.ny;
    k.geo_R = p.R; k.geo_dxi = dxi; k.geo_deta = deta; k.geo_ds = ds; k.geo_s_lo = p.s_lo;
    k.dt_endx = (real)(dt * (p.end_detach_mult - 1.0));
    k.mom_scale = -p.k_spring * ds * dxi * deta;
    k.pf_scale = k.mom_scale / ds;   // the quotient the kernels formed (same rounding as before)
    k.U = (const real *)c->U; k.V = (const real *)c->V; k.Om = (const real *)c->Om;
    k.cos_t = (const real *)c->cos_t; k.sin_t = (const real *)c->sin_t;
    k.kappa = (const real *)c->kappa; k.inside = c->inside;
    return k;
}

// Resident CTAs per SM of `fn` at this block size and dynamic shared memory; sets the kernel's shared-memory limit.
// Cached per context and per (kernel, smem).
inline mm_status kernel_shape(mm_ctx *c, const void *fn, int threads, size_t smem, const char *what, int *blocks_per_sm)
{
    for (const auto &k : c->kshapes)
        if (k.fn == fn && k.smem == smem) { *blocks_per_sm = k.blocks_per_sm; return MM_OK; }
    if (smem > 227 * 1024) return fail(c, MM_ERR_INVALID_ARG, std::string(what) + " needs more shared memory than an SM has");
    CUDA_TRY(c, cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    // these kernels stream through shared memory and keep little in L1: ask for the largest shared-memory carve-out, or
    // the occupancy below is computed (and the launch made) against the default split
    CUDA_TRY(c, cudaFuncSetAttribute(fn, cudaFuncAttributePreferredSharedMemoryCarveout, (int)cudaSharedmemCarveoutMaxShared));
    int n = 0;
    CUDA_TRY(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, fn, threads, smem));
    if (n < 1) return fail(c, MM_ERR_CUDA, std::string(what) + " does not fit on an SM");
    try { c->kshapes.push_back({fn, smem, n}); } catch (...) { return fail(c, MM_ERR_NOMEM, "host allocation failed"); }
    *blocks_per_sm = n;
    return MM_OK;
}

// ---- kernel-family launchers (one translation unit each, so that they compile in parallel)
bool stream_supported(const mm_ctx *c);
mm_status launch_stream(mm_ctx *c, int T, bool mom, double dt, const void *in, void *out);               // mm_launch_stream_tile.cu
mm_status build_tensor_maps(mm_ctx *c);
mm_status launch_tile(mm_ctx *c, int T, bool mom, double dt, int in_idx, void *out);
mm_status launch_coef(mm_ctx *c, int T, bool mom, double dt, const void *in, void *out);                 // mm_launch_coef.cu
mm_status launch_coef_local(mm_ctx *c, bool mom, const void *in, void *out, int32_t done, bool use_list);
mm_status launch_rk2_generic(mm_ctx *c, double dt);                                                     // mm_launch_rk2.cu
mm_status launch_rk2_fused_any(mm_ctx *c, double dt, bool mom);
mm_status launch_rk2_local_generic(mm_ctx *c, int32_t step);
int tm_max_levels(const mm_ctx *c);                                                                     // mm_launch_tm.cu
mm_status launch_tm(mm_ctx *c, int nlev, bool mom, double dt, const void *in, void *out, bool local, int32_t done, bool use_list);
