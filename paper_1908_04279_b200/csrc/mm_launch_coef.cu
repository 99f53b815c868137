// mm_launch_coef.cu -- dispatch of the coefficient-form substep kernels (mm_coef.cuh), global and local-step variants.
#include "mm_ctx.cuh"
#include "mm_coef.cuh"

// ---- coefficient-form kernel dispatch -----------------------------------------------------------
// Launch shape of the coefficient-form kernel, per dtype (measured sweep in profiles/r01b_README.md):
// planes per TMA copy, ring depth, warps per CTA, resident CTAs per SM asked of the register allocator.
#ifndef MM_COEF_P_F32
#define MM_COEF_P_F32 4
#endif
#ifndef MM_COEF_D_F32
#define MM_COEF_D_F32 2
#endif
#ifndef MM_COEF_P_F64
#define MM_COEF_P_F64 2
#endif
#ifndef MM_COEF_D_F64
#define MM_COEF_D_F64 3
#endif
#ifndef MM_COEF_WARPS
#define MM_COEF_WARPS 4
#endif
#ifndef MM_COEF_MINB_F32
#define MM_COEF_MINB_F32 2
#endif
#ifndef MM_COEF_MINB_F64
#define MM_COEF_MINB_F64 2
#endif

template <typename real, int NXI, int NETA, int CB, int T, bool MOM, bool MF>
static mm_status launch_coef_inst_mf(mm_ctx *c, double dt, const void *in, void *out)
{
    constexpr int P = sizeof(real) == 8 ? MM_COEF_P_F64 : MM_COEF_P_F32;
    constexpr int D = sizeof(real) == 8 ? MM_COEF_D_F64 : MM_COEF_D_F32, WARPS = MM_COEF_WARPS;
    constexpr int MINB = sizeof(real) == 8 ? MM_COEF_MINB_F64 : MM_COEF_MINB_F32;
    constexpr bool PM = sizeof(real) == 8;   // post-mask: fp64 only
    constexpr bool CS = sizeof(real) == 8;   // per-configuration constants in shared memory: fp64 only
    using Cfg = CoefCfg<real, NXI, NETA, CB, P, D, WARPS, CS, coef_rs<real>(T)>;
    auto kern = substep_coef_kernel<real, NXI, NETA, CB, T, MOM, P, D, WARPS, MINB, PM, CS, false, MF>;
    // MF: the warps' node tables (16-bit, ns * (NXI + NETA) entries each) sit behind the regular layout
    const size_t smem = MF ? ((Cfg::SMEM_BYTES + 15) / 16) * 16 + (size_t)WARPS * c->g.ns * (NXI + NETA) * 2 : Cfg::SMEM_BYTES;
    int blocks_per_sm = 0;
    {
        mm_status ks = kernel_shape(c, (const void *)kern, WARPS * 32, smem, "coefficient-form kernel", &blocks_per_sm);
        if (ks != MM_OK) return ks;
    }
    int64_t grid = (int64_t)c->sm_count * blocks_per_sm;
    const int64_t need = (c->nc + WARPS - 1) / WARPS;
    if (grid > need) grid = need;
    KParams<real> kp = make_kparams<real>(c, dt);
    kern<<<(unsigned)grid, WARPS * 32, smem, c->stream>>>(kp, (const real *)in, (real *)out, c->mom_force, c->mom_torque,
                                                           nullptr, nullptr, 0, nullptr, nullptr);
    CUDA_TRY(c, cudaGetLastError());
    c->launches++;
    snprintf(c->kname, sizeof c->kname, MF ? "coef_mf<%s,%dx%d,CB=%d,T=%d%s>" : "coef<%s,%dx%d,CB=%d,T=%d%s>", sizeof(real) == 8 ? "f64" : "f32", NXI, NETA,
             CB, T, MOM ? ",mom" : "");
    return MM_OK;
}

template <typename real, int NXI, int NETA, int CB, int T, bool MOM>
static mm_status launch_coef_inst(mm_ctx *c, double dt, const void *in, void *out)
{
    return c->coupled ? launch_coef_inst_mf<real, NXI, NETA, CB, T, MOM, true>(c, dt, in, out)
                      : launch_coef_inst_mf<real, NXI, NETA, CB, T, MOM, false>(c, dt, in, out);
}

template <typename real, int NXI, int NETA, int CB>
static mm_status launch_coef_shape(mm_ctx *c, int T, bool mom, double dt, const void *in, void *out)
{
#define MM_CASE(TT)                                                                                     \
    case TT:                                                                                            \
        return mom ? launch_coef_inst<real, NXI, NETA, CB, TT, true>(c, dt, in, out)                    \
                   : launch_coef_inst<real, NXI, NETA, CB, TT, false>(c, dt, in, out);
    switch (T) {
        MM_CASE(1)
        MM_CASE(2)
        MM_CASE(3)
        MM_CASE(4)
        MM_CASE(5)
        MM_CASE(6)
    }
    if constexpr (sizeof(real) == 4 && NXI == 16) {   // deeper fusion where it pays: fp32, the BASELINE offset plane
        switch (T) {
            MM_CASE(7)
            MM_CASE(8)
            MM_CASE(9)
            MM_CASE(10)
        }
    }
#undef MM_CASE
    return fail(c, MM_ERR_INVALID_ARG, "unsupported fuse depth");
}

// NEXT-3: one pass of the local-step variant (T = MM_LOCAL_FUSE_T levels at most per configuration)
template <typename real, int NXI, int NETA, int CB, bool MOM>
static mm_status launch_coef_local_inst(mm_ctx *c, const void *in, void *out, int32_t done, bool use_list)
{
    constexpr int T = MM_LOCAL_FUSE_T;
    // 2 planes x 3 slots for both dtypes: the kernel holds T+1 straight-line instances of the chunk body (one per
    // level count), so the chunk is kept short to stay inside the instruction cache
    constexpr int P = 2, D = 3, WARPS = MM_COEF_WARPS;
    constexpr int MINB = sizeof(real) == 8 ? MM_COEF_MINB_F64 : MM_COEF_MINB_F32;
    constexpr bool PM = sizeof(real) == 8, CS = sizeof(real) == 8;
    using Cfg = CoefCfg<real, NXI, NETA, CB, P, D, WARPS, CS, coef_rs<real>(T)>;
    auto kern = substep_coef_kernel<real, NXI, NETA, CB, T, MOM, P, D, WARPS, MINB, PM, CS, true>;
    int blocks_per_sm = 0;
    {
        mm_status ks = kernel_shape(c, (const void *)kern, WARPS * 32, Cfg::SMEM_BYTES, "local-step kernel", &blocks_per_sm);
        if (ks != MM_OK) return ks;
    }
    int64_t grid = (int64_t)c->sm_count * blocks_per_sm;
    const int64_t need = (c->nc + WARPS - 1) / WARPS;
    if (grid > need) grid = need;
    KParams<real> kp = make_kparams<real>(c, 1.0);   // per unit dt
    // in may equal out (in-place pass, see the LOC note in mm_coef.cuh)
    kern<<<(unsigned)grid, WARPS * 32, Cfg::SMEM_BYTES, c->stream>>>(kp, (const real *)in, (real *)out, c->mom_force,
                                                                      c->mom_torque, c->loc_n, (const real *)c->loc_dt, done,
                                                                      use_list ? c->loc_list : nullptr,
                                                                      use_list ? c->loc_count : nullptr);
    CUDA_TRY(c, cudaGetLastError());
    c->launches++;
    snprintf(c->kname, sizeof c->kname, "coef_local<%s,%dx%d,CB=%d,T<=%d%s>", sizeof(real) == 8 ? "f64" : "f32", NXI, NETA,
             CB, T, MOM ? ",mom" : "");
    return MM_OK;
}

mm_status launch_coef_local(mm_ctx *c, bool mom, const void *in, void *out, int32_t done, bool use_list)
{
    const bool big = c->g.nxi == 16;
#define MM_LOC(R_, N_, CB_) (mom ? launch_coef_local_inst<R_, N_, N_, CB_, true>(c, in, out, done, use_list) \
                                 : launch_coef_local_inst<R_, N_, N_, CB_, false>(c, in, out, done, use_list))
    if (c->dtype == MM_F64) return big ? MM_LOC(double, 16, 2) : MM_LOC(double, 8, 2);
    return big ? MM_LOC(float, 16, 4) : MM_LOC(float, 8, 2);
#undef MM_LOC
}

mm_status launch_coef(mm_ctx *c, int T, bool mom, double dt, const void *in, void *out)
{
    const bool big = c->g.nxi == 16;
    if (c->dtype == MM_F64)
        return big ? launch_coef_shape<double, 16, 16, 2>(c, T, mom, dt, in, out)
                   : launch_coef_shape<double, 8, 8, 2>(c, T, mom, dt, in, out);
    return big ? launch_coef_shape<float, 16, 16, 4>(c, T, mom, dt, in, out)
               : launch_coef_shape<float, 8, 8, 2>(c, T, mom, dt, in, out);
}

