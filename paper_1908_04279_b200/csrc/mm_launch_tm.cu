// mm_launch_tm.cu -- dispatch of the upwind-sparse, tensor-memory-staged substep kernel (mm_tm.cuh): ONE instance per
// (dtype, offset plane, source kind); the fuse depth, the moments and the local-step mode are run-time arguments.
#include "mm_ctx.cuh"
#include "mm_tm.cuh"

// Launch shape per dtype (sweeps in profiles/r02a_README.md): planes per TMA copy, ring depth, warps per CTA, CTAs per SM.
// fp32: 2 x 8 warps = 16 warps per SM at <= 128 registers; fp64: 2 x 4 warps (the coefficient set alone is 96 registers).
#ifndef MM_TM_P_F32
#define MM_TM_P_F32 4
#endif
#ifndef MM_TM_D_F32
#define MM_TM_D_F32 2
#endif
#ifndef MM_TM_WARPS_F32
#define MM_TM_WARPS_F32 8
#endif
#ifndef MM_TM_MINB_F32
#define MM_TM_MINB_F32 2
#endif
#ifndef MM_TM_P_F64
#define MM_TM_P_F64 2
#endif
#ifndef MM_TM_D_F64
#define MM_TM_D_F64 3
#endif
#ifndef MM_TM_WARPS_F64
#define MM_TM_WARPS_F64 4
#endif
#ifndef MM_TM_MINB_F64
#define MM_TM_MINB_F64 2
#endif

template <typename real, int NXI, int NETA, int CB>
struct TmShape {
    static constexpr bool F64 = sizeof(real) == 8;
    static constexpr int P = F64 ? MM_TM_P_F64 : MM_TM_P_F32, D = F64 ? MM_TM_D_F64 : MM_TM_D_F32;
    static constexpr int WARPS = F64 ? MM_TM_WARPS_F64 : MM_TM_WARPS_F32, MINB = F64 ? MM_TM_MINB_F64 : MM_TM_MINB_F32;
    using Cfg = TmCfg<real, NXI, NETA, CB, P, D, WARPS, MINB>;
};

template <typename real, int NXI, int NETA, int CB, bool MF, bool LOC, bool PF>
static mm_status launch_tm_inst(mm_ctx *c, int nlev, bool mom, double dt, const void *in, void *out, int32_t done, bool use_list)
{
    constexpr bool local = LOC;
    using S = TmShape<real, NXI, NETA, CB>;
    using Cfg = typename S::Cfg;
    constexpr int WARPS = S::WARPS;
    auto kern = substep_tm_kernel<real, NXI, NETA, CB, S::P, S::D, WARPS, S::MINB, MF, LOC, PF>;
    if (nlev < 1 || nlev > Cfg::TMAX) return fail(c, MM_ERR_INVALID_ARG, "fuse depth beyond the tensor-memory budget of the kernel");
    // MF: the warps' node tables (16-bit, ns * (NXI + NETA) entries each) sit behind the regular layout
    const size_t smem = MF ? ((Cfg::SMEM_BYTES + 15) / 16) * 16 + (size_t)WARPS * c->g.ns * (NXI + NETA) * 2 : Cfg::SMEM_BYTES;
    int blocks_per_sm = 0;
    {
        mm_status ks = kernel_shape(c, (const void *)kern, WARPS * 32, smem, "tensor-memory-staged kernel", &blocks_per_sm);
        if (ks != MM_OK) return ks;
    }
    // The occupancy calculator answers 1 CTA per SM for every kernel that contains tcgen05.alloc, whatever its size
    // (measured: profiles/r02a_README.md), while the hardware co-schedules CTAs as long as registers, shared memory AND
    // tensor-memory columns last.  So the resident count is computed here from the three budgets; every resident CTA
    // holds Cfg::TC of the SM's 512 columns for its whole life, and one CTA too many would wait in tcgen05.alloc.
    {
        cudaFuncAttributes fa;
        CUDA_TRY(c, cudaFuncGetAttributes(&fa, (const void *)kern));
        const int regs_per_warp = ((fa.numRegs + 7) / 8) * 8 * 32;
        int by_regs = 65536 / (regs_per_warp * WARPS), by_smem = (int)((size_t)(227 * 1024) / (smem + 1024)), by_tmem = 512 / Cfg::TC;
        int n = by_regs < by_smem ? by_regs : by_smem;
        if (by_tmem < n) n = by_tmem;
        if (S::MINB < n) n = S::MINB;
        if (n > blocks_per_sm) blocks_per_sm = n;
        if (blocks_per_sm > by_tmem) blocks_per_sm = by_tmem;
    }
    int64_t grid = (int64_t)c->sm_count * blocks_per_sm;
    const int64_t need = (c->nc + WARPS - 1) / WARPS;
    if (grid > need) grid = need;
    KParams<real> kp = make_kparams<real>(c, local ? 1.0 : dt);   // local-step mode: factors per unit dt
    kern<<<(unsigned)grid, WARPS * 32, smem, c->stream>>>(kp, (const real *)in, (real *)out, c->mom_force, c->mom_torque, nlev,
                                                           mom ? 1 : 0, local ? c->loc_n : nullptr,
                                                           local ? (const real *)c->loc_dt : nullptr, done,
                                                           (local && use_list) ? c->loc_list : nullptr,
                                                           (local && use_list) ? c->loc_count : nullptr,
                                                           PF ? c->fline : nullptr);
    CUDA_TRY(c, cudaGetLastError());
    c->launches++;
    snprintf(c->kname, sizeof c->kname, "%s<%s,%dx%d,CB=%d,T%s%d%s>", MF ? (local ? "tm_mf_local" : "tm_mf") : (local ? "tm_local" : "tm"),
             sizeof(real) == 8 ? "f64" : "f32", NXI, NETA, CB, local ? "<=" : "=", nlev, mom ? ",mom" : "");
    return MM_OK;
}

template <typename real, int NXI, int NETA, int CB>
static mm_status launch_tm_shape(mm_ctx *c, int nlev, bool mom, double dt, const void *in, void *out, bool local, int32_t done,
                                 bool use_list)
{
    // PF: the pass that reduces the moments also stores the plane forces when mm_spread_force is in use
    const bool pf = mom && c->fline != nullptr;
#define MM_TM_GO(MF_, LOC_) (pf ? launch_tm_inst<real, NXI, NETA, CB, MF_, LOC_, true>(c, nlev, mom, dt, in, out, done, use_list) \
                                : launch_tm_inst<real, NXI, NETA, CB, MF_, LOC_, false>(c, nlev, mom, dt, in, out, done, use_list))
    if (local) return c->coupled ? MM_TM_GO(true, true) : MM_TM_GO(false, true);
    return c->coupled ? MM_TM_GO(true, false) : MM_TM_GO(false, false);
#undef MM_TM_GO
}

mm_status launch_tm(mm_ctx *c, int nlev, bool mom, double dt, const void *in, void *out, bool local, int32_t done, bool use_list)
{
    const bool big = c->g.nxi == 16;
    if (c->dtype == MM_F64)
        return big ? launch_tm_shape<double, 16, 16, 2>(c, nlev, mom, dt, in, out, local, done, use_list)
                   : launch_tm_shape<double, 8, 8, 2>(c, nlev, mom, dt, in, out, local, done, use_list);
    return big ? launch_tm_shape<float, 16, 16, 4>(c, nlev, mom, dt, in, out, local, done, use_list)
               : launch_tm_shape<float, 8, 8, 2>(c, nlev, mom, dt, in, out, local, done, use_list);
}

// deepest fusion one pass of the kernel supports for this context (tensor-memory columns per warp / columns per level)
int tm_max_levels(const mm_ctx *c)
{
    const bool big = c->g.nxi == 16;
    if (c->dtype == MM_F64) return big ? TmShape<double, 16, 16, 2>::Cfg::TMAX : TmShape<double, 8, 8, 2>::Cfg::TMAX;
    return big ? TmShape<float, 16, 16, 4>::Cfg::TMAX : TmShape<float, 8, 8, 2>::Cfg::TMAX;
}
