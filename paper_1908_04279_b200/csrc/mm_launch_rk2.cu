// mm_launch_rk2.cu -- dispatch of the RK2 + Superbee kernels (mm_rk2.cuh).
#include "mm_ctx.cuh"
#include "mm_rk2.cuh"

// One RK2 + Superbee substep with the generic stage kernel: m* into the spare buffer, m^{n+1} in place.
template <typename real>
static mm_status launch_rk2_generic_t(mm_ctx *c, double dt)
{
    int64_t blocks = (c->cells + 255) / 256;
    const int64_t cap = (int64_t)c->sm_count * 64;
    if (blocks > cap) blocks = cap;
    real *A = (real *)c->buf[c->cur], *B = (real *)c->buf[c->cur ^ 1];
    rk2_stage_generic_kernel<real><<<(unsigned)blocks, 256, 0, c->stream>>>(make_kparams<real>(c, 0.5 * dt), A, A, B);
    CUDA_TRY(c, cudaGetLastError());
    rk2_stage_generic_kernel<real><<<(unsigned)blocks, 256, 0, c->stream>>>(make_kparams<real>(c, dt), A, B, A);
    CUDA_TRY(c, cudaGetLastError());
    c->launches += 2;
    snprintf(c->kname, sizeof c->kname, "rk2_generic<%s>", sizeof(real) == 8 ? "f64" : "f32");
    return MM_OK;
}

// One LOCAL RK2 + Superbee step of every unit that still owes one (step < n_c), each with its own dt_c (generic stages)
template <typename real>
static mm_status launch_rk2_local_generic_t(mm_ctx *c, int32_t step)
{
    int64_t blocks = (c->cells + 255) / 256;
    const int64_t cap = (int64_t)c->sm_count * 64;
    if (blocks > cap) blocks = cap;
    real *A = (real *)c->buf[c->cur], *B = (real *)c->buf[c->cur ^ 1];
    const KParams<real> kp = make_kparams<real>(c, 1.0);   // per unit dt
    rk2_stage_generic_kernel<real><<<(unsigned)blocks, 256, 0, c->stream>>>(kp, A, A, B, c->loc_n, (const real *)c->loc_dt, step, real(0.5));
    CUDA_TRY(c, cudaGetLastError());
    rk2_stage_generic_kernel<real><<<(unsigned)blocks, 256, 0, c->stream>>>(kp, A, B, A, c->loc_n, (const real *)c->loc_dt, step, real(1));
    CUDA_TRY(c, cudaGetLastError());
    c->launches += 2;
    snprintf(c->kname, sizeof c->kname, "rk2_local_generic<%s>", sizeof(real) == 8 ? "f64" : "f32");
    return MM_OK;
}

mm_status launch_rk2_local_generic(mm_ctx *c, int32_t step)
{
    return c->dtype == MM_F64 ? launch_rk2_local_generic_t<double>(c, step) : launch_rk2_local_generic_t<float>(c, step);
}

// One RK2 + Superbee substep in one HBM pass (rk2_fused_kernel): reads buf[cur], writes buf[cur^1].
#ifndef MM_RK2_MINB_F32
#define MM_RK2_MINB_F32 2
#endif
#ifndef MM_RK2_KEEPC
#define MM_RK2_KEEPC 0   // 1: the round-1 variant (stage 2's coefficient set in registers / rebuilt) instead of tensor memory
#endif
template <typename real, int NXI, int NETA, int CB>
static mm_status launch_rk2_fused(mm_ctx *c, double dt, bool mom)
{
    constexpr int P = 2, D = 3, WARPS = 4, MINB = sizeof(real) == 8 ? 2 : MM_RK2_MINB_F32;
    constexpr bool PM = sizeof(real) == 8, CS = sizeof(real) == 8;
    using Cfg = CoefCfg<real, NXI, NETA, CB, P, D, WARPS, CS>;
    constexpr bool KEEPC = MM_RK2_KEEPC != 0 && sizeof(real) == 4;
    constexpr bool TM = !(MM_RK2_KEEPC != 0);
    auto kern = rk2_fused_kernel<real, NXI, NETA, CB, P, D, WARPS, MINB, PM, CS, TM ? false : KEEPC>;
    const size_t smem = Cfg::SMEM_BYTES + 16;   // + the tensor-memory base address
    int blocks_per_sm = 0;
    {
        mm_status ks = kernel_shape(c, (const void *)kern, WARPS * 32, smem, "fused RK2 kernel", &blocks_per_sm);
        if (ks != MM_OK) return ks;
    }
    if (TM) {
        // kernels with tcgen05.alloc: the occupancy calculator answers 1 CTA per SM (mm_launch_tm.cu); own count
        using TmR = Rk2Tm<real, Cfg::QA, CB>;
        cudaFuncAttributes fa;
        CUDA_TRY(c, cudaFuncGetAttributes(&fa, (const void *)kern));
        const int regs_per_warp = ((fa.numRegs + 7) / 8) * 8 * 32;
        int n = 65536 / (regs_per_warp * WARPS);
        const int by_smem = (int)((size_t)(227 * 1024) / (smem + 1024)), by_tmem = 512 / TmR::COLS;
        if (by_smem < n) n = by_smem;
        if (by_tmem < n) n = by_tmem;
        if (n > 4) n = 4;
        if (n > blocks_per_sm) blocks_per_sm = n;
    }
    int64_t grid = (int64_t)c->sm_count * blocks_per_sm;
    const int64_t need = (c->nc + WARPS - 1) / WARPS;
    if (grid > need) grid = need;
    // in place when asked: stage 2 stores plane i-2 when plane i has arrived, every input plane is read once
    const int dst = c->opt_inplace ? c->cur : c->cur ^ 1;
    kern<<<(unsigned)grid, WARPS * 32, smem, c->stream>>>(make_kparams<real>(c, dt), (const real *)c->buf[c->cur],
                                                           (real *)c->buf[dst], c->mom_force, c->mom_torque, mom ? 1 : 0);
    CUDA_TRY(c, cudaGetLastError());
    c->launches++;
    c->cur = dst;
    snprintf(c->kname, sizeof c->kname, "rk2_fused<%s,%dx%d,CB=%d%s>", sizeof(real) == 8 ? "f64" : "f32", NXI, NETA, CB, mom ? ",mom" : "");
    return MM_OK;
}

mm_status launch_rk2_fused_any(mm_ctx *c, double dt, bool mom)
{
    const bool big = c->g.nxi == 16;
    if (c->dtype == MM_F64)
        return big ? launch_rk2_fused<double, 16, 16, 2>(c, dt, mom) : launch_rk2_fused<double, 8, 8, 2>(c, dt, mom);
    return big ? launch_rk2_fused<float, 16, 16, 4>(c, dt, mom) : launch_rk2_fused<float, 8, 8, 2>(c, dt, mom);
}

mm_status launch_rk2_generic(mm_ctx *c, double dt)
{
    return c->dtype == MM_F64 ? launch_rk2_generic_t<double>(c, dt) : launch_rk2_generic_t<float>(c, dt);
}
