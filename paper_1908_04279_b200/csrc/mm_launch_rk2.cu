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

// One RK2 + Superbee substep in one HBM pass (rk2_fused_kernel): reads buf[cur], writes buf[cur^1].
template <typename real, int NXI, int NETA, int CB>
static mm_status launch_rk2_fused(mm_ctx *c, double dt)
{
    constexpr int P = 2, D = 3, WARPS = 4, MINB = 2;
    constexpr bool PM = sizeof(real) == 8, CS = sizeof(real) == 8;
    using Cfg = CoefCfg<real, NXI, NETA, CB, P, D, WARPS, CS>;
    constexpr bool KEEPC = sizeof(real) == 4;
    auto kern = rk2_fused_kernel<real, NXI, NETA, CB, P, D, WARPS, MINB, PM, CS, KEEPC>;
    int blocks_per_sm = 0;
    {
        mm_status ks = kernel_shape(c, (const void *)kern, WARPS * 32, Cfg::SMEM_BYTES, "fused RK2 kernel", &blocks_per_sm);
        if (ks != MM_OK) return ks;
    }
    int64_t grid = (int64_t)c->sm_count * blocks_per_sm;
    const int64_t need = (c->nc + WARPS - 1) / WARPS;
    if (grid > need) grid = need;
    // in place when asked: stage 2 stores plane i-2 when plane i has arrived, every input plane is read once
    const int dst = c->opt_inplace ? c->cur : c->cur ^ 1;
    kern<<<(unsigned)grid, WARPS * 32, Cfg::SMEM_BYTES, c->stream>>>(make_kparams<real>(c, dt), (const real *)c->buf[c->cur],
                                                                      (real *)c->buf[dst]);
    CUDA_TRY(c, cudaGetLastError());
    c->launches++;
    c->cur = dst;
    snprintf(c->kname, sizeof c->kname, "rk2_fused<%s,%dx%d,CB=%d>", sizeof(real) == 8 ? "f64" : "f32", NXI, NETA, CB);
    return MM_OK;
}

mm_status launch_rk2_fused_any(mm_ctx *c, double dt)
{
    const bool big = c->g.nxi == 16;
    if (c->dtype == MM_F64)
        return big ? launch_rk2_fused<double, 16, 16, 2>(c, dt) : launch_rk2_fused<double, 8, 8, 2>(c, dt);
    return big ? launch_rk2_fused<float, 16, 16, 4>(c, dt) : launch_rk2_fused<float, 8, 8, 2>(c, dt);
}

mm_status launch_rk2_generic(mm_ctx *c, double dt)
{
    return c->dtype == MM_F64 ? launch_rk2_generic_t<double>(c, dt) : launch_rk2_generic_t<float>(c, dt);
}
