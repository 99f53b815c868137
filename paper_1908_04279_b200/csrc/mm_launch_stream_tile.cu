// mm_launch_stream_tile.cu -- dispatch of the warp-streamed (mm_stream.cuh) and tiled-TMA (mm_tile.cuh) substep kernels.
#include "mm_ctx.cuh"
#include "mm_stream.cuh"
#include "mm_tile.cuh"

// ---- streamed-kernel dispatch -----------------------------------------------------------------
template <typename real, int NXI, int NETA, int CB, int T, bool MOM>
static mm_status launch_stream_inst(mm_ctx *c, double dt, const void *in, void *out)
{
    constexpr int P = 2, D = 3, WARPS = 4;
    using Cfg = StreamCfg<real, NXI, NETA, CB, P, D, WARPS>;
    auto kern = substep_stream_kernel<real, NXI, NETA, CB, T, MOM, P, D, WARPS>;
    int blocks_per_sm = 0;
    {
        mm_status ks = kernel_shape(c, (const void *)kern, WARPS * 32, Cfg::SMEM_BYTES, "streamed kernel", &blocks_per_sm);
        if (ks != MM_OK) return ks;
    }
    int64_t grid = (int64_t)c->sm_count * blocks_per_sm;
    const int64_t need = (c->nc + WARPS - 1) / WARPS;
    if (grid > need) grid = need;
    KParams<real> kp = make_kparams<real>(c, dt);
    kern<<<(unsigned)grid, WARPS * 32, Cfg::SMEM_BYTES, c->stream>>>(kp, (const real *)in, (real *)out, c->mom_force,
                                                                      c->mom_torque);
    CUDA_TRY(c, cudaGetLastError());
    c->launches++;
    snprintf(c->kname, sizeof c->kname, "stream<%s,%dx%d,CB=%d,T=%d%s>", sizeof(real) == 8 ? "f64" : "f32", NXI, NETA,
             CB, T, MOM ? ",mom" : "");
    return MM_OK;
}

template <typename real, int NXI, int NETA, int CB>
static mm_status launch_stream_shape(mm_ctx *c, int T, bool mom, double dt, const void *in, void *out)
{
#define MM_CASE(TT)                                                                                     \
    case TT:                                                                                            \
        return mom ? launch_stream_inst<real, NXI, NETA, CB, TT, true>(c, dt, in, out)                  \
                   : launch_stream_inst<real, NXI, NETA, CB, TT, false>(c, dt, in, out);
    switch (T) {
        MM_CASE(1)
        MM_CASE(2)
        MM_CASE(3)
        MM_CASE(4)
    }
#undef MM_CASE
    return fail(c, MM_ERR_INVALID_ARG, "unsupported fuse depth");
}

bool stream_supported(const mm_ctx *c)
{
    if (c->p.flags & (MM_FLAG_S_PERIODIC | MM_FLAG_OFFSET_PERIODIC_NOMASK)) return false;
    return (c->g.nxi == 16 && c->g.neta == 16) || (c->g.nxi == 8 && c->g.neta == 8);
}

mm_status launch_stream(mm_ctx *c, int T, bool mom, double dt, const void *in, void *out)
{
    const bool big = c->g.nxi == 16;
    if (c->dtype == MM_F64)
        return big ? launch_stream_shape<double, 16, 16, 2>(c, T, mom, dt, in, out)
                   : launch_stream_shape<double, 8, 8, 2>(c, T, mom, dt, in, out);
    return big ? launch_stream_shape<float, 16, 16, 4>(c, T, mom, dt, in, out)
               : launch_stream_shape<float, 8, 8, 2>(c, T, mom, dt, in, out);
}

// ---- tile-kernel dispatch ---------------------------------------------------------------------
typedef CUresult (*encode_tiled_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                    const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static constexpr int TILE_P = 2;   // planes per TMA box

static bool tile_shape_supported(const mm_ctx *c)
{
    if (c->p.flags & (MM_FLAG_S_PERIODIC | MM_FLAG_OFFSET_PERIODIC_NOMASK)) return false;
    return (c->g.nxi == 16 && c->g.neta == 16) || (c->g.nxi == 8 && c->g.neta == 8);
}

// 4-D view (eta, xi, s, c) of a density buffer; box = one padded plane pair of CPW configurations,
// out-of-bounds elements read as zero (the ghost cells of S5).
mm_status build_tensor_maps(mm_ctx *c)
{
    c->tile_ok = false;
    if (!tile_shape_supported(c) || c->single) return MM_OK;
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn ||
        qres != cudaDriverEntryPointSuccess) {
        cudaGetLastError();
        return fail(c, MM_ERR_CUDA, "cuTensorMapEncodeTiled not available from the driver");
    }
    const int cpw = 256 / (c->g.nxi * c->g.neta);
    const cuuint64_t dims[4] = {(cuuint64_t)c->g.neta, (cuuint64_t)c->g.nxi, (cuuint64_t)c->g.ns, (cuuint64_t)c->nc};
    const cuuint64_t strides[3] = {(cuuint64_t)c->g.neta * c->esize, (cuuint64_t)c->g.nxi * c->g.neta * c->esize,
                                   (cuuint64_t)c->inner * c->esize};
    const cuuint32_t box[4] = {(cuuint32_t)c->g.neta + (cuuint32_t)(32 / c->esize), (cuuint32_t)c->g.nxi + 2, (cuuint32_t)TILE_P, (cuuint32_t)cpw};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    for (int b = 0; b < 2; ++b) {
        CUresult r = ((encode_tiled_fn)fn)(&c->tmap[b], c->dtype == MM_F64 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64
                                                                          : CU_TENSOR_MAP_DATA_TYPE_FLOAT32,
                                           4, c->buf[b], dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                           CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return fail(c, MM_ERR_CUDA, "cuTensorMapEncodeTiled failed (" + std::to_string((int)r) + ")");
    }
    c->tile_ok = true;
    return MM_OK;
}

template <typename real, int NXI, int NETA, int CB, int T, bool MOM>
static mm_status launch_tile_inst(mm_ctx *c, double dt, int in_idx, void *out)
{
    constexpr int P = TILE_P, D = (T == 1 ? 4 : 3), WARPS = 4, MINB = 2;
    using Cfg = TileCfg<real, NXI, NETA, CB, T, P, D, WARPS>;
    auto kern = substep_tile_kernel<real, NXI, NETA, CB, T, MOM, P, D, WARPS, MINB>;
    int blocks_per_sm = 0;
    {
        mm_status ks = kernel_shape(c, (const void *)kern, WARPS * 32, Cfg::SMEM_BYTES, "tile kernel", &blocks_per_sm);
        if (ks != MM_OK) return ks;
    }
    int64_t grid = (int64_t)c->sm_count * blocks_per_sm;
    const int64_t groups = (c->nc + Cfg::CPW - 1) / Cfg::CPW;
    const int64_t need = (groups + WARPS - 1) / WARPS;
    if (grid > need) grid = need;
    KParams<real> kp = make_kparams<real>(c, dt);
    kern<<<(unsigned)grid, WARPS * 32, Cfg::SMEM_BYTES, c->stream>>>(kp, c->tmap[in_idx], (real *)out, c->mom_force,
                                                                      c->mom_torque);
    CUDA_TRY(c, cudaGetLastError());
    c->launches++;
    snprintf(c->kname, sizeof c->kname, "tile<%s,%dx%d,T=%d%s>", sizeof(real) == 8 ? "f64" : "f32", NXI, NETA, T,
             MOM ? ",mom" : "");
    return MM_OK;
}

template <typename real, int NXI, int NETA, int CB>
static mm_status launch_tile_shape(mm_ctx *c, int T, bool mom, double dt, int in_idx, void *out)
{
#define MM_CASE(TT)                                                                                     \
    case TT:                                                                                            \
        return mom ? launch_tile_inst<real, NXI, NETA, CB, TT, true>(c, dt, in_idx, out)                \
                   : launch_tile_inst<real, NXI, NETA, CB, TT, false>(c, dt, in_idx, out);
    switch (T) {
        MM_CASE(1)
        MM_CASE(2)
        MM_CASE(3)
        MM_CASE(4)
    }
#undef MM_CASE
    return fail(c, MM_ERR_INVALID_ARG, "unsupported fuse depth");
}

mm_status launch_tile(mm_ctx *c, int T, bool mom, double dt, int in_idx, void *out)
{
    const bool big = c->g.nxi == 16;
    if (c->dtype == MM_F64)
        return big ? launch_tile_shape<double, 16, 16, 2>(c, T, mom, dt, in_idx, out)
                   : launch_tile_shape<double, 8, 8, 2>(c, T, mom, dt, in_idx, out);
    return big ? launch_tile_shape<float, 16, 16, 4>(c, T, mom, dt, in_idx, out)
               : launch_tile_shape<float, 8, 8, 4>(c, T, mom, dt, in_idx, out);
}

