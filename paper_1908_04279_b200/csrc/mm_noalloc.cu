// mm_noalloc.cu -- mm_free_motors_noalloc (include/mm.h): the free-motor update of mm_update_free_motors (SURVEY.md
// 8(f) NEXT-2; Eq. 5-6, Alg. 2 l.14-20 PAPER.md:206-220) for callers that cannot allocate: code under
// CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  No context, no cudaMalloc / cudaFree: the
// node tables the pass needs between its three kernels (raw sums, 128-bit fixed-point sums, cap factors, the "any node
// capped" flag) live in ONE file-scope device array of fixed size, which every GPU that loads the library holds until
// exit.  Limits and sharing: nx * ny <= MM_NOALLOC_MAX_NODES; every call on a device uses the same array, so calls that
// overlap on the GPU (different streams, no ordering between them) race; the array keeps the last call's contents and
// each call clears what must start at zero.
#include "mm_ctx.cuh"
// mm_free.cuh defines three non-template functions with host-side symbols (free_cap_kernel, node_table_kernel,
// fx_deposit_rare), which mm_api.cu already emits: this unit's copies get names of their own (the first two are not
// used here -- the node pass below names the scratch array directly, and without a context there are no node tables)
#define free_cap_kernel free_cap_kernel_unused_in_noalloc_unit
#define node_table_kernel node_table_kernel_unused_in_noalloc_unit
#define fx_deposit_rare fx_deposit_rare_noalloc_unit
#include "mm_free.cuh"
#undef free_cap_kernel
#undef node_table_kernel
#undef fx_deposit_rare

#include <mutex>

namespace mm {

constexpr int NA_MAXN = MM_NOALLOC_MAX_NODES;
// layout of the scratch array, byte offsets: raw sums [MAXN] fp64 | cap factors [MAXN] fp64 | fixed-point sums
// [MAXN][2] u64 | flag (int, on a line of its own)
constexpr size_t NA_OFF_RAW = 0, NA_OFF_FACTOR = (size_t)NA_MAXN * 8, NA_OFF_FX = (size_t)NA_MAXN * 16,
                 NA_OFF_ANY = (size_t)NA_MAXN * 32, NA_BYTES = (size_t)NA_MAXN * 32 + 256;
static __device__ __align__(256) unsigned char g_na_scratch[NA_BYTES];

// Per node: cap, factor, M_b,coarse, M_f (free_cap_kernel's arithmetic), reading the sums from and writing the factors
// to the scratch array, which device code of this file names directly.
__global__ void noalloc_cap_kernel(int nn, double m_total, double *__restrict__ Mbc, double *__restrict__ Mf, int use_fx, double unit)
{
    const double *raw = reinterpret_cast<const double *>(g_na_scratch + NA_OFF_RAW);
    double *factor = reinterpret_cast<double *>(g_na_scratch + NA_OFF_FACTOR);
    const unsigned long long *raw_fx = reinterpret_cast<const unsigned long long *>(g_na_scratch + NA_OFF_FX);
    int *any_capped = reinterpret_cast<int *>(g_na_scratch + NA_OFF_ANY);
    for (int n = blockIdx.x * blockDim.x + threadIdx.x; n < nn; n += gridDim.x * blockDim.x) {
        const double r = use_fx ? ((double)(long long)raw_fx[2 * n + 1] + (double)raw_fx[2 * n] * 5.421010862427522e-20) * unit : raw[n];
        const bool over = r > m_total;
        factor[n] = over ? m_total / r : 1.0;
        const double capped = over ? m_total : r;
        Mbc[n] = capped;
        Mf[n] = m_total - capped;
        if (over) *any_capped = 1;
    }
}

// In host code `g_na_scratch` is a host-side stand-in, not a device address: the address the kernels get comes from
// cudaGetSymbolAddress, asked once per device with that device current.
constexpr int NA_MAX_DEVICES = 64;
static std::mutex g_na_mutex;
static unsigned char *g_na_ptr[NA_MAX_DEVICES];
static int g_na_sms[NA_MAX_DEVICES];

static mm_status noalloc_setup(unsigned char **scratch, int *sm_count)
{
    int dev = -1;
    CUDA_TRY(nullptr, cudaGetDevice(&dev));
    if (dev < 0 || dev >= NA_MAX_DEVICES) return fail(nullptr, MM_ERR_INVALID_ARG, "mm_free_motors_noalloc: device ordinal out of range");
    std::lock_guard<std::mutex> lock(g_na_mutex);
    if (!g_na_ptr[dev]) {
        void *p = nullptr;
        CUDA_TRY(nullptr, cudaGetSymbolAddress(&p, g_na_scratch));
        int sms = 0;
        CUDA_TRY(nullptr, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
        if (!p || sms < 1) return fail(nullptr, MM_ERR_CUDA, "mm_free_motors_noalloc: no device address for the scratch array");
        g_na_sms[dev] = sms;
        g_na_ptr[dev] = (unsigned char *)p;
    }
    *scratch = g_na_ptr[dev];
    *sm_count = g_na_sms[dev];
    return MM_OK;
}

template <typename real>
static mm_status noalloc_impl(const mm_grid &g, const mm_params &p, real *dens, const double *psi, double *Mbc, double *Mf,
                              cudaStream_t stream, unsigned char *scratch, int sm_count)
{
    FreeGeom q;
    q.R = p.R; q.dxi = 2.0 * p.R / g.nxi; q.deta = 2.0 * p.R / g.neta; q.ds = (p.s_hi - p.s_lo) / g.ns; q.s_lo = p.s_lo;
    q.ns = g.ns; q.nxi = g.nxi; q.neta = g.neta; q.ntheta = g.ntheta; q.nx = g.nx; q.ny = g.ny;
    q.tabx = q.taby = nullptr;   // no context, no tables: the nodes are evaluated inline
    const int nn = g.nx * g.ny;
    const int64_t nc = (int64_t)nn * g.ntheta;
    const double w = 2.0 * 3.14159265358979323846264338327950288 / (double)g.ntheta * q.ds * q.dxi * q.deta;
    double *raw = reinterpret_cast<double *>(scratch + NA_OFF_RAW), *factor = reinterpret_cast<double *>(scratch + NA_OFF_FACTOR);
    unsigned long long *raw_fx = reinterpret_cast<unsigned long long *>(scratch + NA_OFF_FX);
    int *any = reinterpret_cast<int *>(scratch + NA_OFF_ANY);
    // the array holds the previous call's sums and flag: what the deposits add to starts at zero (the factors are all
    // rewritten by the node pass)
    CUDA_TRY(nullptr, cudaMemsetAsync(raw, 0, (size_t)nn * sizeof(double), stream));
    CUDA_TRY(nullptr, cudaMemsetAsync(raw_fx, 0, (size_t)nn * 16, stream));
    CUDA_TRY(nullptr, cudaMemsetAsync(any, 0, sizeof(int), stream));
    int64_t blocks = (nc + 7) / 8;
    const int64_t cap = (int64_t)sm_count * 8;
    if (blocks > cap) blocks = cap;
    // kernel choice as in mm_update_free_motors (mm_api.cu, free_impl): the BASELINE offset planes run the vector
    // kernels, with a CTA-private fixed-point table in shared memory where it fits
    const int vw = (g.nxi == 16 && g.neta == 16) || (g.nxi == 8 && g.neta == 8) ? 1 : 0;
    const size_t tab_bytes = vw ? (size_t)g.nx * (g.ny | 1) * 12 : (size_t)nn * sizeof(double);
    const bool priv = tab_bytes <= 200 * 1024;
    const bool fx = priv && vw;
    double unit = 1.0;   // power of two >= M_total
    if (p.m_free > 0) { int e = 0; std::frexp(p.m_free, &e); unit = std::ldexp(1.0, e); }
    auto run = [&](auto kern0, auto kern1, int threads, size_t smem) -> mm_status {
        // attributes and occupancy are asked on every call: nothing is cached, nothing allocated
        CUDA_TRY(nullptr, cudaFuncSetAttribute((const void *)kern0, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        CUDA_TRY(nullptr, cudaFuncSetAttribute((const void *)kern0, cudaFuncAttributePreferredSharedMemoryCarveout, (int)cudaSharedmemCarveoutMaxShared));
        int bps = 0;
        CUDA_TRY(nullptr, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, (const void *)kern0, threads, smem));
        if (bps < 1) return fail(nullptr, MM_ERR_CUDA, "mm_free_motors_noalloc: the deposit kernel does not fit on an SM");
        const int wpb = threads / 32;
        int64_t pb = (int64_t)sm_count * bps;
        if (pb > (nc + wpb - 1) / wpb) pb = (nc + wpb - 1) / wpb;
        kern0<<<(unsigned)pb, threads, smem, stream>>>(q, nc, dens, psi, w, raw, nullptr, nullptr, raw_fx, 1.0 / unit);
        CUDA_TRY(nullptr, cudaGetLastError());
        noalloc_cap_kernel<<<(nn + 255) / 256, 256, 0, stream>>>(nn, p.m_free, Mbc, Mf, fx ? 1 : 0, unit);
        CUDA_TRY(nullptr, cudaGetLastError());
        kern1<<<(unsigned)blocks, 256, 0, stream>>>(q, nc, dens, nullptr, 0.0, nullptr, factor, any, nullptr, 1.0);
        CUDA_TRY(nullptr, cudaGetLastError());
        return MM_OK;
    };
#define MM_NA_VEC(N_) (priv ? run(free_cells_vec_kernel<real, 0, true, N_, N_, MM_FREE_PRIV_PL>, free_cells_vec_kernel<real, 1, false, N_, N_, 4>, sizeof(real) == 4 ? MM_FREE_PRIV_THREADS_F32 : 512, tab_bytes) \
                           : run(free_cells_vec_kernel<real, 0, false, N_, N_, 4>, free_cells_vec_kernel<real, 1, false, N_, N_, 4>, 256, 0))
    if (vw && g.nxi == 16) return MM_NA_VEC(16);
    if (vw) return MM_NA_VEC(8);
#undef MM_NA_VEC
    return priv ? run(free_cells_kernel<real, 0, true>, free_cells_kernel<real, 1, false>, 1024, tab_bytes)
                : run(free_cells_kernel<real, 0, false>, free_cells_kernel<real, 1, false>, 256, 0);
}

}  // namespace mm

using namespace mm;

extern "C" mm_status mm_free_motors_noalloc(const mm_grid *grid, const mm_params *params, mm_dtype dtype, void *density,
                                            const double *psi, double *Mb_coarse, double *M_free, void *cuda_stream)
{
    if (!grid || !params || !density || !psi || !Mb_coarse || !M_free)
        return fail(nullptr, MM_ERR_INVALID_ARG, "mm_free_motors_noalloc: NULL argument");
    if (dtype != MM_F32 && dtype != MM_F64) return fail(nullptr, MM_ERR_INVALID_ARG, "mm_free_motors_noalloc: dtype");
    const mm_grid &g = *grid;
    const mm_params &p = *params;
    if (g.nx < 1 || g.ny < 1 || g.ntheta < 1 || g.ns < 1 || g.nxi < 1 || g.neta < 1)
        return fail(nullptr, MM_ERR_INVALID_ARG, "mm_free_motors_noalloc: every grid dimension must be >= 1");
    if ((int64_t)g.nx * g.ny > MM_NOALLOC_MAX_NODES)
        return fail(nullptr, MM_ERR_INVALID_ARG, "mm_free_motors_noalloc: nx * ny = " + std::to_string((int64_t)g.nx * g.ny) +
                                                     " exceeds MM_NOALLOC_MAX_NODES = " + std::to_string(MM_NOALLOC_MAX_NODES) +
                                                     " (the fixed scratch array); use mm_update_free_motors");
    if ((int64_t)g.nx * g.ny * g.ntheta > INT32_MAX || (int64_t)g.ns * g.nxi * g.neta > INT32_MAX)
        return fail(nullptr, MM_ERR_INVALID_ARG, "mm_free_motors_noalloc: grid too large");
    if (!(std::isfinite(p.R) && p.R > 0) || !(std::isfinite(p.s_lo) && std::isfinite(p.s_hi) && p.s_hi > p.s_lo) ||
        !(std::isfinite(p.m_free) && p.m_free >= 0))
        return fail(nullptr, MM_ERR_INVALID_ARG, "mm_free_motors_noalloc: need finite R > 0, s_hi > s_lo, m_free >= 0");
    unsigned char *scratch = nullptr;
    int sms = 0;
    mm_status s = noalloc_setup(&scratch, &sms);
    if (s != MM_OK) return s;
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    return dtype == MM_F64 ? noalloc_impl<double>(g, p, (double *)density, psi, Mb_coarse, M_free, stream, scratch, sms)
                           : noalloc_impl<float>(g, p, (float *)density, psi, Mb_coarse, M_free, stream, scratch, sms);
}
