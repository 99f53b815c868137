// mm_peak.cuh -- register-only FMA issue-rate probe behind mm_measure_fma_peak (include/mm.h): the second roof of the
// fused substep kernels.  Every thread runs ILP independent chains x <- x * a + b with loop-invariant a, b (so the FMA
// unit, not the register file, is what is measured); 32 warps per SM, one CTA per SM.  Product code (sm_100a).
#pragma once
#include <cuda_runtime.h>

namespace mm {

template <typename real>
__global__ void __launch_bounds__(1024, 1) fma_peak_kernel(real *out, real a, real b, int iters)
{
    constexpr int ILP = 8;
    real x[ILP];
#pragma unroll
    for (int i = 0; i < ILP; ++i) x[i] = real(threadIdx.x + i) * real(1e-3);
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u)
#pragma unroll
            for (int i = 0; i < ILP; ++i) x[i] = fma(x[i], a, b);
    }
    real s = 0;
#pragma unroll
    for (int i = 0; i < ILP; ++i) s += x[i];
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;   // keeps the chains alive
}
constexpr int FMA_PEAK_PER_ITER = 8 * 8;   // FMAs per thread and loop iteration

// The same probe with THREE fresh register operands per FMA (coefficient, value and accumulator all change from one
// instruction to the next, as in a stencil whose coefficients are per-lane data): what the register file, not the FMA
// unit, sustains.  The FMAs are volatile so that their order -- no operand repeated by the next instruction -- stays.
__device__ __forceinline__ void fma_acc(float &acc, float a, float b) { asm volatile("fma.rn.f32 %0, %1, %2, %0;" : "+f"(acc) : "f"(a), "f"(b)); }
__device__ __forceinline__ void fma_acc(double &acc, double a, double b) { asm volatile("fma.rn.f64 %0, %1, %2, %0;" : "+d"(acc) : "d"(a), "d"(b)); }
template <typename real>
__global__ void __launch_bounds__(512, 1) fma_fresh_kernel(real *out, const real *in, int iters)
{
    real c[8], x[8], a[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        c[i] = in[i] + real(threadIdx.x) * real(1e-9);   // |c x| < 1: the accumulators stay finite
        x[i] = in[8 + i];
        a[i] = in[16 + i];
    }
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 8; ++r)
#pragma unroll
            for (int i = 0; i < 8; ++i) fma_acc(a[i], c[(i + r) & 7], x[(i + 3 * r + 1) & 7]);
    }
    real s = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += a[i];
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace mm
