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

}  // namespace mm
