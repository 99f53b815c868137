// mm_common.cuh -- kernel parameter block and small device helpers shared by the libmm kernels.
// Product code (sm_100a).  Shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace mm {

// Everything a substep / moments kernel needs, by value (__grid_constant__).
// Geometry and rates follow DESIGN.md S1-S9 (restating SURVEY.md 8(c)).
template <typename real>
struct KParams {
    int64_t nc;        // configurations
    int32_t ns, nxi, neta, ntheta;
    int32_t n_end;     // end cells at each end of s (S6, Q8)
    uint32_t flags;    // MM_FLAG_*
    // model / geometry in the kernel's arithmetic type
    real v0, kload;    // kload = k_spring / f_stall   (S3)
    real R, dxi, deta, ds, s_lo;
    // dt-dependent factors (refreshed by every mm_substep call)
    real dt, dt_ds, dt_dxi, dt_deta;   // dt, dt/ds, dt/dxi, dt/deta
    real dt_src;                       // dt * k_on * m_free                 (S6)
    real dt_endx;                      // dt * (end_detach_mult - 1)         (S6)
    double mom_scale;                  // -k_spring * ds*dxi*deta            (S9)
    // per-configuration inputs and tables (device pointers)
    const real *U, *V, *Om;            // [nc]
    const real *cos_t, *sin_t;         // [ntheta], cos/sin(2 pi k / ntheta) evaluated in fp64
    const real *kappa;                 // [nxi*neta], k_off0 * exp(k r_ab / f_d) evaluated in fp64 (S6)
    const uint8_t *inside;             // [nxi*neta], 1 inside the capture disc (S1)
};

// S3: walking speed with the stall clamp; `load` = kload * (xi cos + eta sin)
template <typename real>
__device__ __forceinline__ real walk_speed(real v0, real kload, real ct, real st, real xi, real eta)
{
    real f = real(1) - kload * (xi * ct + eta * st);
    return v0 * (f > real(0) ? f : real(0));
}

template <typename real> __device__ __forceinline__ real rmax0(real x) { return x > real(0) ? x : real(0); }
template <typename real> __device__ __forceinline__ real rmin0(real x) { return x < real(0) ? x : real(0); }

__device__ __forceinline__ double shfl_down_r(double v, int d) { return __shfl_down_sync(0xffffffffu, v, d); }
__device__ __forceinline__ float shfl_down_r(float v, int d) { return __shfl_down_sync(0xffffffffu, v, d); }
__device__ __forceinline__ double shfl_up_r(double v, int d) { return __shfl_up_sync(0xffffffffu, v, d); }
__device__ __forceinline__ float shfl_up_r(float v, int d) { return __shfl_up_sync(0xffffffffu, v, d); }

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

}  // namespace mm
