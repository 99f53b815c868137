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
    real dt_kon;                       // dt * k_on  (coupled source: dt k_on M_f(r0))
    real dt_endx;                      // dt * (end_detach_mult - 1)         (S6)
    double mom_scale;                  // -k_spring * ds*dxi*deta            (S9)
    double pf_scale;                   // -k_spring * dxi*deta: scale of a plane force (NEXT-4), = mom_scale / ds
    // per-configuration inputs and tables (device pointers)
    const real *U, *V, *Om;            // [nc]
    const real *cos_t, *sin_t;         // [ntheta], cos/sin(2 pi k / ntheta) evaluated in fp64
    const real *kappa;                 // [nxi*neta], k_off0 * exp(k r_ab / f_d) evaluated in fp64 (S6)
    const uint8_t *inside;             // [nxi*neta], 1 inside the capture disc (S1)
    const double *Mf;                  // NULL, or the free-motor table [nx][ny] (NEXT-2); generic kernels only
    const real *Mf_r;                  // the same table rounded to `real` (fp64 contexts: the table itself): what the
                                       // coefficient-form kernels gather -- no conversion per cell, half the bytes in L1
    const unsigned short *node_x, *node_y;   // NULL, or the context's anchor-node tables (mm_free.cuh, node_table_kernel)
    int32_t nx, ny;
    double geo_R, geo_dxi, geo_deta, geo_ds, geo_s_lo;   // fp64 geometry for the anchor map (never rounded to fp32)
};

// S3: walking speed with the stall clamp; `load` = kload * (xi cos + eta sin)
template <typename real>
__device__ __forceinline__ real walk_speed(real v0, real kload, real ct, real st, real xi, real eta)
{
    real f = real(1) - kload * (xi * ct + eta * st);
    return v0 * (f > real(0) ? f : real(0));
}

// Source increment of a cell: dt k_on m_free, or -- with the free-motor table of SURVEY.md 8(f) NEXT-2 -- dt k_on M_f at
// the nearest node to the cell's anchor r0 = x_c + s_j p_c - (xi_a, eta_b) (readings Q38, Q39, Q42).  The node is an
// integer decided by floating point, so it is computed in fp64 by the oracle's expression in every context dtype.
template <typename real>
__device__ __forceinline__ real source_increment(const KParams<real> &kp, int64_t c, int j, int a, int b)
{
    if (!kp.Mf) return kp.dt_src;
    const int itheta = (int)(c % kp.ntheta);
    const int iy = (int)((c / kp.ntheta) % kp.ny), ix = (int)(c / ((int64_t)kp.ntheta * kp.ny));
    const double theta = 2.0 * 3.14159265358979323846264338327950288 * (double)itheta / (double)kp.ntheta;
    // every operation rounded separately (no FMA contraction), as the oracle does: exact ties (an anchor half-way
    // between two nodes, e.g. at theta = 0 on some grids) must break the same way on both sides
    const double sj = __dadd_rn(kp.geo_s_lo, __dmul_rn(j + 0.5, kp.geo_ds));
    const double xi = __dadd_rn(-kp.geo_R, __dmul_rn(a + 0.5, kp.geo_dxi)), eta = __dadd_rn(-kp.geo_R, __dmul_rn(b + 0.5, kp.geo_deta));
    const double rx = __dmul_rn(__dsub_rn(__dadd_rn(__ddiv_rn((double)ix, (double)kp.nx), __dmul_rn(sj, cos(theta))), xi), (double)kp.nx);
    const double ry = __dmul_rn(__dsub_rn(__dadd_rn(__ddiv_rn((double)iy, (double)kp.ny), __dmul_rn(sj, sin(theta))), eta), (double)kp.ny);
    long nx_ = (long)floor(__dadd_rn(rx, 0.5)) % kp.nx, ny_ = (long)floor(__dadd_rn(ry, 0.5)) % kp.ny;
    if (nx_ < 0) nx_ += kp.nx;
    if (ny_ < 0) ny_ += kp.ny;
    return kp.dt_kon * (real)kp.Mf[nx_ * kp.ny + ny_];
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
