// mm_free.cuh -- SURVEY.md 8(f) NEXT-2: free-motor coupling.
// Eq. 5 M_b,coarse = iiint M_b Psi ds dx dtheta per r0; Eq. 6 M_f = M - M_b,coarse; Alg. 2
// l.14-20: reduction, cap (scale all M_b of an r0 whose coarse density exceeds M_total), M_f.
// Readings Q38-Q42: anchor r0 = x_c + s_j p_c - (xi_a, eta_b), binned to the NEAREST node of the periodic
// (x, y) grid; M_b,coarse[n] = dtheta ds dxi deta sum_{cells -> n} Psi_c m; M_total = m_free; f[n] = min(1, M_total /
// M_b,coarse[n]); M_f[n] = M_total - min(M_b,coarse[n], M_total); source of Eq. 4 = k_on M_f(r0) 1_disc.
// The node of an anchor is an integer decided by floating point: it is taken in fp64, by the same expression, in
// every context dtype.
#pragma once
#include "mm_common.cuh"

namespace mm {

struct FreeGeom {   // fp64 geometry of the anchor map
    double R, dxi, deta, ds, s_lo;
    int32_t ns, nxi, neta, ntheta, nx, ny;
};

__device__ __forceinline__ int anchor_node(const FreeGeom &q, int ix, int iy, double ct, double st, double sj, double xi,
                                           double eta)
{
    // every operation rounded separately (no FMA contraction), as the oracle does: exact ties must break alike
    const double rx = __dmul_rn(__dsub_rn(__dadd_rn(__ddiv_rn((double)ix, (double)q.nx), __dmul_rn(sj, ct)), xi), (double)q.nx);
    const double ry = __dmul_rn(__dsub_rn(__dadd_rn(__ddiv_rn((double)iy, (double)q.ny), __dmul_rn(sj, st)), eta), (double)q.ny);
    long nx_ = (long)floor(__dadd_rn(rx, 0.5)) % q.nx, ny_ = (long)floor(__dadd_rn(ry, 0.5)) % q.ny;
    if (nx_ < 0) nx_ += q.nx;
    if (ny_ < 0) ny_ += q.ny;
    return (int)(nx_ * q.ny + ny_);
}

// floor(r) wrapped into [0, n) without integer division (same construction as wrap_node in mm_coef.cuh)
__device__ __forceinline__ int wrap_floor(double r, int n)
{
    const double f = floor(r), qd = floor(f * (1.0 / (double)n));
    int m = __double2int_rn(f - qd * (double)n);
    m += m < 0 ? n : 0;
    m -= m >= n ? n : 0;
    return m;
}

// MODE 0: raw[n] += w Psi_c m over all cells (fp64 atomic adds, macro cadence).  MODE 1: m *= f[n] (cap rescale), skipped
// entirely when no node was capped.  One warp per configuration, lanes stride over the cells of each plane.
template <typename real, int MODE>
__global__ void __launch_bounds__(256) free_cells_kernel(const FreeGeom q, int64_t nc, real *__restrict__ dens,
                                                         const double *__restrict__ psi, double w, double *__restrict__ raw,
                                                         const double *__restrict__ factor, const int *__restrict__ any_capped)
{
    if (MODE == 1 && *any_capped == 0) return;
    const int lane = threadIdx.x & 31;
    const int64_t warp0 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = ((int64_t)gridDim.x * blockDim.x) >> 5;
    const int plane = q.nxi * q.neta;
    for (int64_t c = warp0; c < nc; c += nwarps) {
        const int itheta = (int)(c % q.ntheta);
        const int iy = (int)((c / q.ntheta) % q.ny), ix = (int)(c / ((int64_t)q.ntheta * q.ny));
        const double theta = 2.0 * 3.14159265358979323846264338327950288 * (double)itheta / (double)q.ntheta;
        const double ct = cos(theta), st = sin(theta);
        const double wp = MODE == 0 ? w * psi[c] : 0.0;
        real *mc = dens + c * (int64_t)plane * q.ns;
        const bool small = q.nxi <= 16 && q.neta <= 16;   // node index separates: 32 node coordinates per plane, not 2 per cell
        for (int j = 0; j < q.ns; ++j) {
            const double sj = __dadd_rn(q.s_lo, __dmul_rn(j + 0.5, q.ds));
            int my_node = 0;   // lanes 0..15: x node of row a = lane (times ny); lanes 16..31: y node of column b = lane - 16
            if (small) {
                const int k = lane & 15;
                if (lane < 16) {
                    const double xi = __dadd_rn(-q.R, __dmul_rn(k + 0.5, q.dxi));
                    const double rx = __dmul_rn(__dsub_rn(__dadd_rn(__ddiv_rn((double)ix, (double)q.nx), __dmul_rn(sj, ct)), xi), (double)q.nx);
                    my_node = wrap_floor(__dadd_rn(rx, 0.5), q.nx) * q.ny;
                } else {
                    const double eta = __dadd_rn(-q.R, __dmul_rn(k + 0.5, q.deta));
                    const double ry = __dmul_rn(__dsub_rn(__dadd_rn(__ddiv_rn((double)iy, (double)q.ny), __dmul_rn(sj, st)), eta), (double)q.ny);
                    my_node = wrap_floor(__dadd_rn(ry, 0.5), q.ny);
                }
            }
            for (int i0 = 0; i0 < plane; i0 += 32) {
                const int i = i0 + lane;
                const bool in_plane = i < plane;
                const int a = in_plane ? i / q.neta : 0, b = in_plane ? i - a * q.neta : 0;
                int n;
                if (small) {
                    n = __shfl_sync(0xffffffffu, my_node, a) + __shfl_sync(0xffffffffu, my_node, 16 + b);
                } else {
                    const double xi = __dadd_rn(-q.R, __dmul_rn(a + 0.5, q.dxi)), eta = __dadd_rn(-q.R, __dmul_rn(b + 0.5, q.deta));
                    n = anchor_node(q, ix, iy, ct, st, sj, xi, eta);
                }
                if (!in_plane) continue;
                real *v = mc + (int64_t)j * plane + i;
                if (MODE == 0) {
                    const double val = (double)*v;
                    if (val != 0.0 && wp != 0.0) atomicAdd(&raw[n], wp * val);
                } else {
                    const double f = factor[n];
                    if (f != 1.0) *v = (real)((double)*v * f);
                }
            }
        }
    }
}

// Per node: cap, factor, M_b,coarse, M_f.
__global__ void free_cap_kernel(int nn, double m_total, const double *__restrict__ raw, double *__restrict__ factor,
                                double *__restrict__ Mbc, double *__restrict__ Mf, int *__restrict__ any_capped)
{
    for (int n = blockIdx.x * blockDim.x + threadIdx.x; n < nn; n += gridDim.x * blockDim.x) {
        const double r = raw[n];
        const bool over = r > m_total;
        factor[n] = over ? m_total / r : 1.0;
        const double capped = over ? m_total : r;
        Mbc[n] = capped;
        Mf[n] = m_total - capped;
        if (over) *any_capped = 1;
    }
}

}  // namespace mm
