// mm_generic.cuh -- generic (any grid size, all flags) global-memory kernels.
// One thread per cell, neighbours read straight from global memory (L1/L2 serve the re-reads).
// This is the fallback for grids / flags the warp-streamed kernels do not cover (odd sizes, the
// test-only periodic modes) and the internal baseline they are measured against.
#pragma once
#include "mm_common.cuh"

namespace mm {

// Tables evaluated once per context in fp64 (S1, S2, S6), stored in the context's dtype.
template <typename real>
__global__ void setup_tables_kernel(int nxi, int neta, int ntheta, double R, double k_spring, double k_off0,
                                    double f_detach, int nomask, real *kappa, uint8_t *inside, real *cos_t,
                                    real *sin_t)
{
    const int tid = blockIdx.x * blockDim.x + threadIdx.x;
    const int nthreads = gridDim.x * blockDim.x;
    const double dxi = 2.0 * R / nxi, deta = 2.0 * R / neta;
    for (int i = tid; i < nxi * neta; i += nthreads) {
        const int a = i / neta, b = i % neta;
        const double xi = -R + (a + 0.5) * dxi, eta = -R + (b + 0.5) * deta;
        const double r = sqrt(xi * xi + eta * eta);
        kappa[i] = (real)(k_off0 * exp(k_spring * r / f_detach));   // Bell law (S6)
        const long long u = 2LL * a + 1 - nxi, v = 2LL * b + 1 - neta;
        const long long nx2 = (long long)nxi * nxi, ne2 = (long long)neta * neta;
        inside[i] = nomask ? 1 : (u * u * ne2 + v * v * nx2 <= nx2 * ne2);   // exact integer disc test (S1)
    }
    for (int k = tid; k < ntheta; k += nthreads) {
        const double th = 2.0 * 3.14159265358979323846264338327950288 * (double)k / (double)ntheta;
        cos_t[k] = (real)cos(th);
        sin_t[k] = (real)sin(th);
    }
}

// One explicit substep (S2-S7), one thread per cell, grid-stride.
template <typename real>
__global__ void __launch_bounds__(256) substep_generic_kernel(const __grid_constant__ KParams<real> kp,
                                                              const real *__restrict__ in, real *__restrict__ out)
{
    const int ns = kp.ns, nxi = kp.nxi, neta = kp.neta;
    const int64_t plane = (int64_t)nxi * neta, inner = plane * ns, total = inner * kp.nc;
    const bool per_s = kp.flags & 1u, per_o = kp.flags & 2u;
    for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total;
         idx += (int64_t)gridDim.x * blockDim.x) {
        const int64_t c = idx / inner;
        int rem = (int)(idx - c * inner);
        const int j = rem / (int)plane;
        rem -= j * (int)plane;
        const int a = rem / neta, b = rem - a * neta;
        const real *mc = in + c * inner;
        const int kth = (int)(c % kp.ntheta);
        const real ct = kp.cos_t[kth], st = kp.sin_t[kth];
        const real U = kp.U[c], V = kp.V[c], Om = kp.Om[c];
        const real sj = kp.s_lo + (real(j) + real(0.5)) * kp.ds;
        const real xi = -kp.R + (real(a) + real(0.5)) * kp.dxi, eta = -kp.R + (real(b) + real(0.5)) * kp.deta;
        const real m = mc[rem + (int64_t)j * plane];
        auto at = [&](int jj, int aa, int bb) -> real { return mc[((int64_t)jj * nxi + aa) * neta + bb]; };
        // s faces: upwind cell is always j-1 (W >= 0)
        const real W = walk_speed(kp.v0, kp.kload, ct, st, xi, eta);
        const real m_sm = j > 0 ? at(j - 1, a, b) : (per_s ? at(ns - 1, a, b) : real(0));
        const real div_s = W * m - W * m_sm;
        // xi faces a+1/2 (index a+1) and a-1/2 (index a); periodic: face nxi is face 0 (ONE face)
        real m_am, m_ap, m_bm, m_bp;
        int fa_hi = a + 1, fb_hi = b + 1;
        if (per_o) {
            m_am = at(j, (a + nxi - 1) % nxi, b);
            m_ap = at(j, (a + 1) % nxi, b);
            m_bm = at(j, a, (b + neta - 1) % neta);
            m_bp = at(j, a, (b + 1) % neta);
            if (fa_hi == nxi) fa_hi = 0;
            if (fb_hi == neta) fb_hi = 0;
        } else {
            m_am = a > 0 ? at(j, a - 1, b) : real(0);
            m_ap = a + 1 < nxi ? at(j, a + 1, b) : real(0);
            m_bm = b > 0 ? at(j, a, b - 1) : real(0);
            m_bp = b + 1 < neta ? at(j, a, b + 1) : real(0);
        }
        const real rot_xi = -sj * Om * st, rot_eta = sj * Om * ct;
        const real Axh = U + walk_speed(kp.v0, kp.kload, ct, st, -kp.R + real(fa_hi) * kp.dxi, eta) * ct + rot_xi;
        const real Axl = U + walk_speed(kp.v0, kp.kload, ct, st, -kp.R + real(a) * kp.dxi, eta) * ct + rot_xi;
        const real Aeh = V + walk_speed(kp.v0, kp.kload, ct, st, xi, -kp.R + real(fb_hi) * kp.deta) * st + rot_eta;
        const real Ael = V + walk_speed(kp.v0, kp.kload, ct, st, xi, -kp.R + real(b) * kp.deta) * st + rot_eta;
        const real Fxh = rmax0(Axh) * m + rmin0(Axh) * m_ap;
        const real Fxl = rmax0(Axl) * m_am + rmin0(Axl) * m;
        const real Feh = rmax0(Aeh) * m + rmin0(Aeh) * m_bp;
        const real Fel = rmax0(Ael) * m_bm + rmin0(Ael) * m;
        // reactions
        const bool endc = (j < kp.n_end) || (j >= ns - kp.n_end);
        const real kap = kp.kappa[rem];
        real acc = m - kp.dt_ds * div_s - kp.dt_dxi * (Fxh - Fxl) - kp.dt_deta * (Feh - Fel);
        acc += source_increment(kp, c, j, a, b) - kp.dt * kap * m;
        if (endc) acc -= kp.dt_endx * kap * m;
        out[idx] = kp.inside[rem] ? acc : real(0);
    }
}

// S9 moments, one block per configuration (grid-stride), no atomics: per-thread partial sums,
// warp shuffles, one shared-memory combine, one plain store per configuration.
// fp32 contexts: fp32 partial sums within a thread, fp64 from the warp reduction on (configs[2]).
template <typename real>
__global__ void __launch_bounds__(256) moments_generic_kernel(const __grid_constant__ KParams<real> kp,
                                                              const real *__restrict__ dens,
                                                              double *__restrict__ force, double *__restrict__ torque)
{
    const int ns = kp.ns, nxi = kp.nxi, neta = kp.neta;
    const int plane = nxi * neta, inner = plane * ns;
    __shared__ double red[3][8];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int64_t c = blockIdx.x; c < kp.nc; c += gridDim.x) {
        const real *mc = dens + c * (int64_t)inner;
        const int kth = (int)(c % kp.ntheta);
        const real ct = kp.cos_t[kth], st = kp.sin_t[kth];
        real sx = 0, sy = 0, sq = 0;
        for (int i = threadIdx.x; i < inner; i += blockDim.x) {
            const int j = i / plane, r = i - j * plane, a = r / neta, b = r - a * neta;
            const real sj = kp.s_lo + (real(j) + real(0.5)) * kp.ds;
            const real xi = -kp.R + (real(a) + real(0.5)) * kp.dxi, eta = -kp.R + (real(b) + real(0.5)) * kp.deta;
            const real v = mc[i];
            sx += xi * v;
            sy += eta * v;
            sq += sj * (eta * ct - xi * st) * v;
        }
        double dx = warp_sum((double)sx), dy = warp_sum((double)sy), dq = warp_sum((double)sq);
        if (lane == 0) { red[0][warp] = dx; red[1][warp] = dy; red[2][warp] = dq; }
        __syncthreads();
        if (threadIdx.x == 0) {
            double tx = 0, ty = 0, tq = 0;
            for (int w = 0; w < (int)(blockDim.x >> 5); ++w) { tx += red[0][w]; ty += red[1][w]; tq += red[2][w]; }
            if (force) { force[2 * c] = kp.mom_scale * tx; force[2 * c + 1] = kp.mom_scale * ty; }
            if (torque) torque[c] = kp.mom_scale * tq;
        }
        __syncthreads();
    }
}

// S9 moments for planes that tile a warp (nxi*neta a multiple of 32*VW: the 16x16 and 8x8 BASELINE shapes): one
// WARP per configuration, VW-element (64/128-bit) coalesced loads straight from HBM, a lane's (xi, eta) weights fixed
// once, per-plane partial sums, one fp64 shuffle reduction and one plain store per configuration.  Used when the
// moments are not fused into a substep pass (MM_OPT_FUSE_MOMENTS = 0, and the RK2 / generic paths).
template <typename real, int VW>
__global__ void __launch_bounds__(256) moments_warp_kernel(const __grid_constant__ KParams<real> kp,
                                                           const real *__restrict__ dens, double *__restrict__ force,
                                                           double *__restrict__ torque)
{
    struct alignas(sizeof(real) * VW) Vec { real v[VW]; };
    constexpr int MAXK = 4;                       // vectors per lane per plane (host guarantees plane <= 32*VW*MAXK)
    const int plane = kp.nxi * kp.neta, nk = plane / (32 * VW);
    const int lane = threadIdx.x & 31;
    const int64_t warp0 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = ((int64_t)gridDim.x * blockDim.x) >> 5;
    real wx[MAXK][VW], wy[MAXK][VW];
#pragma unroll
    for (int k = 0; k < MAXK; ++k)
#pragma unroll
        for (int e = 0; e < VW; ++e) {
            const int i = (k * 32 + lane) * VW + e;
            const int a = i / kp.neta, b = i - a * kp.neta;
            wx[k][e] = -kp.R + (real(a) + real(0.5)) * kp.dxi;
            wy[k][e] = -kp.R + (real(b) + real(0.5)) * kp.deta;
        }
    for (int64_t c = warp0; c < kp.nc; c += nwarps) {
        const Vec *mc = reinterpret_cast<const Vec *>(dens + c * (int64_t)plane * kp.ns);
        const int kth = (int)(c % kp.ntheta);
        const real ct = kp.cos_t[kth], st = kp.sin_t[kth];
        real FX = 0, FY = 0, TQ = 0;
#pragma unroll 4
        for (int j = 0; j < kp.ns; ++j) {
            const real sj = kp.s_lo + (real(j) + real(0.5)) * kp.ds;
            real px = 0, py = 0;
#pragma unroll
            for (int k = 0; k < MAXK; ++k)
                if (k < nk) {
                    const Vec v = mc[(int64_t)j * (plane / VW) + k * 32 + lane];
#pragma unroll
                    for (int e = 0; e < VW; ++e) {
                        px = fma(wx[k][e], v.v[e], px);
                        py = fma(wy[k][e], v.v[e], py);
                    }
                }
            FX += px;
            FY += py;
            TQ = fma(sj, ct * py - st * px, TQ);
        }
        const double fx = warp_sum((double)FX), fy = warp_sum((double)FY), tq = warp_sum((double)TQ);
        if (lane == 0) {
            if (force) { force[2 * c] = kp.mom_scale * fx; force[2 * c + 1] = kp.mom_scale * fy; }
            if (torque) torque[c] = kp.mom_scale * tq;
        }
    }
}

}  // namespace mm
