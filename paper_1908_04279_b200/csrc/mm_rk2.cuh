// mm_rk2.cuh -- second scheme (MM_FLAG_RK2_SUPERBEE): the paper's own integrator,
// Runge-Kutta 2 through the half step (Alg. 2 l.9-10) with the Superbee flux
// limiter in the arclength dimension.  Readings Q27-Q30:
//     m* = mask (m^n + (dt/2) L(m^n)),   m^{n+1} = mask (m^n + dt L(m*)),   L(m) = -div F(m) + src - kappa m,
//     F_s[j+1/2] = W (m_j + sigma_j / 2),  sigma_j = maxmod(minmod(2a, b), minmod(a, 2b)),
//     a = m_j - m_{j-1}, b = m_{j+1} - m_j, ghosts beyond both ends of s are 0, F_s[-1/2] = 0;
// (xi, eta) fluxes, reactions and mask as in S5-S7.  Two density buffers suffice, as the paper stresses: stage 2
// reads m* through the stencil but m^n only at its own cell, so it overwrites m^n in place.
#pragma once
#include "mm_common.cuh"

namespace mm {

template <typename real> __device__ __forceinline__ real minmod2(real a, real b)
{
    if (a * b <= real(0)) return real(0);
    return a > real(0) ? (a < b ? a : b) : (a > b ? a : b);
}
template <typename real> __device__ __forceinline__ real maxmod2(real a, real b)
{
    if (a * b <= real(0)) return real(0);
    return a > real(0) ? (a > b ? a : b) : (a < b ? a : b);
}
// Superbee-limited slope, division-free (= phi(r) b, phi(r) = max(0, min(2r,1), min(r,2)), r = a/b)
template <typename real> __device__ __forceinline__ real superbee_slope(real a, real b)
{
    return maxmod2(minmod2(real(2) * a, b), minmod2(a, real(2) * b));
}

// One RK2 stage, one thread per cell, any grid, all flags:  out = inside ? base + dt L(state) : 0, with the
// dt-dependent factors of `kp` built for this stage's dt.  `base` and `out` may alias (stage 2).
template <typename real>
__global__ void __launch_bounds__(256) rk2_stage_generic_kernel(const __grid_constant__ KParams<real> kp,
                                                                const real *base, const real *__restrict__ state,
                                                                real *out)
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
        const real *mc = state + c * inner;
        const int kth = (int)(c % kp.ntheta);
        const real ct = kp.cos_t[kth], st = kp.sin_t[kth];
        const real U = kp.U[c], V = kp.V[c], Om = kp.Om[c];
        const real sj = kp.s_lo + (real(j) + real(0.5)) * kp.ds;
        const real xi = -kp.R + (real(a) + real(0.5)) * kp.dxi, eta = -kp.R + (real(b) + real(0.5)) * kp.deta;
        auto at = [&](int jj, int aa, int bb) -> real { return mc[((int64_t)jj * nxi + aa) * neta + bb]; };
        // value of s-cell jj with the boundary rule: wrap (test flag) or ghost 0
        auto at_s = [&](int jj) -> real {
            if (jj < 0) return per_s ? at(jj + ns, a, b) : real(0);
            if (jj >= ns) return per_s ? at(jj - ns, a, b) : real(0);
            return at(jj, a, b);
        };
        const real m = at(j, a, b);
        // ---- s faces, Superbee-limited, upwind cell j-1 / j (W >= 0)
        const real W = walk_speed(kp.v0, kp.kload, ct, st, xi, eta);
        const real m1 = at_s(j - 1), m2 = at_s(j - 2), p1 = at_s(j + 1);
        const real f_hi = m + real(0.5) * superbee_slope(m - m1, p1 - m);
        real f_lo = m1 + real(0.5) * superbee_slope(m1 - m2, m - m1);
        if (j == 0 && !per_s) f_lo = real(0);   // zero inflow at s_lo (Q9)
        const real div_s = W * f_hi - W * f_lo;
        // ---- (xi, eta) faces: first-order upwind as in substep_generic_kernel (S5)
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
        // ---- reactions (S6) and update (S7) from the base level
        const bool endc = (j < kp.n_end) || (j >= ns - kp.n_end);
        const real kap = kp.kappa[rem];
        real acc = base[idx] - kp.dt_ds * div_s - kp.dt_dxi * (Fxh - Fxl) - kp.dt_deta * (Feh - Fel);
        acc += kp.dt_src - kp.dt * kap * m;
        if (endc) acc -= kp.dt_endx * kap * m;
        out[idx] = kp.inside[rem] ? acc : real(0);
    }
}

}  // namespace mm
