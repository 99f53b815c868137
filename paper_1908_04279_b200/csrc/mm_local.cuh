// mm_local.cuh -- SURVEY.md 8(f) NEXT-3: local adaptive time step per independent unit.
// "We instead compute a local dt* for each r0 at the beginning of each inner time step and update M_b at each r0
// asynchronously"; Alg. 2 l.2-5: t*_end = t + dt; while t* < t*_end: compute adaptive
// dt*; "restricted by the motor speed and binding/unbinding rates".  Readings Q31-Q33: the
// unit is the configuration c; lambda_c = the S8 positivity rate maximised over its disc cells; n_c = max(1,
// ceil(dt lambda_c / cfl)) equal local steps dt / n_c.
#pragma once
#include "mm_common.cuh"

namespace mm {

struct LocalParams {   // fp64 copies of what the rate needs, whatever the context dtype
    double v0, f_stall, R, dxi, deta, ds, s_lo, k_spring, k_off0, f_detach, end_mult;
    double dt, cfl;
    int32_t ns, nxi, neta, ntheta, n_end;
};

__device__ __forceinline__ double walk_d(const LocalParams &p, double ct, double st, double xi, double eta)
{
    // same expression order as the model definition S3: v0 * max(0, 1 - k (xi cos + eta sin) / f_stall)
    const double load = p.k_spring * (xi * ct + eta * st) / p.f_stall;
    const double f = 1.0 - load;
    return p.v0 * (f > 0.0 ? f : 0.0);
}

// lambda_c, n_c and dt_c for every configuration; one warp per configuration, fp64 throughout (the step COUNT is an
// integer decided by floating point: it is taken in fp64 from the velocities as stored, in every context dtype).
// For fixed (a, b) the rate is convex in s_j inside each zone of constant end-detachment factor, so its maximum
// over a zone sits at the zone's first or last plane: only those (at most 6) planes are evaluated.
template <typename real>
__global__ void __launch_bounds__(256) local_rate_kernel(const LocalParams p, int64_t nc, const real *__restrict__ U,
                                                         const real *__restrict__ V, const real *__restrict__ Om,
                                                         const uint8_t *__restrict__ inside, double *__restrict__ lambda,
                                                         int32_t *__restrict__ n_steps, real *__restrict__ dt_c,
                                                         int32_t *__restrict__ n_max /* [2]: max, -min */)
{
    const int lane = threadIdx.x & 31;
    const int64_t warp0 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = ((int64_t)gridDim.x * blockDim.x) >> 5;
    int jl[6], nj = 0;
    {
        const int cand[6] = {0, p.n_end - 1, p.n_end, p.ns - p.n_end - 1, p.ns - p.n_end, p.ns - 1};
        for (int i = 0; i < 6; ++i) {
            const int j = cand[i];
            bool ok = j >= 0 && j < p.ns;
            for (int k = 0; k < nj; ++k) ok = ok && jl[k] != j;
            if (ok) jl[nj++] = j;
        }
    }
    const int plane = p.nxi * p.neta;
    for (int64_t c = warp0; c < nc; c += nwarps) {
        const int kth = (int)(c % p.ntheta);
        const double th = 2.0 * 3.14159265358979323846264338327950288 * (double)kth / (double)p.ntheta;
        const double ct = cos(th), st = sin(th);
        const double Uc = (double)U[c], Vc = (double)V[c], Oc = (double)Om[c];
        double lam = 0.0;
        for (int i = lane; i < plane; i += 32) {
            if (!inside[i]) continue;
            const int a = i / p.neta, b = i - a * p.neta;
            const double xi = -p.R + (a + 0.5) * p.dxi, eta = -p.R + (b + 0.5) * p.deta;
            const double W = walk_d(p, ct, st, xi, eta);
            const double wxh = walk_d(p, ct, st, -p.R + (a + 1) * p.dxi, eta) * ct, wxl = walk_d(p, ct, st, -p.R + a * p.dxi, eta) * ct;
            const double weh = walk_d(p, ct, st, xi, -p.R + (b + 1) * p.deta) * st, wel = walk_d(p, ct, st, xi, -p.R + b * p.deta) * st;
            const double kap0 = p.k_off0 * exp(p.k_spring * sqrt(xi * xi + eta * eta) / p.f_detach);
            for (int k = 0; k < nj; ++k) {
                const int j = jl[k];
                const double sj = p.s_lo + (j + 0.5) * p.ds;
                const double E = (j < p.n_end || j >= p.ns - p.n_end) ? p.end_mult : 1.0;
                const double Axh = Uc + wxh - sj * Oc * st, Axl = Uc + wxl - sj * Oc * st;
                const double Aeh = Vc + weh + sj * Oc * ct, Ael = Vc + wel + sj * Oc * ct;
                const double rate = W / p.ds + (fmax(Axh, 0.0) - fmin(Axl, 0.0)) / p.dxi +
                                    (fmax(Aeh, 0.0) - fmin(Ael, 0.0)) / p.deta + kap0 * E;
                lam = fmax(lam, rate);
            }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) lam = fmax(lam, __shfl_xor_sync(0xffffffffu, lam, o));
        if (lane == 0) {
            const double need = ceil(p.dt * lam / p.cfl);
            const int32_t n = need < 1.0 ? 1 : (need > 2147483647.0 ? 2147483647 : (int32_t)need);
            lambda[c] = lam;
            n_steps[c] = n;
            dt_c[c] = (real)(p.dt / (double)n);
            atomicMax(n_max, n);   // once per configuration, at the macro cadence -- not on the hot loop
            atomicMax(n_max + 1, -n);
        }
    }
}

// Compact list of the configurations that still owe steps after `done` (order irrelevant: units are independent).
__global__ void __launch_bounds__(256) local_list_kernel(int64_t nc, const int32_t *__restrict__ n_steps, int32_t done,
                                                         int32_t *__restrict__ list, int32_t *__restrict__ count)
{
    for (int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; c < nc; c += (int64_t)gridDim.x * blockDim.x)
        if (n_steps[c] > done) list[atomicAdd(count, 1)] = (int32_t)c;   // macro cadence, not the hot loop
}

// One local Euler step (S2-S7) for the configurations that still have steps to take (step < n_c), a copy for the
// others; one thread per cell, any grid.  `kp` is built for dt = 1: every dt factor is scaled by dt_c here.
template <typename real>
__global__ void __launch_bounds__(256) substep_generic_local_kernel(const __grid_constant__ KParams<real> kp,
                                                                    const real *__restrict__ in, real *__restrict__ out,
                                                                    const int32_t *__restrict__ n_steps,
                                                                    const real *__restrict__ dt_c, int32_t step)
{
    const int ns = kp.ns, nxi = kp.nxi, neta = kp.neta;
    const int64_t plane = (int64_t)nxi * neta, inner = plane * ns, total = inner * kp.nc;
    const bool per_s = kp.flags & 1u, per_o = kp.flags & 2u;
    for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total;
         idx += (int64_t)gridDim.x * blockDim.x) {
        const int64_t c = idx / inner;
        if (step >= n_steps[c]) { out[idx] = in[idx]; continue; }
        const real dtc = dt_c[c];
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
        const real W = walk_speed(kp.v0, kp.kload, ct, st, xi, eta);
        const real m_sm = j > 0 ? at(j - 1, a, b) : (per_s ? at(ns - 1, a, b) : real(0));
        const real div_s = W * m - W * m_sm;
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
        const bool endc = (j < kp.n_end) || (j >= ns - kp.n_end);
        const real kap = kp.kappa[rem];
        // kp.* factors are per unit dt
        real rhs = -kp.dt_ds * div_s - kp.dt_dxi * (Fxh - Fxl) - kp.dt_deta * (Feh - Fel);
        rhs += kp.dt_src - kp.dt * kap * m;
        if (endc) rhs -= kp.dt_endx * kap * m;
        const real acc = fma(dtc, rhs, m);
        out[idx] = kp.inside[rem] ? acc : real(0);
    }
}

}  // namespace mm
