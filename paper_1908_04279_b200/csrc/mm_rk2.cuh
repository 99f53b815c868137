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
#include "mm_ptx.cuh"
#include "mm_coef.cuh"   // CoefCfg, CVec, and_mask, rabs
#include "mm_tm.cuh"     // tensor memory as lane-private scratch

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
// Local-step mode (n_steps != NULL; NEXT-3 with NEXT-1, Alg. 2 l.5 driving l.9-10): `kp` carries the factors per unit
// dt, configuration c takes the stage with dt = stage * dt_c[c] while step < n_steps[c] and is left untouched after.
template <typename real>
__global__ void __launch_bounds__(256) rk2_stage_generic_kernel(const __grid_constant__ KParams<real> kp,
                                                                const real *base, const real *__restrict__ state,
                                                                real *out, const int32_t *__restrict__ n_steps = nullptr,
                                                                const real *__restrict__ dt_c = nullptr, int32_t step = 0,
                                                                real stage = real(1))
{
    const int ns = kp.ns, nxi = kp.nxi, neta = kp.neta;
    const int64_t plane = (int64_t)nxi * neta, inner = plane * ns, total = inner * kp.nc;
    const bool per_s = kp.flags & 1u, per_o = kp.flags & 2u;
    for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total;
         idx += (int64_t)gridDim.x * blockDim.x) {
        const int64_t c = idx / inner;
        if (n_steps && step >= n_steps[c]) continue;   // this unit has reached t + dt
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
        real acc;
        if (n_steps) {   // factors per unit dt, scaled by this unit's stage step
            real rhs = -kp.dt_ds * div_s - kp.dt_dxi * (Fxh - Fxl) - kp.dt_deta * (Feh - Fel);
            rhs += source_increment(kp, c, j, a, b) - kp.dt * kap * m;
            if (endc) rhs -= kp.dt_endx * kap * m;
            acc = fma(stage * dt_c[c], rhs, base[idx]);
        } else {
            acc = base[idx] - kp.dt_ds * div_s - kp.dt_dxi * (Fxh - Fxl) - kp.dt_deta * (Feh - Fel);
            acc += source_increment(kp, c, j, a, b) - kp.dt * kap * m;
            if (endc) acc -= kp.dt_endx * kap * m;
        }
        out[idx] = kp.inside[rem] ? acc : real(0);
    }
}

// ------------------------------------------------------------------------------------------------------------
// Fused RK2 + Superbee kernel: BOTH stages of one substep in ONE HBM pass (read m^n once, write m^{n+1} once; m*
// never touches memory).  Data movement and patch layout are those of substep_coef_kernel (one warp streams one
// configuration through its planes; 1-D TMA ring; 8 cells per lane).  The s stencil looks one plane downstream
// (the limited slope of cell j needs m_{j+1}), so the two stages run skewed: when plane i arrives the warp
// finishes stage 1 of plane i-1 and then stage 2 of plane i-2; two ghost iterations drain each configuration.
// Per lane and owned cell the state carried between iterations is: m_{i-1}, its backward difference, the stage-1
// flux through its lower s face; the same three for m*; m_{i-2} (the base of stage 2); and the level-independent
// offset coefficients of plane i-1, built once (as in mm_coef.cuh) and used by stage 1 now and stage 2 next time.
// Both stages apply the same operator  D(y) = dt L(y) = c0L y + sum_nb c_nb y_nb + src dt - (F_hi - F_lo):
//     m* = mask m + D(m) / 2,      m^{n+1} = mask m + D(m*).
// Superbee slope without compares:  sigma = (sgn a + sgn b)/2 * max(min(2|a|,|b|), min(|a|,2|b|)).
__device__ __forceinline__ float rmin(float a, float b) { return fminf(a, b); }    // FMNMX, full rate
__device__ __forceinline__ float rmax(float a, float b) { return fmaxf(a, b); }
__device__ __forceinline__ double rmin(double a, double b) { return a < b ? a : b; }   // DSETP + 2 SEL (max.f64 is microcoded)
__device__ __forceinline__ double rmax(double a, double b) { return a > b ? a : b; }
__device__ __forceinline__ float rcopysign(float m, float s) { return copysignf(m, s); }
__device__ __forceinline__ double rcopysign(double m, double s) { return copysign(m, s); }
template <typename real> __device__ __forceinline__ real superbee_half_slope(real a, real b)
{
    const real aa = rabs(a), ab = rabs(b);
    const real t = rmax(rmin(aa + aa, ab), rmin(aa, ab + ab));
    return (rcopysign(real(0.25), a) + rcopysign(real(0.25), b)) * t;   // sigma / 2
}

// The coefficient set of plane i-1 (40 values per lane), built for stage 1, is needed again by stage 2 one iteration
// later: it waits in the warp's block of TENSOR MEMORY (one tcgen05.st, one tcgen05.ld per plane) instead of 40
// registers (fp32: 254 registers, the occupancy limit) or a second build (fp64, where it did not fit: 0.7 KB of spills
// per thread in round 1).  KEEPC = true keeps the round-1 register variant selectable.
// mom != 0: the S9 moments of the new density are reduced in the same pass (as in mm_coef.cuh).
template <typename real, int QA, int CB>
struct Rk2Tm {
    static constexpr int NCV = 5 * QA * CB;                                          // coefficient values per lane
    static constexpr int NSV = 4 * QA * CB;                                          // stage-2 state values per lane
    static constexpr int CW = NCV * (int)sizeof(real) / 4;                            // columns of one coefficient set
    // two coefficient slots (iteration parity: the set of plane i-1 is parked as soon as stage 1 has used it, while
    // the set of plane i-2 is still waiting for stage 2) + the stage-2 state
    static constexpr int COLS = tm_pow2_ge((2 * NCV + NSV) * (int)sizeof(real) / 4) < 32 ? 32 : tm_pow2_ge((2 * NCV + NSV) * (int)sizeof(real) / 4);
};
// N reals to / from consecutive columns, N = sum of powers of two >= 2
template <int N, typename real>
__device__ __forceinline__ void tm_st_any(uint32_t ta, const real *v)
{
    constexpr int H = tm_pow2_ge(N) == N ? N : tm_pow2_ge(N) / 2;
    tm_st<H>(ta, *reinterpret_cast<const real(*)[H]>(v));
    if constexpr (N > H) tm_st_any<N - H, real>(ta + H * (int)sizeof(real) / 4, v + H);
}
template <int N, typename real>
__device__ __forceinline__ void tm_ld_any(uint32_t ta, real *v)
{
    constexpr int H = tm_pow2_ge(N) == N ? N : tm_pow2_ge(N) / 2;
    tm_ld<H>(ta, *reinterpret_cast<real(*)[H]>(v));
    if constexpr (N > H) tm_ld_any<N - H, real>(ta + H * (int)sizeof(real) / 4, v + H);
}

template <typename real, int NXI, int NETA, int CB, int P, int D, int WARPS, int MINB, bool PM, bool CS, bool KEEPC>
__global__ void __launch_bounds__(WARPS * 32, MINB)
    rk2_fused_kernel(const __grid_constant__ KParams<real> kp, const real *__restrict__ in, real *__restrict__ out,
                     double *__restrict__ force, double *__restrict__ torque, int mom)
{
    using Cfg = CoefCfg<real, NXI, NETA, CB, P, D, WARPS, CS>;
    constexpr int LB = Cfg::LB, G = Cfg::G, QA = Cfg::QA, PLANE = Cfg::PLANE, NK = Cfg::NK, NKV = Cfg::NKV;
    constexpr int VW = Cfg::VW;
    using V128 = CVec<real, VW>;
    constexpr int OX = 0, OE = (QA + 1) * CB, OC = OE + QA * (CB + 1);   // offsets of h0x, h0e, c0L0 in the block

    extern __shared__ __align__(128) unsigned char smem_raw[];
    real *kap_s = reinterpret_cast<real *>(smem_raw);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    real *ring = reinterpret_cast<real *>(smem_raw + Cfg::TABLE_BYTES + (size_t)warp * Cfg::WARP_BYTES);
    real *cst = ring + Cfg::RING_BYTES / sizeof(real) + lane * VW;
    uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw + Cfg::TABLE_BYTES + (size_t)WARPS * Cfg::WARP_BYTES) +
                     warp * D;

    using TmR = Rk2Tm<real, QA, CB>;
    static_assert(WARPS == 4, "one tensor-memory lane quarter per warp");
    uint32_t *tm_slot = reinterpret_cast<uint32_t *>(smem_raw + Cfg::SMEM_BYTES);
    for (int i = threadIdx.x; i < PLANE; i += WARPS * 32) kap_s[i] = kp.kappa[i];
    if (lane == 0) {
#pragma unroll
        for (int d = 0; d < D; ++d) mbar_init(&full[d], 1);
        mbar_fence_init();
    }
    if (!KEEPC && warp == 0) tm_alloc(tm_slot, TmR::COLS);
    tm_fence_before_sync();
    __syncthreads();
    tm_fence_after_sync();
    const uint32_t tm_cta = KEEPC ? 0u : *tm_slot;
    const uint32_t tm_c = tm_cta + ((uint32_t)(warp * 32) << 16);   // this warp's lane quarter

    const int g = lane / LB, lb = lane - g * LB;
    const int a0 = g * QA, b0 = lb * CB;
    const bool is_g0 = (g == 0), is_gtop = (g == G - 1), is_l0 = (lb == 0), is_lr = (lb == LB - 1);
    real maskf[QA][CB], srcm[QA][CB], xiq[QA], etab[CB];
    real FX = 0, FY = 0, TQ = 0, ctc = 0, stc = 0;
    int maskw[QA][CB];
#pragma unroll
    for (int q = 0; q < QA; ++q) {
        xiq[q] = -kp.R + (real(a0 + q) + real(0.5)) * kp.dxi;
#pragma unroll
        for (int cb = 0; cb < CB; ++cb) {
            const bool inn = kp.inside[(a0 + q) * NETA + b0 + cb] != 0;
            maskw[q][cb] = -(int)kp.inside[(a0 + q) * NETA + b0 + cb];
            maskf[q][cb] = inn ? real(1) : real(0);
            srcm[q][cb] = maskf[q][cb] * kp.dt_src;
        }
    }
#pragma unroll
    for (int cb = 0; cb < CB; ++cb) etab[cb] = -kp.R + (real(b0 + cb) + real(0.5)) * kp.deta;
    const real hdx = real(0.5) * kp.dt_dxi, hde = real(0.5) * kp.dt_deta;

    const int ns = kp.ns;
    const int64_t inner = (int64_t)ns * PLANE;
    const int CH = (ns + P - 1) / P;
    const int64_t gw = (int64_t)blockIdx.x * WARPS + warp, nw = (int64_t)gridDim.x * WARPS;
    const int64_t my_n = gw < kp.nc ? (kp.nc - gw + nw - 1) / nw : 0;
    const int64_t total = my_n * CH;

    int64_t pk = 0;
    int pch = 0, pslot = 0;
    auto issue = [&]() {   // lane 0 only: TMA bulk copy of the next stream chunk into its ring slot
        const int64_t c = gw + pk * nw;
        const int planes = min(P, ns - pch * P);
        const uint32_t bytes = (uint32_t)(planes * PLANE * sizeof(real));
        mbar_expect_tx(&full[pslot], bytes);
        tma_load_1d(ring + (size_t)pslot * P * PLANE, in + c * inner + (int64_t)pch * P * PLANE, bytes, &full[pslot]);
        if (++pslot == D) pslot = 0;
        if (++pch == CH) { pch = 0; ++pk; }
    };
    if (lane == 0)
        for (int64_t i = 0; i < total && i < D; ++i) issue();

    // ---- per-configuration constants (as in mm_coef.cuh, but for the operator D = dt L: no identity, no s term)
    // kc[OX..] = h0x, kc[OE..] = h0e (half face velocities at s = 0), kc[OC..] = c0L0 = mask (-dt kappa - lin)
    real kc[NKV * VW];
    real Wm[QA][CB];        // mask dt W / ds
    real hbx = 0, hbe = 0;
    // ---- state carried from one plane to the next (see the header comment)
    real x1[QA][CB], a1[QA][CB], Flo1[QA][CB], base2[QA][CB], xs[QA][CB], as_[QA][CB], Flo2[QA][CB];
    real Cp[KEEPC ? 5 : 1][QA][CB];     // offset coefficients of plane i-2: c0L, cxm, cxp, cem, cep (KEEPC only)

    real *oc = out;
    // one skewed iteration: plane i of m arrives as y (zeros for the two ghost iterations)
    auto iter = [&](const int i, const real (&y)[QA][CB]) {
        const int j1 = i - 1, j2 = i - 2;
        // level-independent offset coefficients of plane jp (as in mm_coef.cuh, for the operator D = dt L)
        auto build = [&](const int jp, real (&Cn)[5][QA][CB]) {
            const real sj = kp.s_lo + (real(jp) + real(0.5)) * kp.ds;
            real kl[NKV * VW];
            if (CS) {
#pragma unroll
                for (int v = 0; v < NKV; ++v) {
                    const V128 t = *reinterpret_cast<const V128 *>(cst + v * 32 * VW);
#pragma unroll
                    for (int e = 0; e < VW; ++e) kl[v * VW + e] = t.v[e];
                }
            } else {
#pragma unroll
                for (int e = 0; e < NK; ++e) kl[e] = kc[e];
            }
            real hx[QA + 1][CB], he[QA][CB + 1];
#pragma unroll
            for (int fq = 0; fq <= QA; ++fq)
#pragma unroll
                for (int cb = 0; cb < CB; ++cb) hx[fq][cb] = fma(sj, hbx, kl[OX + fq * CB + cb]);
#pragma unroll
            for (int q = 0; q < QA; ++q)
#pragma unroll
                for (int fb = 0; fb <= CB; ++fb) he[q][fb] = fma(sj, hbe, kl[OE + q * (CB + 1) + fb]);
            const bool endp = (jp < kp.n_end) || (jp >= ns - kp.n_end);
#pragma unroll
            for (int q = 0; q < QA; ++q)
#pragma unroll
                for (int cb = 0; cb < CB; ++cb) {
                    const real sabs = (rabs(hx[q][cb]) + rabs(hx[q + 1][cb])) + (rabs(he[q][cb]) + rabs(he[q][cb + 1]));
                    const real pb = hx[q][cb] + rabs(hx[q][cb]);
                    const real nt = rabs(hx[q + 1][cb]) - hx[q + 1][cb];
                    const real pl_ = he[q][cb] + rabs(he[q][cb]);
                    const real nr = rabs(he[q][cb + 1]) - he[q][cb + 1];
                    const real m = PM ? real(1) : maskf[q][cb];
                    real c0 = PM ? kl[OC + q * CB + cb] - sabs : fma(-m, sabs, kl[OC + q * CB + cb]);
                    if (endp) c0 = fma(PM ? -kp.dt_endx : -kp.dt_endx * m, kap_s[(a0 + q) * NETA + b0 + cb], c0);
                    Cn[0][q][cb] = c0;
                    Cn[1][q][cb] = PM ? pb : m * pb;
                    Cn[2][q][cb] = PM ? nt : m * nt;
                    Cn[3][q][cb] = PM ? pl_ : m * pl_;
                    Cn[4][q][cb] = PM ? nr : m * nr;
                }
#pragma unroll
            for (int cb = 0; cb < CB; ++cb) {
                Cn[1][0][cb] = is_g0 ? real(0) : Cn[1][0][cb];
                Cn[2][QA - 1][cb] = is_gtop ? real(0) : Cn[2][QA - 1][cb];
            }
#pragma unroll
            for (int q = 0; q < QA; ++q) {
                Cn[3][q][0] = is_l0 ? real(0) : Cn[3][q][0];
                Cn[4][q][CB - 1] = is_lr ? real(0) : Cn[4][q][CB - 1];
            }
        };
        real Cn[5][QA][CB];
        build(j1, Cn);
        // D(v) - (F_hi - F_lo) part: offset neighbours + self + source, for state v with coefficient set C
        auto offsets = [&](const real (&v)[QA][CB], const real (&C)[5][QA][CB], real (&acc)[QA][CB]) {
            real up[CB], dn[CB], lf[QA], rt[QA];
#pragma unroll
            for (int cb = 0; cb < CB; ++cb) {
                up[cb] = shfl_down_r(v[0][cb], LB);
                dn[cb] = shfl_up_r(v[QA - 1][cb], LB);
            }
#pragma unroll
            for (int q = 0; q < QA; ++q) {
                rt[q] = shfl_down_r(v[q][0], 1);
                lf[q] = shfl_up_r(v[q][CB - 1], 1);
            }
#pragma unroll
            for (int q = 0; q < QA; ++q)
#pragma unroll
                for (int cb = 0; cb < CB; ++cb) {
                    real t = fma(C[0][q][cb], v[q][cb], PM ? kp.dt_src : srcm[q][cb]);
                    t = fma(C[1][q][cb], q > 0 ? v[q - 1][cb] : dn[cb], t);
                    t = fma(C[2][q][cb], q + 1 < QA ? v[q + 1][cb] : up[cb], t);
                    t = fma(C[3][q][cb], cb > 0 ? v[q][cb - 1] : lf[q], t);
                    t = fma(C[4][q][cb], cb + 1 < CB ? v[q][cb + 1] : rt[q], t);
                    acc[q][cb] = t;
                }
        };
        // ---- stage 1 on plane i-1:  m* = mask m + D(m)/2
        real ms[QA][CB], b1[QA][CB], Fh1[QA][CB];
        {
            real acc[QA][CB];
            offsets(x1, Cn, acc);
            if constexpr (!KEEPC) tm_st_any<TmR::NCV, real>(tm_c + (i & 1) * TmR::CW, &Cn[0][0][0]);   // park it for stage 2 of the next iteration
            const bool valid1 = (j1 >= 0) && (j1 < ns);
#pragma unroll
            for (int q = 0; q < QA; ++q)
#pragma unroll
                for (int cb = 0; cb < CB; ++cb) {
                    b1[q][cb] = y[q][cb] - x1[q][cb];
                    Fh1[q][cb] = Wm[q][cb] * (x1[q][cb] + superbee_half_slope(a1[q][cb], b1[q][cb]));
                    const real dv = (acc[q][cb] - Fh1[q][cb]) + Flo1[q][cb];
                    real r = PM ? and_mask(fma(real(0.5), dv, x1[q][cb]), maskw[q][cb])
                                : fma(real(0.5), dv, maskf[q][cb] * x1[q][cb]);
                    ms[q][cb] = valid1 ? r : real(0);   // ghost planes of m* are 0
                }
        }
        // ---- stage 2 on plane i-2:  m^{n+1} = mask m + D(m*)
        real bs[QA][CB], Fh2[QA][CB], o[QA][CB];
        if constexpr (!KEEPC) {   // the state of stage 2 (m*_{i-2}, its difference and lower-face flux, m_{i-2}) waits in tensor memory too
            real s2[4][QA][CB];
            tm_wait_st();
            tm_ld_any<TmR::NSV, real>(tm_c + 2 * TmR::CW, &s2[0][0][0]);
            tm_wait_ld();
#pragma unroll
            for (int q = 0; q < QA; ++q)
#pragma unroll
                for (int cb = 0; cb < CB; ++cb) {
                    xs[q][cb] = s2[0][q][cb]; as_[q][cb] = s2[1][q][cb]; Flo2[q][cb] = s2[2][q][cb]; base2[q][cb] = s2[3][q][cb];
                }
        }
        {
            real acc[QA][CB];
            if constexpr (KEEPC) {
                offsets(xs, Cp, acc);
            } else {
                real C2[5][QA][CB];
                tm_ld_any<TmR::NCV, real>(tm_c + ((i + 1) & 1) * TmR::CW, &C2[0][0][0]);   // the set of plane i-2, parked one iteration ago
                tm_wait_ld();
                offsets(xs, C2, acc);
            }
#pragma unroll
            for (int q = 0; q < QA; ++q)
#pragma unroll
                for (int cb = 0; cb < CB; ++cb) {
                    bs[q][cb] = ms[q][cb] - xs[q][cb];
                    Fh2[q][cb] = Wm[q][cb] * (xs[q][cb] + superbee_half_slope(as_[q][cb], bs[q][cb]));
                    const real dv = (acc[q][cb] - Fh2[q][cb]) + Flo2[q][cb];
                    o[q][cb] = PM ? and_mask(base2[q][cb] + dv, maskw[q][cb]) : fma(maskf[q][cb], base2[q][cb], dv);
                }
        }
        if (j2 >= 0 && j2 < ns) {
#pragma unroll
            for (int q = 0; q < QA; ++q)
#pragma unroll
                for (int v4 = 0; v4 < CB / VW; ++v4) {
                    V128 v;
#pragma unroll
                    for (int e = 0; e < VW; ++e) v.v[e] = o[q][v4 * VW + e];
                    *reinterpret_cast<V128 *>(oc + q * NETA + v4 * VW) = v;
                }
            oc += PLANE;   // this lane's first cell of the next plane stored (carried: the 64-bit address is not rebuilt)
            if (mom) {   // S9 partial sums of the new density
                const real sj2 = kp.s_lo + (real(j2) + real(0.5)) * kp.ds;
                real fxp = 0, fyp = 0;
#pragma unroll
                for (int q = 0; q < QA; ++q) {
                    real rs = o[q][0];
#pragma unroll
                    for (int cb = 1; cb < CB; ++cb) rs += o[q][cb];
                    fxp = fma(xiq[q], rs, fxp);
                }
#pragma unroll
                for (int cb = 0; cb < CB; ++cb) {
                    real csum = o[0][cb];
#pragma unroll
                    for (int q = 1; q < QA; ++q) csum += o[q][cb];
                    fyp = fma(etab[cb], csum, fyp);
                }
                FX += fxp;
                FY += fyp;
                TQ = fma(sj2, ctc * fyp - stc * fxp, TQ);
            }
        }
        // ---- rotate the state
        if constexpr (!KEEPC) {
            real s2[4][QA][CB];
#pragma unroll
            for (int q = 0; q < QA; ++q)
#pragma unroll
                for (int cb = 0; cb < CB; ++cb) {
                    s2[0][q][cb] = ms[q][cb]; s2[1][q][cb] = bs[q][cb]; s2[2][q][cb] = Fh2[q][cb]; s2[3][q][cb] = x1[q][cb];
                }
            tm_st_any<TmR::NSV, real>(tm_c + 2 * TmR::CW, &s2[0][0][0]);
        }
#pragma unroll
        for (int q = 0; q < QA; ++q)
#pragma unroll
            for (int cb = 0; cb < CB; ++cb) {
                if constexpr (!KEEPC) {   // only stage 1's state stays in registers
                    x1[q][cb] = y[q][cb];
                    a1[q][cb] = b1[q][cb];
                    Flo1[q][cb] = Fh1[q][cb];
                    continue;
                }
                base2[q][cb] = x1[q][cb];
                x1[q][cb] = y[q][cb];
                a1[q][cb] = b1[q][cb];
                Flo1[q][cb] = Fh1[q][cb];
                xs[q][cb] = ms[q][cb];
                as_[q][cb] = bs[q][cb];
                Flo2[q][cb] = Fh2[q][cb];
                if constexpr (KEEPC) {
#pragma unroll
                    for (int e = 0; e < 5; ++e) Cp[e][q][cb] = Cn[e][q][cb];
                }
            }
    };

    int64_t k = 0, c = 0;
    int ch = 0, slot = 0;
    uint32_t phase = 0;
    for (int64_t it = 0; it < total; ++it) {
        if (ch == 0) {
            c = gw + k * nw;
            oc = out + c * inner + a0 * NETA + b0;
            const int kth = (int)(c % kp.ntheta);
            const real ct = kp.cos_t[kth], st = kp.sin_t[kth];
            ctc = ct; stc = st;
            FX = FY = TQ = real(0);
            if constexpr (!KEEPC) {   // the parked set read by the first (ghost) stage 2 of this configuration: zeros
                real z[TmR::NCV + TmR::NSV];
#pragma unroll
                for (int e = 0; e < TmR::NCV + TmR::NSV; ++e) z[e] = real(0);
                tm_wait_st();
                tm_st_any<TmR::NCV, real>(tm_c, z);
                tm_st_any<TmR::NCV, real>(tm_c + TmR::CW, z);
                tm_st_any<TmR::NSV, real>(tm_c + 2 * TmR::CW, z);
            }
            const real U = kp.U[c], Vv = kp.V[c], Om = kp.Om[c];
            hbx = -hdx * Om * st;
            hbe = hde * Om * ct;
#pragma unroll
            for (int fq = 0; fq <= QA; ++fq) {
                const real xif = -kp.R + real(a0 + fq) * kp.dxi;
#pragma unroll
                for (int cb = 0; cb < CB; ++cb)
                    kc[OX + fq * CB + cb] = hdx * (U + walk_speed(kp.v0, kp.kload, ct, st, xif, etab[cb]) * ct);
            }
#pragma unroll
            for (int q = 0; q < QA; ++q) {
#pragma unroll
                for (int fb = 0; fb <= CB; ++fb) {
                    const real etaf = -kp.R + real(b0 + fb) * kp.deta;
                    kc[OE + q * (CB + 1) + fb] = hde * (Vv + walk_speed(kp.v0, kp.kload, ct, st, xiq[q], etaf) * st);
                }
#pragma unroll
                for (int cb = 0; cb < CB; ++cb) {
                    const real w = kp.dt_ds * walk_speed(kp.v0, kp.kload, ct, st, xiq[q], etab[cb]);
                    const real lin = (kc[OX + (q + 1) * CB + cb] - kc[OX + q * CB + cb]) +
                                     (kc[OE + q * (CB + 1) + cb + 1] - kc[OE + q * (CB + 1) + cb]);
                    const real c0 = -kp.dt * kap_s[(a0 + q) * NETA + b0 + cb] - lin;
                    Wm[q][cb] = PM ? w : maskf[q][cb] * w;
                    kc[OC + q * CB + cb] = PM ? c0 : maskf[q][cb] * c0;
                }
            }
            if (CS) {
#pragma unroll
                for (int v = 0; v < NKV; ++v) {
                    V128 t;
#pragma unroll
                    for (int e = 0; e < VW; ++e) t.v[e] = (v * VW + e < NK) ? kc[v * VW + e] : real(0);
                    *reinterpret_cast<V128 *>(cst + v * 32 * VW) = t;
                }
            }
#pragma unroll
            for (int q = 0; q < QA; ++q)
#pragma unroll
                for (int cb = 0; cb < CB; ++cb) {
                    x1[q][cb] = a1[q][cb] = Flo1[q][cb] = base2[q][cb] = real(0);   // ghosts below s_lo are 0 (S5)
                    xs[q][cb] = as_[q][cb] = Flo2[q][cb] = real(0);
#pragma unroll
                    for (int e = 0; e < (KEEPC ? 5 : 1); ++e) Cp[e][q][cb] = real(0);
                }
        }

        mbar_wait(&full[slot], phase);
        const real *sp = ring + (size_t)slot * P * PLANE;
        constexpr int UNRP = sizeof(real) == 8 ? 1 : P;   // fp64: one copy of the iteration body (register pressure)
#pragma unroll UNRP
        for (int pl = 0; pl < P; ++pl) {
            const int j = ch * P + pl;
            if (j < ns) {
                real y[QA][CB];
#pragma unroll
                for (int q = 0; q < QA; ++q)
#pragma unroll
                    for (int v4 = 0; v4 < CB / VW; ++v4) {
                        const V128 v = *reinterpret_cast<const V128 *>(sp + pl * PLANE + (a0 + q) * NETA + b0 + v4 * VW);
#pragma unroll
                        for (int e = 0; e < VW; ++e) y[q][v4 * VW + e] = v.v[e];
                    }
                iter(j, y);
            }
        }
        // every lane has copied this slot's planes into registers: refill it
        __syncwarp();
        if (lane == 0 && it + D < total) issue();
        if (++slot == D) { slot = 0; phase ^= 1u; }

        if (++ch == CH) {
            // two ghost planes (0 beyond s_hi) finish stage 1 of plane ns-1 and stage 2 of planes ns-2, ns-1
            real z[QA][CB];
#pragma unroll
            for (int q = 0; q < QA; ++q)
#pragma unroll
                for (int cb = 0; cb < CB; ++cb) z[q][cb] = real(0);
#pragma unroll 1
            for (int e = 0; e < 2; ++e) iter(ns + e, z);
            if (mom) {   // S9: fp64 from the cross-lane reduction on
                double fx = warp_sum((double)FX), fy = warp_sum((double)FY), tq = warp_sum((double)TQ);
                if (lane == 0) {
                    force[2 * c] = kp.mom_scale * fx;
                    force[2 * c + 1] = kp.mom_scale * fy;
                    torque[c] = kp.mom_scale * tq;
                }
            }
            ch = 0;
            ++k;
        }
    }
    if constexpr (!KEEPC) {
        tm_wait_st();
        tm_fence_before_sync();
        __syncthreads();
        if (warp == 0) tm_dealloc(tm_cta, TmR::COLS);
    }
}

}  // namespace mm
