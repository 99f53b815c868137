// mm_stream.cuh -- warp-streamed, TMA-fed fused advect+react(+moments) kernel for sm_100a.
//
// Design:
//  * One WARP owns one configuration c at a time (configurations never interact) and
//    streams its Ns offset-planes [Nxi][Neta] in s order.  A warp-private ring of D shared-memory
//    slots is filled by TMA bulk copies (cp.async.bulk -> SASS UBLKCP) completing on mbarriers, P
//    planes per copy; the ring runs across configuration boundaries, so the next configuration's
//    first planes are in flight while the current one finishes.  No block-level barrier in the loop.
//  * A thread owns a QA x CB patch of every plane (rows a, CB contiguous columns b -> 128-bit
//    shared loads and global stores for fp64 CB=2 / fp32 CB=4).  Each interior face flux is computed
//    ONCE (by the cell below/left of the face) and handed to the neighbour patch with a warp
//    shuffle; the only redundant work is one boundary face per patch edge.
//  * The s stencil is one-sided (W >= 0: plane j at level n+1 needs planes j and j-1 at level n), so T
//    consecutive substeps are applied to plane j as soon as it arrives, keeping plane j-1 of every
//    intermediate level in registers: T substeps per HBM pass, no halo, no redundant work
//    ("temporal fusion", BASELINE.json north_star; residency idea of PAPER.md:145).
//  * MOM: the final level also accumulates sum_j m and sum_j s_j m per owned cell; one warp-shuffle
//    reduction per configuration, one plain store -- no atomics (S9).
#pragma once
#include "mm_common.cuh"
#include "mm_ptx.cuh"

namespace mm {

template <typename real, int N>
struct alignas(sizeof(real) * N) Vec {
    real v[N];
};

template <typename real, int NXI, int NETA, int CB, int P, int D, int WARPS>
struct StreamCfg {
    static constexpr int LB = NETA / CB;       // lanes per row
    static constexpr int G = 32 / LB;          // row groups per warp
    static constexpr int QA = NXI / G;         // rows per thread
    static constexpr int PLANE = NXI * NETA;
    static_assert(NETA % CB == 0 && 32 % LB == 0 && LB <= 32 && NXI % G == 0, "unsupported patch shape");
    static_assert((PLANE * sizeof(real)) % 16 == 0, "TMA bulk copies need 16-byte multiples");
    static constexpr size_t RING_BYTES = (size_t)D * P * PLANE * sizeof(real);
    static constexpr size_t TABLE_BYTES = (((size_t)PLANE * sizeof(real)) + 127) / 128 * 128;
    static constexpr size_t SMEM_BYTES = TABLE_BYTES + WARPS * RING_BYTES + (size_t)WARPS * D * sizeof(uint64_t);
};

template <typename real, int NXI, int NETA, int CB, int T, bool MOM, int P, int D, int WARPS>
__global__ void __launch_bounds__(WARPS * 32, 1)
    substep_stream_kernel(const __grid_constant__ KParams<real> kp, const real *__restrict__ in,
                          real *__restrict__ out, double *__restrict__ force, double *__restrict__ torque)
{
    using Cfg = StreamCfg<real, NXI, NETA, CB, P, D, WARPS>;
    constexpr int LB = Cfg::LB, G = Cfg::G, QA = Cfg::QA, PLANE = Cfg::PLANE;
    using V = Vec<real, CB>;

    extern __shared__ __align__(128) unsigned char smem_raw[];
    real *kap_s = reinterpret_cast<real *>(smem_raw);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    real *ring = reinterpret_cast<real *>(smem_raw + Cfg::TABLE_BYTES + (size_t)warp * Cfg::RING_BYTES);
    uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw + Cfg::TABLE_BYTES + (size_t)WARPS * Cfg::RING_BYTES) +
                     warp * D;

    for (int i = threadIdx.x; i < PLANE; i += WARPS * 32) kap_s[i] = kp.kappa[i];
    if (lane == 0) {
#pragma unroll
        for (int d = 0; d < D; ++d) mbar_init(&full[d], 1);
        mbar_fence_init();
    }
    __syncthreads();

    // ---- thread's patch and configuration-independent constants
    const int g = lane / LB, lb = lane - g * LB;
    const int a0 = g * QA, b0 = lb * CB;
    const bool is_g0 = (g == 0), is_gtop = (g == G - 1), is_l0 = (lb == 0), is_lr = (lb == LB - 1);
    uint32_t maskbits = 0;
#pragma unroll
    for (int q = 0; q < QA; ++q)
#pragma unroll
        for (int cb = 0; cb < CB; ++cb)
            if (kp.inside[(a0 + q) * NETA + b0 + cb]) maskbits |= 1u << (q * CB + cb);

    const int ns = kp.ns;
    const int64_t inner = (int64_t)ns * PLANE;
    const int CH = (ns + P - 1) / P;
    const int64_t gw = (int64_t)blockIdx.x * WARPS + warp, nw = (int64_t)gridDim.x * WARPS;
    const int64_t my_n = gw < kp.nc ? (kp.nc - gw + nw - 1) / nw : 0;
    const int64_t total = my_n * CH;

    auto issue = [&](int64_t i) {   // lane 0 only: TMA copy of stream chunk i into its ring slot
        const int64_t k = i / CH;
        const int ch = (int)(i - k * CH);
        const int64_t c = gw + k * nw;
        const int slot = (int)(i % D);
        const int planes = min(P, ns - ch * P);
        const uint32_t bytes = (uint32_t)(planes * PLANE * sizeof(real));
        mbar_expect_tx(&full[slot], bytes);
        tma_load_1d(ring + (size_t)slot * P * PLANE, in + c * inner + (int64_t)ch * P * PLANE, bytes, &full[slot]);
    };
    if (lane == 0)
        for (int64_t i = 0; i < total && i < D; ++i) issue(i);

    // ---- per-configuration registers
    real axi[QA][CB], aeta[QA][CB], c0[QA][CB], cs[QA][CB], abot[CB], aleft[QA];
    real bxi = 0, beta = 0, ct = 0, st = 0;
    real prev[T][QA][CB];
    real S0[QA][CB], S1[QA][CB];

    int64_t k = 0;
    int ch = 0;
    for (int64_t i = 0; i < total; ++i) {
        const int64_t c = gw + k * nw;
        if (ch == 0) {
            // S2-S4, S6 folded into per-thread coefficients (everything that does not depend on s)
            const int kth = (int)(c % kp.ntheta);
            ct = kp.cos_t[kth];
            st = kp.sin_t[kth];
            const real U = kp.U[c], Vv = kp.V[c], Om = kp.Om[c];
            bxi = -kp.dt_dxi * Om * st;    // d/ds_j of dt/dxi * A_xi
            beta = kp.dt_deta * Om * ct;   // d/ds_j of dt/deta * A_eta
#pragma unroll
            for (int q = 0; q < QA; ++q) {
                const real xi = -kp.R + (real(a0 + q) + real(0.5)) * kp.dxi;
                const real xif = -kp.R + real(a0 + q + 1) * kp.dxi;   // face a+1/2
#pragma unroll
                for (int cb = 0; cb < CB; ++cb) {
                    const real eta = -kp.R + (real(b0 + cb) + real(0.5)) * kp.deta;
                    const real etaf = -kp.R + real(b0 + cb + 1) * kp.deta;   // face b+1/2
                    axi[q][cb] = kp.dt_dxi * (U + walk_speed(kp.v0, kp.kload, ct, st, xif, eta) * ct);
                    aeta[q][cb] = kp.dt_deta * (Vv + walk_speed(kp.v0, kp.kload, ct, st, xi, etaf) * st);
                    cs[q][cb] = kp.dt_ds * walk_speed(kp.v0, kp.kload, ct, st, xi, eta);
                    c0[q][cb] = real(1) - cs[q][cb] - kp.dt * kap_s[(a0 + q) * NETA + b0 + cb];
                }
                aleft[q] = kp.dt_deta * (Vv + walk_speed(kp.v0, kp.kload, ct, st, xi, -kp.R) * st);
            }
#pragma unroll
            for (int cb = 0; cb < CB; ++cb) {
                const real eta = -kp.R + (real(b0 + cb) + real(0.5)) * kp.deta;
                abot[cb] = kp.dt_dxi * (U + walk_speed(kp.v0, kp.kload, ct, st, -kp.R, eta) * ct);
            }
#pragma unroll
            for (int l = 0; l < T; ++l)
#pragma unroll
                for (int q = 0; q < QA; ++q)
#pragma unroll
                    for (int cb = 0; cb < CB; ++cb) prev[l][q][cb] = real(0);   // zero inflow at s_lo (S5)
            if (MOM) {
#pragma unroll
                for (int q = 0; q < QA; ++q)
#pragma unroll
                    for (int cb = 0; cb < CB; ++cb) S0[q][cb] = S1[q][cb] = real(0);
            }
        }

        const int slot = (int)(i % D);
        mbar_wait(&full[slot], (uint32_t)((i / D) & 1));
        const real *sp = ring + (size_t)slot * P * PLANE;
        real *oc = out + c * inner;
        const int planes = min(P, ns - ch * P);
        for (int pl = 0; pl < planes; ++pl) {
            const int j = ch * P + pl;
            const real sj = kp.s_lo + (real(j) + real(0.5)) * kp.ds;
            const bool endp = (j < kp.n_end) || (j >= ns - kp.n_end);
            real cur[QA][CB];
#pragma unroll
            for (int q = 0; q < QA; ++q) {
                const V v = *reinterpret_cast<const V *>(sp + pl * PLANE + (a0 + q) * NETA + b0);
#pragma unroll
                for (int cb = 0; cb < CB; ++cb) cur[q][cb] = v.v[cb];
            }
#pragma unroll
            for (int l = 0; l < T; ++l) {
                // ---- xi faces (a+1/2): flux computed by the lower cell, handed up by shuffle
                real mup[CB], Fx[QA][CB], Fxb[CB];
#pragma unroll
                for (int cb = 0; cb < CB; ++cb) {
                    const real t = shfl_down_r(cur[0][cb], LB);
                    mup[cb] = is_gtop ? real(0) : t;   // ghost = 0 beyond +R (S5)
                }
#pragma unroll
                for (int q = 0; q < QA; ++q)
#pragma unroll
                    for (int cb = 0; cb < CB; ++cb) {
                        const real mR = (q + 1 < QA) ? cur[q + 1][cb] : mup[cb];
                        const real A = fma(sj, bxi, axi[q][cb]);
                        const real p = rmax0(A), n = A - p;
                        Fx[q][cb] = fma(p, cur[q][cb], n * mR);
                    }
#pragma unroll
                for (int cb = 0; cb < CB; ++cb) {
                    const real t = shfl_up_r(Fx[QA - 1][cb], LB);
                    const real bnd = rmin0(fma(sj, bxi, abot[cb])) * cur[0][cb];   // face at -R: ghost 0 on the left
                    Fxb[cb] = is_g0 ? bnd : t;
                }
                // ---- eta faces (b+1/2)
                real mrt[QA], Fe[QA][CB], Fel[QA];
#pragma unroll
                for (int q = 0; q < QA; ++q) {
                    const real t = shfl_down_r(cur[q][0], 1);
                    mrt[q] = is_lr ? real(0) : t;
                }
#pragma unroll
                for (int q = 0; q < QA; ++q)
#pragma unroll
                    for (int cb = 0; cb < CB; ++cb) {
                        const real mR = (cb + 1 < CB) ? cur[q][cb + 1] : mrt[q];
                        const real A = fma(sj, beta, aeta[q][cb]);
                        const real p = rmax0(A), n = A - p;
                        Fe[q][cb] = fma(p, cur[q][cb], n * mR);
                    }
#pragma unroll
                for (int q = 0; q < QA; ++q) {
                    const real t = shfl_up_r(Fe[q][CB - 1], 1);
                    const real bnd = rmin0(fma(sj, beta, aleft[q])) * cur[q][0];
                    Fel[q] = is_l0 ? bnd : t;
                }
                // ---- update (S7) with the s flux in coefficient form: c0 = 1 - dt W/ds - dt kappa
#pragma unroll
                for (int q = 0; q < QA; ++q)
#pragma unroll
                    for (int cb = 0; cb < CB; ++cb) {
                        real acc = fma(c0[q][cb], cur[q][cb], kp.dt_src);
                        acc = fma(cs[q][cb], prev[l][q][cb], acc);
                        acc -= Fx[q][cb];
                        acc += (q > 0) ? Fx[q - 1][cb] : Fxb[cb];
                        acc -= Fe[q][cb];
                        acc += (cb > 0) ? Fe[q][cb - 1] : Fel[q];
                        if (endp) acc = fma(-kp.dt_endx * kap_s[(a0 + q) * NETA + b0 + cb], cur[q][cb], acc);
                        prev[l][q][cb] = cur[q][cb];
                        cur[q][cb] = ((maskbits >> (q * CB + cb)) & 1u) ? acc : real(0);
                    }
            }
#pragma unroll
            for (int q = 0; q < QA; ++q) {
                V v;
#pragma unroll
                for (int cb = 0; cb < CB; ++cb) {
                    v.v[cb] = cur[q][cb];
                    if (MOM) {
                        S0[q][cb] += cur[q][cb];
                        S1[q][cb] = fma(sj, cur[q][cb], S1[q][cb]);
                    }
                }
                *reinterpret_cast<V *>(oc + (int64_t)j * PLANE + (a0 + q) * NETA + b0) = v;
            }
        }
        // every lane has consumed this slot (its values fed the stores above): refill it
        __syncwarp();
        if (lane == 0 && i + D < total) issue(i + D);

        if (++ch == CH) {
            if (MOM) {
                // S9: Fx = sum xi_a S0, Fy = sum eta_b S0, tau = sum (eta_b cos - xi_a sin) S1, fp64 from here on
                double fx = 0, fy = 0, tq = 0;
#pragma unroll
                for (int q = 0; q < QA; ++q) {
                    const double xi = -(double)kp.R + ((double)(a0 + q) + 0.5) * (double)kp.dxi;
#pragma unroll
                    for (int cb = 0; cb < CB; ++cb) {
                        const double eta = -(double)kp.R + ((double)(b0 + cb) + 0.5) * (double)kp.deta;
                        fx += xi * (double)S0[q][cb];
                        fy += eta * (double)S0[q][cb];
                        tq += (eta * (double)ct - xi * (double)st) * (double)S1[q][cb];
                    }
                }
                fx = warp_sum(fx);
                fy = warp_sum(fy);
                tq = warp_sum(tq);
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
}

}  // namespace mm
