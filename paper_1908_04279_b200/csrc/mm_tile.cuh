// mm_tile.cuh -- the bandwidth kernel: fused advect + react (+ moments), T substeps per HBM pass (sm_100a).
//
// Design:
//  * One WARP streams one configuration c (or CPW small ones side by side) through its Ns offset planes
//    [Nxi][Neta] in s order; configurations never interact, so there is no block-level barrier.
//  * Planes arrive by tiled TMA (cp.async.bulk.tensor.4d, SASS UTMALDG) into a warp-private ring of D slots of
//    P planes, completing on mbarriers.  The tensor map's box starts one cell outside the plane, so the TMA
//    unit's out-of-bounds zero fill delivers every plane already surrounded by its ghost cells (S5: zero inflow
//    across xi, eta = +-R): the stencil has no boundary branches and no boundary selects.
//  * A lane owns a QA x CB patch (CB contiguous eta cells = one 128-bit access) of every plane, 8 cells, and
//    marches along s.  The s stencil is one-sided (W >= 0: plane j at level n+1 needs planes j and j-1 at level
//    n), so T consecutive substeps are applied to plane j as soon as it arrives, with plane j-1 of every
//    intermediate level held in registers: T substeps per HBM pass, no halo in s, no redundant work (temporal
//    fusion, BASELINE.json north_star; the residency idea of PAPER.md:145).  Between levels the lanes swap
//    patch-edge values through a warp-private, zero-ringed scratch plane in shared memory (double buffered:
//    one __syncwarp per level).
//  * Arithmetic per cell and level: one FMA per owned face for the scaled face velocity
//    A(j) = A0 + s_j * B, an integer sign test + select for the upwind value (S5: max(A,0) mL + min(A,0) mR ==
//    A * m_upwind), and 6 FMAs for the update in coefficient form (S7).  Everything that does not depend on s
//    (S3, S4, S6) is folded into per-lane registers once per configuration.
//  * MOM: the last level also accumulates the three S9 sums per lane; one shuffle reduction and one plain store
//    per configuration -- no atomics.
#pragma once
#include "mm_common.cuh"
#include "mm_ptx.cuh"
#include "mm_coef.cuh"   // and_mask

namespace mm {

template <typename real, int N>
struct alignas(sizeof(real) * N) TVec {
    real v[N];
};

template <typename real, int NXI, int NETA, int CB, int T, int P, int D, int WARPS>
struct TileCfg {
    static constexpr int CELLS = 8;                       // cells per lane per plane
    static constexpr int LPC = NXI * NETA / CELLS;        // lanes per configuration
    static constexpr int CPW = 32 / LPC;                  // configurations per warp
    static constexpr int LB = NETA / CB;                  // lanes per patch row
    static constexpr int G = LPC / LB;                    // patch rows per configuration
    static constexpr int QA = NXI / G;                    // rows per patch
    static constexpr int RS = NETA + 2 * CB;              // padded row: eta index -CB .. NETA+CB-1 (keeps 128-bit alignment)
    static constexpr int ROWS = NXI + 2;                  // padded rows: xi index -1 .. NXI
    static constexpr int PPLANE = ROWS * RS;              // padded plane, elements
    static constexpr int PLANE = NXI * NETA;
    static_assert(NXI * NETA % CELLS == 0 && LPC >= 1 && LPC <= 32 && 32 % LPC == 0, "plane must map onto a warp");
    static_assert(NETA % CB == 0 && LPC % LB == 0 && NXI % G == 0 && QA * CB == CELLS, "unsupported patch shape");
    static_assert(CB * sizeof(real) == 16, "a patch row is one 128-bit access");
    static_assert((RS * sizeof(real)) % 16 == 0, "TMA box rows are multiples of 16 bytes");
    static constexpr uint32_t BOX_BYTES = (uint32_t)(CPW * P * PPLANE * sizeof(real));
    static constexpr size_t SLOT_BYTES = ((size_t)BOX_BYTES + 127) / 128 * 128;
    static constexpr size_t SCRATCH_BYTES = T > 1 ? ((size_t)2 * CPW * PPLANE * sizeof(real) + 127) / 128 * 128 : 0;
    static constexpr size_t TABLE_BYTES = ((size_t)PLANE * sizeof(real) + 127) / 128 * 128;
    static constexpr size_t WARP_BYTES = D * SLOT_BYTES + SCRATCH_BYTES;
    static constexpr size_t SMEM_BYTES = TABLE_BYTES + WARPS * WARP_BYTES + (size_t)WARPS * D * sizeof(uint64_t);
};

__device__ __forceinline__ bool is_neg(double a) { return __double2hiint(a) < 0; }
__device__ __forceinline__ bool is_neg(float a) { return __float_as_int(a) < 0; }

template <typename real, int NXI, int NETA, int CB, int T, bool MOM, int P, int D, int WARPS, int MINB>
__global__ void __launch_bounds__(WARPS * 32, MINB)
    substep_tile_kernel(const __grid_constant__ KParams<real> kp, const __grid_constant__ CUtensorMap tmap,
                        real *__restrict__ out, double *__restrict__ force, double *__restrict__ torque)
{
    using Cfg = TileCfg<real, NXI, NETA, CB, T, P, D, WARPS>;
    constexpr int LPC = Cfg::LPC, CPW = Cfg::CPW, LB = Cfg::LB, QA = Cfg::QA, RS = Cfg::RS;
    constexpr int PPLANE = Cfg::PPLANE, PLANE = Cfg::PLANE;
    using V = TVec<real, CB>;

    extern __shared__ __align__(128) unsigned char smem_raw[];
    real *kap_s = reinterpret_cast<real *>(smem_raw);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    unsigned char *wbase = smem_raw + Cfg::TABLE_BYTES + (size_t)warp * Cfg::WARP_BYTES;
    real *scratch = reinterpret_cast<real *>(wbase + D * Cfg::SLOT_BYTES);
    uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw + Cfg::TABLE_BYTES + (size_t)WARPS * Cfg::WARP_BYTES) +
                     warp * D;

    for (int i = threadIdx.x; i < PLANE; i += WARPS * 32) kap_s[i] = kp.kappa[i];
    if (T > 1)   // ghost ring of the scratch planes stays zero for the whole kernel
        for (int i = lane; i < 2 * CPW * PPLANE; i += 32) scratch[i] = real(0);
    if (lane == 0) {
        prefetch_tensormap(&tmap);
#pragma unroll
        for (int d = 0; d < D; ++d) mbar_init(&full[d], 1);
        mbar_fence_init();
    }
    __syncthreads();

    // ---- lane's patch and configuration-independent constants
    const int cw = lane / LPC, l = lane - cw * LPC;
    const int g = l / LB, lb = l - g * LB;
    const int a0 = g * QA, b0 = lb * CB;
    const int own = (a0 + 1) * RS + b0 + CB;   // offset of patch cell (0,0) in a padded plane
    int maskw[QA][CB];
#pragma unroll
    for (int q = 0; q < QA; ++q)
#pragma unroll
        for (int cb = 0; cb < CB; ++cb) maskw[q][cb] = kp.inside[(a0 + q) * NETA + b0 + cb] ? -1 : 0;

    const int ns = kp.ns;
    const int64_t inner = (int64_t)ns * PLANE;
    const int CH = (ns + P - 1) / P;
    const int64_t ngroups = (kp.nc + CPW - 1) / CPW;
    const int64_t gw = (int64_t)blockIdx.x * WARPS + warp, nw = (int64_t)gridDim.x * WARPS;
    const int64_t my_n = gw < ngroups ? (ngroups - gw + nw - 1) / nw : 0;
    const int64_t total = my_n * CH;

    // producer state (lane 0): next chunk to request
    int64_t pk = 0;
    int pch = 0, pslot = 0;
    auto issue = [&]() {   // lane 0 only: tiled TMA load of the next stream chunk into its ring slot
        const int64_t grp = gw + pk * nw;
        mbar_expect_tx(&full[pslot], Cfg::BOX_BYTES);
        tma_load_4d(wbase + (size_t)pslot * Cfg::SLOT_BYTES, &tmap, -CB, -1, pch * P, (int)(grp * CPW), &full[pslot]);
        if (++pslot == D) pslot = 0;
        if (++pch == CH) { pch = 0; ++pk; }
    };
    if (lane == 0)
        for (int64_t i = 0; i < total && i < D; ++i) issue();

    // ---- per-configuration registers (S2-S4, S6 folded; everything that does not depend on s)
    real a0x[QA + 1][CB], a0e[QA][CB + 1], c0[QA][CB], cs[QA][CB];
    real bx = 0, be = 0, ct = 0, st = 0;
    real R[T][QA][CB];
    real FX = 0, FY = 0, TQ = 0;
    real xiq[QA], etab[CB];
#pragma unroll
    for (int q = 0; q < QA; ++q) xiq[q] = -kp.R + (real(a0 + q) + real(0.5)) * kp.dxi;
#pragma unroll
    for (int cb = 0; cb < CB; ++cb) etab[cb] = -kp.R + (real(b0 + cb) + real(0.5)) * kp.deta;

    int64_t k = 0, c = 0;
    int ch = 0, slot = 0;
    uint32_t phase = 0;
    bool valid = false;
    for (int64_t i = 0; i < total; ++i) {
        if (ch == 0) {
            c = (gw + k * nw) * CPW + cw;
            valid = c < kp.nc;
            const int64_t ce = valid ? c : kp.nc - 1;
            const int kth = (int)(ce % kp.ntheta);
            ct = kp.cos_t[kth];
            st = kp.sin_t[kth];
            const real U = kp.U[ce], Vv = kp.V[ce], Om = kp.Om[ce];
            bx = -kp.dt_dxi * Om * st;   // d/ds_j of dt/dxi * A_xi   (S4)
            be = kp.dt_deta * Om * ct;   // d/ds_j of dt/deta * A_eta
#pragma unroll
            for (int fq = 0; fq <= QA; ++fq) {
                const real xif = -kp.R + real(a0 + fq) * kp.dxi;   // face below row a0+fq
#pragma unroll
                for (int cb = 0; cb < CB; ++cb)
                    a0x[fq][cb] = kp.dt_dxi * (U + walk_speed(kp.v0, kp.kload, ct, st, xif, etab[cb]) * ct);
            }
#pragma unroll
            for (int q = 0; q < QA; ++q) {
#pragma unroll
                for (int fb = 0; fb <= CB; ++fb) {
                    const real etaf = -kp.R + real(b0 + fb) * kp.deta;   // face left of column b0+fb
                    a0e[q][fb] = kp.dt_deta * (Vv + walk_speed(kp.v0, kp.kload, ct, st, xiq[q], etaf) * st);
                }
#pragma unroll
                for (int cb = 0; cb < CB; ++cb) {
                    cs[q][cb] = kp.dt_ds * walk_speed(kp.v0, kp.kload, ct, st, xiq[q], etab[cb]);
                    c0[q][cb] = real(1) - cs[q][cb] - kp.dt * kap_s[(a0 + q) * NETA + b0 + cb];
                }
            }
#pragma unroll
            for (int lv = 0; lv < T; ++lv)
#pragma unroll
                for (int q = 0; q < QA; ++q)
#pragma unroll
                    for (int cb = 0; cb < CB; ++cb) R[lv][q][cb] = real(0);   // zero inflow at s_lo (S5)
            FX = FY = TQ = real(0);
        }

        mbar_wait(&full[slot], phase);
        const real *sp = reinterpret_cast<const real *>(wbase + (size_t)slot * Cfg::SLOT_BYTES) + cw * P * PPLANE;
        real *oc = out + c * inner;
#pragma unroll
        for (int pl = 0; pl < P; ++pl) {
            const int j = ch * P + pl;
            if (j < ns) {
                const real sj = kp.s_lo + (real(j) + real(0.5)) * kp.ds;
                const bool endp = (j < kp.n_end) || (j >= ns - kp.n_end);
                real Ax[QA + 1][CB], Ae[QA][CB + 1];
#pragma unroll
                for (int fq = 0; fq <= QA; ++fq)
#pragma unroll
                    for (int cb = 0; cb < CB; ++cb) Ax[fq][cb] = fma(sj, bx, a0x[fq][cb]);
#pragma unroll
                for (int q = 0; q < QA; ++q)
#pragma unroll
                    for (int fb = 0; fb <= CB; ++fb) Ae[q][fb] = fma(sj, be, a0e[q][fb]);

                const real *tp = sp + pl * PPLANE;   // level-0 plane with its ghost ring, straight from TMA
                real x[QA][CB];
#pragma unroll
                for (int q = 0; q < QA; ++q) {
                    const V v = *reinterpret_cast<const V *>(tp + own + q * RS);
#pragma unroll
                    for (int cb = 0; cb < CB; ++cb) x[q][cb] = v.v[cb];
                }
#pragma unroll
                for (int lv = 0; lv < T; ++lv) {
                    // ---- patch-edge neighbours of this level
                    real up[CB], dn[CB], lf[QA], rt[QA];
                    {
                        const V vu = *reinterpret_cast<const V *>(tp + own + QA * RS);
                        const V vd = *reinterpret_cast<const V *>(tp + own - RS);
#pragma unroll
                        for (int cb = 0; cb < CB; ++cb) { up[cb] = vu.v[cb]; dn[cb] = vd.v[cb]; }
#pragma unroll
                        for (int q = 0; q < QA; ++q) { lf[q] = tp[own + q * RS - 1]; rt[q] = tp[own + q * RS + CB]; }
                    }
                    // ---- upwind value on every owned face (S5): A < 0 takes the upper/right cell
                    real sx[QA + 1][CB], se[QA][CB + 1];
#pragma unroll
                    for (int fq = 0; fq <= QA; ++fq)
#pragma unroll
                        for (int cb = 0; cb < CB; ++cb) {
                            const real lo = fq == 0 ? dn[cb] : x[fq == 0 ? 0 : fq - 1][cb];
                            const real hi = fq == QA ? up[cb] : x[fq == QA ? 0 : fq][cb];
                            sx[fq][cb] = is_neg(Ax[fq][cb]) ? hi : lo;
                        }
#pragma unroll
                    for (int q = 0; q < QA; ++q)
#pragma unroll
                        for (int fb = 0; fb <= CB; ++fb) {
                            const real lo = fb == 0 ? lf[q] : x[q][fb == 0 ? 0 : fb - 1];
                            const real hi = fb == CB ? rt[q] : x[q][fb == CB ? 0 : fb];
                            se[q][fb] = is_neg(Ae[q][fb]) ? hi : lo;
                        }
                    // ---- update (S7) in coefficient form: c0 = 1 - dt W/ds - dt kappa, cs = dt W/ds
                    real nx[QA][CB];
#pragma unroll
                    for (int q = 0; q < QA; ++q)
#pragma unroll
                        for (int cb = 0; cb < CB; ++cb) {
                            real acc = fma(c0[q][cb], x[q][cb], kp.dt_src);
                            acc = fma(cs[q][cb], R[lv][q][cb], acc);
                            acc = fma(-Ax[q + 1][cb], sx[q + 1][cb], acc);
                            acc = fma(Ax[q][cb], sx[q][cb], acc);
                            acc = fma(-Ae[q][cb + 1], se[q][cb + 1], acc);
                            acc = fma(Ae[q][cb], se[q][cb], acc);
                            if (endp) acc = fma(-kp.dt_endx * kap_s[(a0 + q) * NETA + b0 + cb], x[q][cb], acc);
                            nx[q][cb] = acc;
                        }
#pragma unroll
                    for (int q = 0; q < QA; ++q)
#pragma unroll
                        for (int cb = 0; cb < CB; ++cb) {
                            R[lv][q][cb] = x[q][cb];
                            x[q][cb] = and_mask(nx[q][cb], maskw[q][cb]);   // cells outside the disc are 0 (S7)
                        }
                    if (lv + 1 < T) {
                        // hand the new level to the neighbouring lanes through the scratch plane
                        real *sc = scratch + ((lv & 1) * CPW + cw) * PPLANE;
#pragma unroll
                        for (int q = 0; q < QA; ++q) {
                            V v;
#pragma unroll
                            for (int cb = 0; cb < CB; ++cb) v.v[cb] = x[q][cb];
                            *reinterpret_cast<V *>(sc + own + q * RS) = v;
                        }
                        __syncwarp();
                        tp = sc;
                    }
                }
                // ---- store level T of plane j; S9 partial sums
                if (valid) {
#pragma unroll
                    for (int q = 0; q < QA; ++q) {
                        V v;
#pragma unroll
                        for (int cb = 0; cb < CB; ++cb) v.v[cb] = x[q][cb];
                        *reinterpret_cast<V *>(oc + (int64_t)j * PLANE + (a0 + q) * NETA + b0) = v;
                    }
                }
                if (MOM) {
                    real fxp = 0, fyp = 0;
#pragma unroll
                    for (int q = 0; q < QA; ++q) {
                        real rs = x[q][0];
#pragma unroll
                        for (int cb = 1; cb < CB; ++cb) rs += x[q][cb];
                        fxp = fma(xiq[q], rs, fxp);
                    }
#pragma unroll
                    for (int cb = 0; cb < CB; ++cb) {
                        real csum = x[0][cb];
#pragma unroll
                        for (int q = 1; q < QA; ++q) csum += x[q][cb];
                        fyp = fma(etab[cb], csum, fyp);
                    }
                    FX += fxp;
                    FY += fyp;
                    TQ = fma(sj, ct * fyp - st * fxp, TQ);
                }
                if (T > 1) __syncwarp();   // scratch planes are rewritten by the next plane
            }
        }
        // every lane has read this slot's planes (level 0 is the only reader): refill it
        __syncwarp();
        if (lane == 0 && i + D < total) issue();
        if (++slot == D) { slot = 0; phase ^= 1u; }

        if (++ch == CH) {
            if (MOM) {
                // S9: fp64 from the cross-lane reduction on (fp32 contexts: fp32 within a lane)
                double fx = (double)FX, fy = (double)FY, tq = (double)TQ;
#pragma unroll
                for (int o = LPC / 2; o > 0; o >>= 1) {
                    fx += __shfl_xor_sync(0xffffffffu, fx, o);
                    fy += __shfl_xor_sync(0xffffffffu, fy, o);
                    tq += __shfl_xor_sync(0xffffffffu, tq, o);
                }
                if (l == 0 && valid) {
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
