// mm_coef.cuh -- the issue-lean kernel: fused advect + react (+ moments), T substeps per HBM pass (sm_100a).
//
// Same data movement as mm_stream.cuh (one warp streams one configuration through its Ns offset planes; a
// warp-private ring of shared-memory slots filled by 1-D TMA bulk copies on mbarriers; T levels applied to plane j
// as soon as it arrives, plane j-1 of every level kept in registers; direct 128-bit stores).  What differs is the
// arithmetic, rebuilt around the measured issue rates of sm_100a (profiles/r01b_ubench.md): selects, integer
// compares and predicate traffic are half rate, FMNMX-free absolute values ride as operand modifiers, and a
// 64-bit max/min is microcoded.  So:
//  * S5-S7 in COEFFICIENT form.  With the half face velocity h = (dt/2dxi) A the upwind split needs no compare:
//    max(A,0) dt/dxi = h + |h|, min(A,0) dt/dxi = h - |h|.  Everything that does not depend on the level -- the
//    five neighbour coefficients of every owned cell, already multiplied by the disc mask and with the ghost
//    cells' coefficients zeroed -- is built ONCE per plane and reused by all T levels:
//        c0j = mask (1 - dt W/ds - dt kappa_j - [h_t - h_b] - [h_r - h_l]) - mask (|h_t| + |h_b| + |h_r| + |h_l|)
//        cxm = mask (h_b + |h_b|)   cxp = mask (|h_t| - h_t)   cem = mask (h_l + |h_l|)   cep = mask (|h_r| - h_r)
//    ([h_t - h_b] does not depend on s, so it is folded per configuration.)
//  * One level is then 6 FMAs per cell (self + source, s-upwind plane, four offset neighbours) and one shuffle per
//    patch-edge value; there is no select, no compare and no boundary flux in the level loop.  Lanes at the box
//    edge multiply whatever the shuffle returned by an exact 0.
//  * MOM: the last level adds the three S9 sums per lane; one shuffle reduction and one plain store per
//    configuration -- no atomics.
#pragma once
#include <type_traits>
#include "mm_common.cuh"
#include "mm_ptx.cuh"

#ifndef MM_COEF_XSTATIONARY
#define MM_COEF_XSTATIONARY 0   // measured: ptxas reschedules the FMAs anyway, no .reuse gained (profiles/r01e_README.md)
#endif
#ifndef MM_COEF_PACKED
#define MM_COEF_PACKED 0   // measured: 21 % fewer issue slots, same time (profiles/r01c_README.md) -- kept selectable
#endif

namespace mm {

template <typename real, int N>
struct alignas(sizeof(real) * N) CVec {
    real v[N];
};

__device__ __forceinline__ double and_mask(double v, int m)
{
    return __hiloint2double(__double2hiint(v) & m, __double2loint(v) & m);
}
__device__ __forceinline__ float and_mask(float v, int m) { return __int_as_float(__float_as_int(v) & m); }
// fma whose position in the instruction stream is pinned relative to its neighbours (volatile asm): used where the
// ORDER of independent FMAs matters for operand reuse (x-stationary level update)
__device__ __forceinline__ float ofma(float a, float b, float c)
{
    float d;
    asm volatile("fma.rn.f32 %0, %1, %2, %3;" : "=f"(d) : "f"(a), "f"(b), "f"(c));
    return d;
}
__device__ __forceinline__ double ofma(double a, double b, double c) { return fma(a, b, c); }
// floor(r) wrapped into [0, n) without branches or integer division (branches inside the unrolled planes would cost
// the shuffles their convergence guarantee): quotient estimate in fp64, exact remainder, one corrective step each way
__device__ __forceinline__ int wrap_node(double r, int n)
{
    const double f = floor(r), q = floor(f * (1.0 / (double)n));
    int m = __double2int_rn(f - q * (double)n);   // exact: |f| < 2^31, q n is an integer near f
    m += m < 0 ? n : 0;
    m -= m >= n ? n : 0;
    return m;
}
__device__ __forceinline__ float rabs(float x) { return fabsf(x); }
__device__ __forceinline__ double rabs(double x) { return fabs(x); }

#ifndef MM_COEF_RREG
#define MM_COEF_RREG 6   // fuse levels whose upwind plane stays in registers; deeper levels keep it in shared memory
#endif
#ifndef MM_COEF_RREG_F64
#define MM_COEF_RREG_F64 1   // fp64: only the first level's upwind plane in registers (measured, profiles/r01h_README.md)
#endif
template <typename real>
__host__ __device__ constexpr int coef_rs(int T)
{
    return T > (sizeof(real) == 8 ? MM_COEF_RREG_F64 : MM_COEF_RREG) ? T - (sizeof(real) == 8 ? MM_COEF_RREG_F64 : MM_COEF_RREG) : 0;
}

template <typename real, int NXI, int NETA, int CB, int P, int D, int WARPS, bool CS, int RS = 0>
struct CoefCfg {
    static constexpr int LB = NETA / CB;       // lanes per patch row
    static constexpr int G = 32 / LB;          // patch rows per plane
    static constexpr int QA = NXI / G;         // rows per patch
    static constexpr int PLANE = NXI * NETA;
    static_assert(NETA % CB == 0 && 32 % LB == 0 && LB <= 32 && NXI % G == 0 && QA >= 1, "unsupported patch shape");
    static constexpr int VW = CB * sizeof(real) >= 16 ? 16 / sizeof(real) : CB;   // elements per shared/global access
    static_assert((PLANE * sizeof(real)) % 16 == 0 && CB % VW == 0 && (VW * sizeof(real)) % 8 == 0, "16-byte bulk copies, 64/128-bit rows");
    static constexpr size_t RING_BYTES = (size_t)D * P * PLANE * sizeof(real);
    static constexpr size_t TABLE_BYTES = (((size_t)PLANE * sizeof(real)) + 127) / 128 * 128;
    // CS: the per-configuration constants of a lane (h0x, h0e, c0m) live in a warp-private shared-memory block
    // ([vector][lane] so every 128-bit access is conflict-free) and are re-read once per plane, while the plane's
    // coefficient registers are dead -- the fp64 choice, where they would not fit beside 40 coefficient doubles.
    static constexpr int NK = (QA + 1) * CB + QA * (CB + 1) + QA * CB;   // constants per lane
    static constexpr int NKV = (NK + VW - 1) / VW;                       // ... in vectors
    static constexpr size_t CST_BYTES = CS ? (size_t)NKV * 32 * VW * sizeof(real) : 0;
    // RS: levels beyond the register budget keep their upwind plane (plane j-1 at that level) in a warp-private block,
    // [level][row][vector][lane] -- lane-private slots, 128-bit and conflict-free, no synchronisation needed
    static constexpr size_t RSM_BYTES = (size_t)RS * PLANE * sizeof(real);
    static constexpr size_t WARP_BYTES = RING_BYTES + CST_BYTES + RSM_BYTES;
    static constexpr size_t SMEM_BYTES = TABLE_BYTES + WARPS * WARP_BYTES + (size_t)WARPS * D * sizeof(uint64_t);
};

// MF (free-motor coupling): the source of a cell is dt k_on M_f at the nearest node to its anchor
// r0 = x_c + s_j p_c - (xi_a, eta_b) instead of the constant dt k_on m_free.  The node index separates -- its x part
// depends on (j, a) only, its y part on (j, b) -- so at the start of a configuration the warp fills two small
// shared-memory tables, node_x[j][a] and node_y[j][b] (16-bit; Ns (Nxi + Neta) entries, 64 per lane), in fp64 with every
// operation rounded separately exactly as the oracle does (ties); per plane a lane then reads its QA + CB entries and
// gathers its 8 values of M_f (the table is 128 KB at most and lives in L1/L2).  The gathered sources are
// level-independent like the other coefficients.  Needs nx, ny <= 32767 (host-checked).
// LOC (mm_advance_local): every configuration takes its own local step dt_c and only the
// levels it still owes this pass (n_steps[c] - done, clamped to 0..T); `kp` then carries the factors per unit dt and
// they are scaled by dt_c once per configuration.  A LOC pass runs IN PLACE (in == out): plane j of the output
// depends on input planes <= j only, each already copied to shared memory by the time plane j is stored, and a
// configuration is touched by one warp only -- so a pass visits just the configurations in `list` (those still
// unfinished; NULL = all) and the finished ones cost no traffic.  With MOM the moments of a configuration are
// written in the pass in which it finishes.
template <typename real, int NXI, int NETA, int CB, int T, bool MOM, int P, int D, int WARPS, int MINB, bool PM, bool CS,
          bool LOC = false, bool MF = false>
__global__ void __launch_bounds__(WARPS * 32, MINB)
    substep_coef_kernel(const __grid_constant__ KParams<real> kp, const real *__restrict__ in, real *__restrict__ out,
                        double *__restrict__ force, double *__restrict__ torque,
                        const int32_t *__restrict__ n_steps = nullptr, const real *__restrict__ dt_c = nullptr,
                        int32_t done = 0, const int32_t *__restrict__ list = nullptr,
                        const int32_t *__restrict__ list_count = nullptr)
{
    constexpr int RS = coef_rs<real>(T), TR = T - RS;   // levels with the upwind plane in shared memory / in registers
    using Cfg = CoefCfg<real, NXI, NETA, CB, P, D, WARPS, CS, RS>;
    constexpr int LB = Cfg::LB, G = Cfg::G, QA = Cfg::QA, PLANE = Cfg::PLANE, NK = Cfg::NK, NKV = Cfg::NKV;
    constexpr int VW = Cfg::VW;
    constexpr bool XS = MM_COEF_XSTATIONARY != 0;   // operand-reuse-friendly order of the level update
    constexpr bool PK = sizeof(real) == 4 && CB % 2 == 0 && !PM && MM_COEF_PACKED;   // packed f32x2 level loop
    constexpr int UNR = CS ? 1 : P;   // plane-loop unroll: full where registers allow (it removes the R <- x moves)
    using V128 = CVec<real, VW>;
    constexpr int OX = 0, OE = (QA + 1) * CB, OC = OE + QA * (CB + 1);   // offsets of h0x, h0e, c0m in the block

    extern __shared__ __align__(128) unsigned char smem_raw[];
    real *kap_s = reinterpret_cast<real *>(smem_raw);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    real *ring = reinterpret_cast<real *>(smem_raw + Cfg::TABLE_BYTES + (size_t)warp * Cfg::WARP_BYTES);
    real *cst = ring + Cfg::RING_BYTES / sizeof(real) + lane * VW;   // this lane's column of the constants block
    real *rsm = ring + (Cfg::RING_BYTES + Cfg::CST_BYTES) / sizeof(real) + lane * VW;   // ... of the upwind-plane block
    uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw + Cfg::TABLE_BYTES + (size_t)WARPS * Cfg::WARP_BYTES) +
                     warp * D;

    for (int i = threadIdx.x; i < PLANE; i += WARPS * 32) kap_s[i] = kp.kappa[i];
    if (lane == 0) {
#pragma unroll
        for (int d = 0; d < D; ++d) mbar_init(&full[d], 1);
        mbar_fence_init();
    }
    __syncthreads();

    // ---- lane's patch and configuration-independent constants
    const int g = lane / LB, lb = lane - g * LB;
    const int a0 = g * QA, b0 = lb * CB;
    const bool is_g0 = (g == 0), is_gtop = (g == G - 1), is_l0 = (lb == 0), is_lr = (lb == LB - 1);
    // Disc mask (S1/S7).  PM = false: folded into every coefficient (maskf, srcm), free in the level loop.
    // PM = true ("post-mask", the fp64 choice): coefficients stay unmasked and every level's result is ANDed with
    // maskw on the otherwise idle integer pipe -- 32 fewer registers and no mask multiplies on the fp64 pipe.
    real maskf[QA][CB], srcm[QA][CB], xiq[QA], etab[CB];
    int maskw[QA][CB];
#pragma unroll
    for (int q = 0; q < QA; ++q) {
        xiq[q] = -kp.R + (real(a0 + q) + real(0.5)) * kp.dxi;
#pragma unroll
        for (int cb = 0; cb < CB; ++cb) {
            const bool in = kp.inside[(a0 + q) * NETA + b0 + cb] != 0;
            maskw[q][cb] = -(int)kp.inside[(a0 + q) * NETA + b0 + cb];   // 0 / ~0, kept opaque so the AND stays an AND
            maskf[q][cb] = in ? real(1) : real(0);
            srcm[q][cb] = maskf[q][cb] * kp.dt_src;   // S6 source, 0 outside the disc
        }
    }
#pragma unroll
    for (int cb = 0; cb < CB; ++cb) etab[cb] = -kp.R + (real(b0 + cb) + real(0.5)) * kp.deta;
    real hdx = real(0.5) * kp.dt_dxi, hde = real(0.5) * kp.dt_deta;
    real dtc = real(1), dsrc = kp.dt_src;   // LOC: this configuration's local step and source increment
    int nlev = T;                           // LOC: levels this configuration takes in this pass
    bool last_pass = true;                  // LOC: the configuration finishes in this pass (moments are due)
    // MF: this warp's node tables, behind the regular shared-memory layout (host adds WARPS * ns * (NXI + NETA) * 2 bytes)
    unsigned short *nod = reinterpret_cast<unsigned short *>(smem_raw + ((Cfg::SMEM_BYTES + 15) / 16) * 16) +
                          (size_t)warp * kp.ns * (NXI + NETA);

    const int ns = kp.ns;
    const int64_t inner = (int64_t)ns * PLANE;
    const int CH = (ns + P - 1) / P;
    const int64_t gw = (int64_t)blockIdx.x * WARPS + warp, nw = (int64_t)gridDim.x * WARPS;
    const int64_t nact = (LOC && list) ? (int64_t)*list_count : kp.nc;   // configurations this pass visits
    const int64_t my_n = gw < nact ? (nact - gw + nw - 1) / nw : 0;
    const int64_t total = my_n * CH;

    // producer state (lane 0): next chunk to request
    int64_t pk = 0;
    int pch = 0, pslot = 0;
    auto issue = [&]() {   // lane 0 only: TMA bulk copy of the next stream chunk into its ring slot
        const int64_t c = (LOC && list) ? (int64_t)list[gw + pk * nw] : gw + pk * nw;
        const int planes = min(P, ns - pch * P);
        const uint32_t bytes = (uint32_t)(planes * PLANE * sizeof(real));
        mbar_expect_tx(&full[pslot], bytes);
        tma_load_1d(ring + (size_t)pslot * P * PLANE, in + c * inner + (int64_t)pch * P * PLANE, bytes, &full[pslot]);
        if (++pslot == D) pslot = 0;
        if (++pch == CH) { pch = 0; ++pk; }
    };
    if (lane == 0)
        for (int64_t i = 0; i < total && i < D; ++i) issue();

    // ---- per-configuration registers (S2-S4, S6 folded; everything that does not depend on s)
    // kc[OX + fq*CB + cb]     = h0x: (dt/2dxi)  A_xi  at s = 0 on the xi faces below rows a0 .. a0+QA       (S4)
    // kc[OE + q*(CB+1) + fb]  = h0e: (dt/2deta) A_eta at s = 0 on the eta faces left of columns b0 .. b0+CB
    // kc[OC + q*CB + cb]      = c0m: mask (1 - dt W/ds - dt kappa - [h_t - h_b] - [h_r - h_l])
    real kc[NKV * VW];
    real csm[QA][CB];       // mask dt W/ds                                                            (S5, s flux)
    real hbx = 0, hbe = 0, ct = 0, st = 0;
    real R[TR][QA][CB];     // plane j-1 at levels n .. n+TR-1 (levels TR .. T-1: in shared memory, rsm)
    auto rsm_at = [&](int lv, int q, int v4) { return rsm + (((lv - TR) * QA + q) * (CB / VW) + v4) * 32 * VW; };
    real FX = 0, FY = 0, TQ = 0;

    int64_t k = 0, c = 0;
    int ch = 0, slot = 0;
    uint32_t phase = 0;
    for (int64_t i = 0; i < total; ++i) {
        if (ch == 0) {
            c = (LOC && list) ? (int64_t)list[gw + k * nw] : gw + k * nw;
            const int kth = (int)(c % kp.ntheta);
            ct = kp.cos_t[kth];
            st = kp.sin_t[kth];
            const real U = kp.U[c], Vv = kp.V[c], Om = kp.Om[c];
            if (MF) {
                const double theta = 2.0 * 3.14159265358979323846264338327950288 * (double)kth / (double)kp.ntheta;
                const double mf_ct = cos(theta), mf_st = sin(theta);
                const int iy = (int)((c / kp.ntheta) % kp.ny), ix = (int)(c / ((int64_t)kp.ntheta * kp.ny));
                const double mf_tx = __ddiv_rn((double)ix, (double)kp.nx), mf_ty = __ddiv_rn((double)iy, (double)kp.ny);
                __syncwarp();   // the previous configuration's planes are done with the tables
                for (int e = lane; e < kp.ns * (NXI + NETA); e += 32) {
                    const int jj = e / (NXI + NETA), r = e - jj * (NXI + NETA);
                    const double sjd = __dadd_rn(kp.geo_s_lo, __dmul_rn(jj + 0.5, kp.geo_ds));
                    int n;
                    if (r < NXI) {
                        const double xid = __dadd_rn(-kp.geo_R, __dmul_rn(r + 0.5, kp.geo_dxi));
                        const double hx_ = __dadd_rn(mf_tx, __dmul_rn(sjd, mf_ct));
                        n = wrap_node(__dadd_rn(__dmul_rn(__dsub_rn(hx_, xid), (double)kp.nx), 0.5), kp.nx);
                    } else {
                        const double etd = __dadd_rn(-kp.geo_R, __dmul_rn(r - NXI + 0.5, kp.geo_deta));
                        const double hy_ = __dadd_rn(mf_ty, __dmul_rn(sjd, mf_st));
                        n = wrap_node(__dadd_rn(__dmul_rn(__dsub_rn(hy_, etd), (double)kp.ny), 0.5), kp.ny);
                    }
                    nod[e] = (unsigned short)n;
                }
                __syncwarp();
            }
            if (LOC) {
                dtc = dt_c[c];
                const int owed = n_steps[c] - done;
                nlev = owed < 0 ? 0 : (owed > T ? T : owed);
                last_pass = owed <= T;
                hdx = real(0.5) * kp.dt_dxi * dtc;
                hde = real(0.5) * kp.dt_deta * dtc;
                dsrc = kp.dt_src * dtc;
#pragma unroll
                for (int q = 0; q < QA; ++q)
#pragma unroll
                    for (int cb = 0; cb < CB; ++cb) srcm[q][cb] = maskf[q][cb] * dsrc;
            }
            hbx = -hdx * Om * st;   // d/ds_j of h_xi   (S4: A_xi = U + w cos - s Omega sin)
            hbe = hde * Om * ct;    // d/ds_j of h_eta  (S4: A_eta = V + w sin + s Omega cos)
#pragma unroll
            for (int fq = 0; fq <= QA; ++fq) {
                const real xif = -kp.R + real(a0 + fq) * kp.dxi;   // face below row a0+fq
#pragma unroll
                for (int cb = 0; cb < CB; ++cb)
                    kc[OX + fq * CB + cb] = hdx * (U + walk_speed(kp.v0, kp.kload, ct, st, xif, etab[cb]) * ct);
            }
#pragma unroll
            for (int q = 0; q < QA; ++q) {
#pragma unroll
                for (int fb = 0; fb <= CB; ++fb) {
                    const real etaf = -kp.R + real(b0 + fb) * kp.deta;   // face left of column b0+fb
                    kc[OE + q * (CB + 1) + fb] = hde * (Vv + walk_speed(kp.v0, kp.kload, ct, st, xiq[q], etaf) * st);
                }
#pragma unroll
                for (int cb = 0; cb < CB; ++cb) {
                    const real cs = (LOC ? kp.dt_ds * dtc : kp.dt_ds) * walk_speed(kp.v0, kp.kload, ct, st, xiq[q], etab[cb]);
                    const real lin = (kc[OX + (q + 1) * CB + cb] - kc[OX + q * CB + cb]) +
                                     (kc[OE + q * (CB + 1) + cb + 1] - kc[OE + q * (CB + 1) + cb]);
                    const real c0 = real(1) - cs - (LOC ? kp.dt * dtc : kp.dt) * kap_s[(a0 + q) * NETA + b0 + cb] - lin;
                    csm[q][cb] = PM ? cs : maskf[q][cb] * cs;
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
            for (int lv = 0; lv < T; ++lv)
#pragma unroll
                for (int q = 0; q < QA; ++q) {
                    if (lv < TR) {
#pragma unroll
                        for (int cb = 0; cb < CB; ++cb) R[lv < TR ? lv : 0][q][cb] = real(0);   // zero inflow at s_lo (S5)
                    } else {
#pragma unroll
                        for (int v4 = 0; v4 < CB / VW; ++v4) {
                            V128 z;
#pragma unroll
                            for (int e = 0; e < VW; ++e) z.v[e] = real(0);
                            *reinterpret_cast<V128 *>(rsm_at(lv, q, v4)) = z;
                        }
                    }
                }
            FX = FY = TQ = real(0);
        }

        mbar_wait(&full[slot], phase);
        const real *sp = ring + (size_t)slot * P * PLANE;
        real *oc = out + c * inner;
        // The planes of one chunk for a compile-time number NL of levels.  NL = T except in the LOC variant, where the
        // warp-uniform level count of the configuration selects one of the T+1 straight-line instances below (a
        // run-time `lv < nlev` test inside the unrolled planes would break their copy-free register rotation).
        auto chunk = [&](auto NLC) {
        constexpr int NL = decltype(NLC)::value;
#pragma unroll UNR
        for (int pl = 0; pl < P; ++pl) {
            const int j = ch * P + pl;
            // A ragged last chunk (j >= ns) still runs the arithmetic on whatever the slot holds -- straight-line code
            // keeps the register rotation of the unrolled planes free of copies -- but stores and sums nothing; R is
            // re-zeroed at the next configuration.
            const bool live = j < ns;
            const real sj = kp.s_lo + (real(j) + real(0.5)) * kp.ds;
            if constexpr (MF) {
                const unsigned short *nj = nod + (live ? j : 0) * (NXI + NETA);
                int nodx[QA], nody[CB];
#pragma unroll
                for (int q = 0; q < QA; ++q) nodx[q] = (int)nj[a0 + q] * kp.ny;
#pragma unroll
                for (int cb = 0; cb < CB; ++cb) nody[cb] = (int)nj[NXI + b0 + cb];
#pragma unroll
                for (int q = 0; q < QA; ++q)
#pragma unroll
                    for (int cb = 0; cb < CB; ++cb) {
                        const real sv = kp.dt_kon * __ldg(&kp.Mf_r[nodx[q] + nody[cb]]);
                        srcm[q][cb] = PM ? sv : maskf[q][cb] * sv;
                    }
            }
            // ---- level-independent coefficients of this plane
            real c0j[QA][CB], cxm[QA][CB], cxp[QA][CB], cem[QA][CB], cep[QA][CB];
            {
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
                if constexpr (PK) {
                    // packed build: face velocities and the mask products two columns at a time
                    const float2 sj2 = make_float2(sj, sj), bx2 = make_float2(hbx, hbx), be2 = make_float2(hbe, hbe);
#pragma unroll
                    for (int fq = 0; fq <= QA; ++fq)
#pragma unroll
                        for (int h = 0; h < CB / 2; ++h) {
                            const float2 t = __ffma2_rn(sj2, bx2, make_float2(kl[OX + fq * CB + 2 * h], kl[OX + fq * CB + 2 * h + 1]));
                            hx[fq][2 * h] = t.x;
                            hx[fq][2 * h + 1] = t.y;
                        }
#pragma unroll
                    for (int q = 0; q < QA; ++q) {
#pragma unroll
                        for (int h = 0; h < CB / 2; ++h) {
                            const float2 t = __ffma2_rn(sj2, be2, make_float2(kl[OE + q * (CB + 1) + 2 * h], kl[OE + q * (CB + 1) + 2 * h + 1]));
                            he[q][2 * h] = t.x;
                            he[q][2 * h + 1] = t.y;
                        }
                        he[q][CB] = fmaf(sj, hbe, kl[OE + q * (CB + 1) + CB]);
                    }
#pragma unroll
                    for (int q = 0; q < QA; ++q)
#pragma unroll
                        for (int h = 0; h < CB / 2; ++h) {
                            float2 ns2, pb2, nt2, pl2, nr2;
#pragma unroll
                            for (int e = 0; e < 2; ++e) {
                                const int cb = 2 * h + e;
                                const float nsab = (-rabs(hx[q][cb]) - rabs(hx[q + 1][cb])) + (-rabs(he[q][cb]) - rabs(he[q][cb + 1]));
                                const float pb = hx[q][cb] + rabs(hx[q][cb]);
                                const float nt = rabs(hx[q + 1][cb]) - hx[q + 1][cb];
                                const float pl_ = he[q][cb] + rabs(he[q][cb]);
                                const float nr = rabs(he[q][cb + 1]) - he[q][cb + 1];
                                if (e == 0) { ns2.x = nsab; pb2.x = pb; nt2.x = nt; pl2.x = pl_; nr2.x = nr; }
                                else { ns2.y = nsab; pb2.y = pb; nt2.y = nt; pl2.y = pl_; nr2.y = nr; }
                            }
                            const float2 m2 = make_float2(maskf[q][2 * h], maskf[q][2 * h + 1]);
                            const float2 c2 = __ffma2_rn(m2, ns2, make_float2(kl[OC + q * CB + 2 * h], kl[OC + q * CB + 2 * h + 1]));
                            const float2 a2 = __fmul2_rn(m2, pb2), b2 = __fmul2_rn(m2, nt2), d2 = __fmul2_rn(m2, pl2), e2 = __fmul2_rn(m2, nr2);
                            c0j[q][2 * h] = c2.x; c0j[q][2 * h + 1] = c2.y;
                            cxm[q][2 * h] = a2.x; cxm[q][2 * h + 1] = a2.y;
                            cxp[q][2 * h] = b2.x; cxp[q][2 * h + 1] = b2.y;
                            cem[q][2 * h] = d2.x; cem[q][2 * h + 1] = d2.y;
                            cep[q][2 * h] = e2.x; cep[q][2 * h + 1] = e2.y;
                        }
                } else {
#pragma unroll
                for (int fq = 0; fq <= QA; ++fq)
#pragma unroll
                    for (int cb = 0; cb < CB; ++cb) hx[fq][cb] = fma(sj, hbx, kl[OX + fq * CB + cb]);
#pragma unroll
                for (int q = 0; q < QA; ++q)
#pragma unroll
                    for (int fb = 0; fb <= CB; ++fb) he[q][fb] = fma(sj, hbe, kl[OE + q * (CB + 1) + fb]);
#pragma unroll
                for (int q = 0; q < QA; ++q)
#pragma unroll
                    for (int cb = 0; cb < CB; ++cb) {
                        const real sabs = (rabs(hx[q][cb]) + rabs(hx[q + 1][cb])) + (rabs(he[q][cb]) + rabs(he[q][cb + 1]));
                        const real pb = hx[q][cb] + rabs(hx[q][cb]);               // max(A,0) on the face below
                        const real nt = rabs(hx[q + 1][cb]) - hx[q + 1][cb];       // -min(A,0) on the face above
                        const real pl_ = he[q][cb] + rabs(he[q][cb]);
                        const real nr = rabs(he[q][cb + 1]) - he[q][cb + 1];
                        if (PM) {
                            c0j[q][cb] = kl[OC + q * CB + cb] - sabs;
                            cxm[q][cb] = pb; cxp[q][cb] = nt; cem[q][cb] = pl_; cep[q][cb] = nr;
                        } else {
                            const real m = maskf[q][cb];
                            c0j[q][cb] = fma(-m, sabs, kl[OC + q * CB + cb]);
                            cxm[q][cb] = m * pb; cxp[q][cb] = m * nt; cem[q][cb] = m * pl_; cep[q][cb] = m * nr;
                        }
                    }
                }
                // ghost cells beyond the box are 0 (S5): their coefficient is an exact 0 on the edge lanes
#pragma unroll
                for (int cb = 0; cb < CB; ++cb) {
                    cxm[0][cb] = is_g0 ? real(0) : cxm[0][cb];
                    cxp[QA - 1][cb] = is_gtop ? real(0) : cxp[QA - 1][cb];
                }
#pragma unroll
                for (int q = 0; q < QA; ++q) {
                    cem[q][0] = is_l0 ? real(0) : cem[q][0];
                    cep[q][CB - 1] = is_lr ? real(0) : cep[q][CB - 1];
                }
                if ((j < kp.n_end) || (j >= ns - kp.n_end)) {   // enhanced end detachment (S6)
#pragma unroll
                    for (int q = 0; q < QA; ++q)
#pragma unroll
                        for (int cb = 0; cb < CB; ++cb)
                            c0j[q][cb] = fma(PM ? -(LOC ? kp.dt_endx * dtc : kp.dt_endx)
                                                : -(LOC ? kp.dt_endx * dtc : kp.dt_endx) * maskf[q][cb],
                                             kap_s[(a0 + q) * NETA + b0 + cb], c0j[q][cb]);
                }
            }
            real x[QA][CB];
#pragma unroll
            for (int q = 0; q < QA; ++q)
#pragma unroll
                for (int v4 = 0; v4 < CB / VW; ++v4) {
                    const V128 v = *reinterpret_cast<const V128 *>(sp + pl * PLANE + (a0 + q) * NETA + b0 + v4 * VW);
#pragma unroll
                    for (int e = 0; e < VW; ++e) x[q][v4 * VW + e] = v.v[e];
                }
#pragma unroll
            for (int lv = 0; lv < NL; ++lv) {
                real Rl[QA][CB];   // plane j-1 at this level
#pragma unroll
                for (int q = 0; q < QA; ++q) {
                    if (lv < TR) {
#pragma unroll
                        for (int cb = 0; cb < CB; ++cb) Rl[q][cb] = R[lv < TR ? lv : 0][q][cb];
                    } else {
#pragma unroll
                        for (int v4 = 0; v4 < CB / VW; ++v4) {
                            const V128 t = *reinterpret_cast<const V128 *>(rsm_at(lv, q, v4));
#pragma unroll
                            for (int e = 0; e < VW; ++e) Rl[q][v4 * VW + e] = t.v[e];
                        }
                    }
                }
                real up[CB], dn[CB], lf[QA], rt[QA];
#pragma unroll
                for (int cb = 0; cb < CB; ++cb) {
                    up[cb] = shfl_down_r(x[0][cb], LB);
                    dn[cb] = shfl_up_r(x[QA - 1][cb], LB);
                }
#pragma unroll
                for (int q = 0; q < QA; ++q) {
                    rt[q] = shfl_down_r(x[q][0], 1);
                    lf[q] = shfl_up_r(x[q][CB - 1], 1);
                }
                real nx[QA][CB];
                if constexpr (PK) {
                    // fp32: the four aligned terms of a column pair go through the packed FFMA2 pipe form (same FMA
                    // lanes, half the issue slots -- profiles/r01b_README.md section 0); the two eta neighbours are
                    // misaligned by one column and stay scalar FFMAs on the halves of the pair.
#pragma unroll
                    for (int q = 0; q < QA; ++q)
#pragma unroll
                        for (int h = 0; h < CB / 2; ++h) {
                            const int e0 = 2 * h, e1 = 2 * h + 1;
                            float2 acc = __ffma2_rn(make_float2(c0j[q][e0], c0j[q][e1]), make_float2(x[q][e0], x[q][e1]),
                                                    make_float2(srcm[q][e0], srcm[q][e1]));
                            const float2 below = q > 0 ? make_float2(x[q > 0 ? q - 1 : 0][e0], x[q > 0 ? q - 1 : 0][e1])
                                                       : make_float2(dn[e0], dn[e1]);
                            const float2 above = q + 1 < QA ? make_float2(x[q + 1 < QA ? q + 1 : 0][e0], x[q + 1 < QA ? q + 1 : 0][e1])
                                                            : make_float2(up[e0], up[e1]);
                            acc = __ffma2_rn(make_float2(cxm[q][e0], cxm[q][e1]), below, acc);
                            acc = __ffma2_rn(make_float2(cxp[q][e0], cxp[q][e1]), above, acc);
                            acc.x = fmaf(cem[q][e0], e0 > 0 ? x[q][e0 > 0 ? e0 - 1 : 0] : lf[q], acc.x);
                            acc.y = fmaf(cem[q][e1], x[q][e0], acc.y);
                            acc.x = fmaf(cep[q][e0], x[q][e1], acc.x);
                            acc.y = fmaf(cep[q][e1], e1 + 1 < CB ? x[q][e1 + 1 < CB ? e1 + 1 : 0] : rt[q], acc.y);
                            acc = __ffma2_rn(make_float2(csm[q][e0], csm[q][e1]), make_float2(Rl[q][e0], Rl[q][e1]), acc);
                            nx[q][e0] = acc.x;
                            nx[q][e1] = acc.y;
                        }
                } else {
                if constexpr (XS) {
                    // x-stationary order: a 3-register FFMA issues at half rate unless an operand comes from the reuse
                    // cache (profiles/r01e_README.md: 1.9 vs 3.0 FFMA/clk/SM), so every owned value feeds its (up to 5)
                    // accumulators back to back; the halo values -- still in flight from the shuffles -- come last.
#pragma unroll
                    for (int q = 0; q < QA; ++q)
#pragma unroll
                        for (int cb = 0; cb < CB; ++cb) nx[q][cb] = ofma(csm[q][cb], Rl[q][cb], (PM && !MF) ? dsrc : srcm[q][cb]);
#pragma unroll
                    for (int q = 0; q < QA; ++q)
#pragma unroll
                        for (int cb = 0; cb < CB; ++cb) {
                            const real v = x[q][cb];
                            nx[q][cb] = ofma(c0j[q][cb], v, nx[q][cb]);
                            if (q + 1 < QA) nx[q + 1 < QA ? q + 1 : 0][cb] = ofma(cxm[q + 1 < QA ? q + 1 : 0][cb], v, nx[q + 1 < QA ? q + 1 : 0][cb]);
                            if (q > 0) nx[q > 0 ? q - 1 : 0][cb] = ofma(cxp[q > 0 ? q - 1 : 0][cb], v, nx[q > 0 ? q - 1 : 0][cb]);
                            if (cb + 1 < CB) nx[q][cb + 1 < CB ? cb + 1 : 0] = ofma(cem[q][cb + 1 < CB ? cb + 1 : 0], v, nx[q][cb + 1 < CB ? cb + 1 : 0]);
                            if (cb > 0) nx[q][cb > 0 ? cb - 1 : 0] = ofma(cep[q][cb > 0 ? cb - 1 : 0], v, nx[q][cb > 0 ? cb - 1 : 0]);
                        }
#pragma unroll
                    for (int cb = 0; cb < CB; ++cb) {
                        nx[0][cb] = ofma(cxm[0][cb], dn[cb], nx[0][cb]);
                        nx[QA - 1][cb] = ofma(cxp[QA - 1][cb], up[cb], nx[QA - 1][cb]);
                    }
#pragma unroll
                    for (int q = 0; q < QA; ++q) {
                        nx[q][0] = ofma(cem[q][0], lf[q], nx[q][0]);
                        nx[q][CB - 1] = ofma(cep[q][CB - 1], rt[q], nx[q][CB - 1]);
                    }
                    if (PM) {
#pragma unroll
                        for (int q = 0; q < QA; ++q)
#pragma unroll
                            for (int cb = 0; cb < CB; ++cb) nx[q][cb] = and_mask(nx[q][cb], maskw[q][cb]);
                    }
                } else {
#pragma unroll
                for (int q = 0; q < QA; ++q)
#pragma unroll
                    for (int cb = 0; cb < CB; ++cb) {
                        real acc = fma(c0j[q][cb], x[q][cb], (PM && !MF) ? dsrc : srcm[q][cb]);
                        if (q > 0) acc = fma(cxm[q][cb], x[q - 1][cb], acc);
                        if (q + 1 < QA) acc = fma(cxp[q][cb], x[q + 1][cb], acc);
                        if (cb > 0) acc = fma(cem[q][cb], x[q][cb - 1], acc);
                        if (cb + 1 < CB) acc = fma(cep[q][cb], x[q][cb + 1], acc);
                        if (q == 0) acc = fma(cxm[q][cb], dn[cb], acc);
                        if (q + 1 == QA) acc = fma(cxp[q][cb], up[cb], acc);
                        if (cb == 0) acc = fma(cem[q][cb], lf[q], acc);
                        if (cb + 1 == CB) acc = fma(cep[q][cb], rt[q], acc);
                        acc = fma(csm[q][cb], Rl[q][cb], acc);   // last: the result may reuse R's register
                        nx[q][cb] = PM ? and_mask(acc, maskw[q][cb]) : acc;
                    }
                }
                }
#pragma unroll
                for (int q = 0; q < QA; ++q) {
                    if (lv < TR) {
#pragma unroll
                        for (int cb = 0; cb < CB; ++cb) R[lv < TR ? lv : 0][q][cb] = x[q][cb];
                    } else {
#pragma unroll
                        for (int v4 = 0; v4 < CB / VW; ++v4) {
                            V128 t;
#pragma unroll
                            for (int e = 0; e < VW; ++e) t.v[e] = x[q][v4 * VW + e];
                            *reinterpret_cast<V128 *>(rsm_at(lv, q, v4)) = t;
                        }
                    }
#pragma unroll
                    for (int cb = 0; cb < CB; ++cb) x[q][cb] = nx[q][cb];
                }
            }
            // ---- store level T of plane j; S9 partial sums
            if (live) {
#pragma unroll
            for (int q = 0; q < QA; ++q)
#pragma unroll
                for (int v4 = 0; v4 < CB / VW; ++v4) {
                    V128 v;
#pragma unroll
                    for (int e = 0; e < VW; ++e) v.v[e] = x[q][v4 * VW + e];
                    *reinterpret_cast<V128 *>(oc + (int64_t)j * PLANE + (a0 + q) * NETA + b0 + v4 * VW) = v;
                }
            }
            if (MOM && live) {
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
        }
        };
        if constexpr (LOC) {
            static_assert(T == 4, "the LOC dispatch below lists the level counts 0..4");
            switch (nlev) {
            case 0: chunk(std::integral_constant<int, 0>{}); break;
            case 1: chunk(std::integral_constant<int, 1>{}); break;
            case 2: chunk(std::integral_constant<int, 2>{}); break;
            case 3: chunk(std::integral_constant<int, 3>{}); break;
            default: chunk(std::integral_constant<int, 4>{}); break;
            }
        } else {
            chunk(std::integral_constant<int, T>{});
        }
        // every lane has consumed this slot (its values fed the stores above): refill it
        __syncwarp();
        if (lane == 0 && i + D < total) issue();
        if (++slot == D) { slot = 0; phase ^= 1u; }

        if (++ch == CH) {
            if (MOM && (!LOC || last_pass)) {
                // S9: fp64 from the cross-lane reduction on (fp32 contexts: fp32 within a lane)
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
}

}  // namespace mm
