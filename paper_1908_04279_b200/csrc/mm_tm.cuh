// mm_tm.cuh -- the upwind-sparse kernel: fused advect + react (+ moments), any number of substeps per HBM pass, with the
// per-level carry of the s-upwind plane held in TENSOR MEMORY (sm_100a: tcgen05.alloc / tcgen05.st / tcgen05.ld).
//
// Same data movement and patch layout as mm_coef.cuh (one warp streams one configuration through its Ns offset planes;
// warp-private ring of shared-memory slots filled by 1-D TMA bulk copies on mbarriers; all levels applied to plane j as
// soon as it arrives; direct 128-bit stores) and the same compare-free coefficient form of S5-S7.  What differs, each
// point measured first with stand-alone probes (profiles/r02a_README.md):
//  * The carry between planes.  Level lv of plane j needs level lv of plane j-1 (the s-upwind value, S5).  mm_coef.cuh
//    keeps those T planes in registers (T x 8 per lane: the level loop must be unrolled, the kernel is ~9000
//    instructions and one instance per T) or in shared memory (2 x 128-bit accesses per row and level on the same
//    128 B/clk data path as the shuffles: MIO-bound).  Here the carry lives in the SM's tensor memory, which no other
//    part of this path uses: 256 KB per SM, lane-private rows (lane = TMEM lane, 8 or 16 columns per level),
//    addressable with a RUN-TIME column, 12-cycle loads, a data path of its own.  So the level loop is a real loop
//    (rolled by two so that the plane values ping-pong between two register sets without copies), one kernel serves
//    every fuse depth (the depth is an argument), the local-step variant needs no per-level-count instances, and 110
//    registers instead of 254 put 4 warps on a scheduler.
//  * What is carried is not the value m_{j-1} but its complete contribution P = (dt W/ds) m_{j-1} + dt src to the cell
//    downstream: it is produced where m_{j-1} is in registers anyway and lands in a FIXED place (the tensor-memory
//    columns of its level), so nothing rotates.
//  * Upwind sparsity.  A face has ONE donor cell (S5): of the two coefficients a face contributes (h+|h| to the cell
//    above, |h|-h to the cell below) one is an exact zero.  Where the face velocity has one sign over the whole plane
//    -- two planes in three for the BASELINE input distributions, per direction -- the 8 FMAs and the 4 (2) shuffles
//    of the dead direction are skipped: a warp vote per plane picks one of 9 straight-line variants of the level loop
//    (3 states per direction).  Skipping is exact: the skipped terms are products with +0.
// S9 moments, in-place passes, the local-step mode (NEXT-3) and the coupled source (NEXT-2) work as in mm_coef.cuh.
#pragma once
#include "mm_coef.cuh"

namespace mm {

// ---- tensor memory as lane-private scratch (tcgen05; SASS: UTCALLOC / LDTM / STTM) ---------------------------------
__device__ __forceinline__ void tm_alloc(uint32_t *smem_dst, uint32_t ncols)   // one full warp; ncols = 2^k >= 32
{
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(smem_dst)), "r"(ncols)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tm_dealloc(uint32_t taddr, uint32_t ncols)     // one full warp
{
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}
__device__ __forceinline__ void tm_fence_before_sync() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tm_fence_after_sync() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tm_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tm_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

// NW 32-bit columns of this thread's tensor-memory lane, starting at `ta` (shape 32x32b: thread i of the warp owns
// lane base+i); NW in {2, 4, 8, 16, 32, 64}
template <int NW>
__device__ __forceinline__ void tm_ldw(uint32_t ta, uint32_t (&r)[NW])
{
    static_assert(NW == 2 || NW == 4 || NW == 8 || NW == 16 || NW == 32 || NW == 64, "tcgen05.ld .x2 .. .x64");
    if constexpr (NW == 2)
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0,%1}, [%2];" : "=r"(r[0]), "=r"(r[1]) : "r"(ta));
    else if constexpr (NW == 4)
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0,%1,%2,%3}, [%4];"
                     : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(ta));
    else if constexpr (NW == 8)
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                     : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]) : "r"(ta));
    else if constexpr (NW == 16)
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                     : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
                       "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]) : "r"(ta));
    else {
        tm_ldw<NW / 2>(ta, reinterpret_cast<uint32_t(&)[NW / 2]>(r[0]));
        tm_ldw<NW / 2>(ta + NW / 2, reinterpret_cast<uint32_t(&)[NW / 2]>(r[NW / 2]));
    }
}
template <int NW>
__device__ __forceinline__ void tm_stw(uint32_t ta, const uint32_t (&r)[NW])
{
    static_assert(NW == 2 || NW == 4 || NW == 8 || NW == 16 || NW == 32 || NW == 64, "tcgen05.st .x2 .. .x64");
    if constexpr (NW == 2)
        asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1,%2};" ::"r"(ta), "r"(r[0]), "r"(r[1]) : "memory");
    else if constexpr (NW == 4)
        asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1,%2,%3,%4};" ::"r"(ta), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3])
                     : "memory");
    else if constexpr (NW == 8)
        asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"r"(ta), "r"(r[0]), "r"(r[1]),
                     "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]) : "memory");
    else if constexpr (NW == 16)
        asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};" ::"r"(ta),
                     "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]),
                     "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]) : "memory");
    else {
        tm_stw<NW / 2>(ta, reinterpret_cast<const uint32_t(&)[NW / 2]>(r[0]));
        tm_stw<NW / 2>(ta + NW / 2, reinterpret_cast<const uint32_t(&)[NW / 2]>(r[NW / 2]));
    }
}
// N reals <-> N * sizeof(real) / 4 columns
template <int N>
__device__ __forceinline__ void tm_ld(uint32_t ta, float (&v)[N])
{
    uint32_t r[N];
    tm_ldw<N>(ta, r);
#pragma unroll
    for (int i = 0; i < N; ++i) v[i] = __uint_as_float(r[i]);
}
template <int N>
__device__ __forceinline__ void tm_ld(uint32_t ta, double (&v)[N])
{
    uint32_t r[2 * N];
    tm_ldw<2 * N>(ta, r);
#pragma unroll
    for (int i = 0; i < N; ++i) v[i] = __hiloint2double((int)r[2 * i + 1], (int)r[2 * i]);
}
template <int N>
__device__ __forceinline__ void tm_st(uint32_t ta, const float (&v)[N])
{
    uint32_t r[N];
#pragma unroll
    for (int i = 0; i < N; ++i) r[i] = __float_as_uint(v[i]);
    tm_stw<N>(ta, r);
}
template <int N>
__device__ __forceinline__ void tm_st(uint32_t ta, const double (&v)[N])
{
    uint32_t r[2 * N];
#pragma unroll
    for (int i = 0; i < N; ++i) {
        r[2 * i] = (uint32_t)__double2loint(v[i]);
        r[2 * i + 1] = (uint32_t)__double2hiint(v[i]);
    }
    tm_stw<2 * N>(ta, r);
}
__device__ __forceinline__ uint32_t rbits_or(uint32_t o, float v) { return o | __float_as_uint(v); }
__device__ __forceinline__ uint32_t rbits_or(uint32_t o, double v) { return o | (uint32_t)__double2hiint(v) | (uint32_t)__double2loint(v); }

__host__ __device__ constexpr int tm_pow2_ge(int n) { int p = 1; while (p < n) p *= 2; return p; }

template <typename real, int NXI, int NETA, int CB, int P, int D, int WARPS, int MINB>
struct TmCfg {
    using Co = CoefCfg<real, NXI, NETA, CB, P, D, WARPS, false, 0>;
    static constexpr int QA = Co::QA, NC = Co::QA * CB;                      // cells per lane
    static constexpr int CPL = NC * (int)sizeof(real) / 4;                   // tensor-memory columns per level
    static constexpr int NK = Co::NK;                                         // per-configuration constants of a lane
    static constexpr int KCOLS = tm_pow2_ge(NK * (int)sizeof(real) / 4);      // ... columns they take (one .xN access)
    static constexpr int NKP = KCOLS * 4 / (int)sizeof(real);                 // ... padded count
    static constexpr int TC = MINB <= 1 ? 512 : (MINB == 2 ? 256 : (MINB <= 4 ? 128 : 64));   // columns per CTA (2^k)
    static constexpr int WCOLS = TC / ((WARPS + 3) / 4);                      // columns per warp (warps w, w+4 share lanes)
    static constexpr int TMAX = (WCOLS - KCOLS) / CPL;                        // levels a pass can fuse
    static_assert(WARPS % 4 == 0 && TMAX >= 1, "tensor-memory budget");
    static constexpr size_t SMEM_BYTES = Co::SMEM_BYTES + 16;                 // + the allocation's base address
};

// The coefficients of one plane for the cells of a lane (level-independent), and the per-cell source increment.
template <typename real, int QA, int CB>
struct TmCoef {
    real c0j[QA][CB], cxm[QA][CB], cxp[QA][CB], cem[QA][CB], cep[QA][CB], csm[QA][CB], src[QA][CB];
};

#ifndef MM_TM_XSTAT
#define MM_TM_XSTAT 1
#endif
// acc += a * b, kept in program order among its kind (volatile): see tm_level
__device__ __forceinline__ void fma_ord(float &acc, float a, float b) { asm volatile("fma.rn.f32 %0, %1, %2, %0;" : "+f"(acc) : "f"(a), "f"(b)); }
__device__ __forceinline__ void fma_ord(double &acc, double a, double b) { asm volatile("fma.rn.f64 %0, %1, %2, %0;" : "+d"(acc) : "d"(a), "d"(b)); }

// One level of one plane: xo = level lv+1 from xi = level lv and the carry P of level lv (tensor memory, at `ta`), and
// the new carry for the plane downstream.  SK: bit 0 = no cxm terms (all exactly 0 on this plane), 1 = no cxp, 2 = no
// cem, 3 = no cep.
template <int SK, bool XS, typename real, int QA, int CB, int LB>
__device__ __forceinline__ void tm_level(const TmCoef<real, QA, CB> &k, const real (&xi)[QA][CB], real (&xo)[QA][CB], uint32_t ta)
{
    real Pl[QA * CB];
    tm_ld<QA * CB>(ta, Pl);
    real up[CB], dn[CB], lf[QA], rt[QA];
#pragma unroll
    for (int cb = 0; cb < CB; ++cb) {
        if (!(SK & 2)) up[cb] = shfl_down_r(xi[0][cb], LB);
        if (!(SK & 1)) dn[cb] = shfl_up_r(xi[QA - 1][cb], LB);
    }
#pragma unroll
    for (int q = 0; q < QA; ++q) {
        if (!(SK & 8)) rt[q] = shfl_down_r(xi[q][0], 1);
        if (!(SK & 4)) lf[q] = shfl_up_r(xi[q][CB - 1], 1);
    }
    tm_wait_ld();
#if MM_TM_XSTAT
    // taken by the fp64 kernels and the coupled-source fp32 kernels (XS): measured on one box, fp32 plain 2403 G/s
    // without / 2396 with, coupled whole step 1593 / 1611, fp64 plain 1230 / 1265
    if constexpr (sizeof(real) == 8 || XS) {
        // x-stationary, in program order: the (up to) six FMAs that read one xi are adjacent, so that the operand is
        // read once from the register file (.reuse): an FMA pays for its fresh register operands, two per cycle --
        // 1.5 cycles with three, 1 with two (profiles/r02a_README.md).  xo starts as the carry and each product is
        // added exactly once; inside a run the order is chosen so that an accumulator written by three consecutive
        // runs (from the left cell, by the cell itself, from the right cell) is touched at positions 1, 4 and 6: no
        // two writes of one accumulator are closer than 8 instructions, and the scheduler has no reason to break a run.
#pragma unroll
        for (int q = 0; q < QA; ++q)
#pragma unroll
            for (int cb = 0; cb < CB; ++cb) xo[q][cb] = Pl[q * CB + cb];
        real Pn[QA * CB];
#pragma unroll
        for (int q = 0; q < QA; ++q)
#pragma unroll
            for (int cb = 0; cb < CB; ++cb) {
                const real xv = xi[q][cb];
                constexpr int Z = 0;
                if (!(SK & 4) && cb + 1 < CB) fma_ord(xo[q][cb + 1 < CB ? cb + 1 : Z], k.cem[q][cb + 1 < CB ? cb + 1 : Z], xv);
                Pn[q * CB + cb] = k.src[q][cb];
                fma_ord(Pn[q * CB + cb], k.csm[q][cb], xv);
                if (!(SK & 1) && q + 1 < QA) fma_ord(xo[q + 1 < QA ? q + 1 : Z][cb], k.cxm[q + 1 < QA ? q + 1 : Z][cb], xv);
                fma_ord(xo[q][cb], k.c0j[q][cb], xv);
                if (!(SK & 2) && q > 0) fma_ord(xo[q > 0 ? q - 1 : Z][cb], k.cxp[q > 0 ? q - 1 : Z][cb], xv);
                if (!(SK & 8) && cb > 0) fma_ord(xo[q][cb > 0 ? cb - 1 : Z], k.cep[q][cb > 0 ? cb - 1 : Z], xv);
            }
        tm_st<QA * CB>(ta, Pn);
#pragma unroll
        for (int cb = 0; cb < CB; ++cb) {
            if (!(SK & 1)) fma_ord(xo[0][cb], k.cxm[0][cb], dn[cb]);
            if (!(SK & 2)) fma_ord(xo[QA - 1][cb], k.cxp[QA - 1][cb], up[cb]);
        }
#pragma unroll
        for (int q = 0; q < QA; ++q) {
            if (!(SK & 4)) fma_ord(xo[q][0], k.cem[q][0], lf[q]);
            if (!(SK & 8)) fma_ord(xo[q][CB - 1], k.cep[q][CB - 1], rt[q]);
        }
        return;
    }
#endif
    // the old carry is consumed at once (its registers die before the new one is staged for the store)
#pragma unroll
    for (int q = 0; q < QA; ++q)
#pragma unroll
        for (int cb = 0; cb < CB; ++cb) xo[q][cb] = fma(k.c0j[q][cb], xi[q][cb], Pl[q * CB + cb]);
    {
        real Pn[QA * CB];
#pragma unroll
        for (int q = 0; q < QA; ++q)
#pragma unroll
            for (int cb = 0; cb < CB; ++cb) Pn[q * CB + cb] = fma(k.csm[q][cb], xi[q][cb], k.src[q][cb]);
        tm_st<QA * CB>(ta, Pn);
    }
#pragma unroll
    for (int q = 0; q < QA; ++q)
#pragma unroll
        for (int cb = 0; cb < CB; ++cb) {
            real acc = xo[q][cb];
            if (!(SK & 1) && q > 0) acc = fma(k.cxm[q][cb], xi[q > 0 ? q - 1 : 0][cb], acc);
            if (!(SK & 2) && q + 1 < QA) acc = fma(k.cxp[q][cb], xi[q + 1 < QA ? q + 1 : 0][cb], acc);
            if (!(SK & 4) && cb > 0) acc = fma(k.cem[q][cb], xi[q][cb > 0 ? cb - 1 : 0], acc);
            if (!(SK & 8) && cb + 1 < CB) acc = fma(k.cep[q][cb], xi[q][cb + 1 < CB ? cb + 1 : 0], acc);
            if (!(SK & 1) && q == 0) acc = fma(k.cxm[q][cb], dn[cb], acc);
            if (!(SK & 2) && q + 1 == QA) acc = fma(k.cxp[q][cb], up[cb], acc);
            if (!(SK & 4) && cb == 0) acc = fma(k.cem[q][cb], lf[q], acc);
            if (!(SK & 8) && cb + 1 == CB) acc = fma(k.cep[q][cb], rt[q], acc);
            xo[q][cb] = acc;
        }
}

// All `nlev` levels of one plane, in place in x.  The loop is rolled by two: the plane values alternate between x and
// y, so no register copies are needed (an odd count ends with one copy per plane).  Rolled by four it runs at less than
// half the speed: 9 variants x 7 level bodies no longer fit the instruction cache (profiles/r02a_README.md).
// COMPACT (the coupled-source kernels, whose per-plane code is longer): an odd count leaves the loop after its first
// half instead of running a third copy of the level body -- 7 KB less hot code, which keeps the plane loop under the
// instruction-cache cliff; the plain kernels lose 2 % to the extra branch per pair of levels and keep the tail copy.
template <int SK, bool COMPACT, typename real, int QA, int CB, int LB, int CPL>
__device__ __forceinline__ void tm_plane(const TmCoef<real, QA, CB> &k, real (&x)[QA][CB], uint32_t tbase, int nlev)
{
    real y[QA][CB];
    bool odd = false;
    if constexpr (COMPACT) {
#pragma unroll 1
        for (int lv = 0; lv < nlev; lv += 2) {
            tm_level<SK, COMPACT, real, QA, CB, LB>(k, x, y, tbase + lv * CPL);
            if (lv + 1 == nlev) { odd = true; break; }
            tm_level<SK, COMPACT, real, QA, CB, LB>(k, y, x, tbase + lv * CPL + CPL);
        }
    } else {
        int lv = 0;
#pragma unroll 1
        for (; lv + 2 <= nlev; lv += 2) {
            tm_level<SK, COMPACT, real, QA, CB, LB>(k, x, y, tbase + lv * CPL);
            tm_level<SK, COMPACT, real, QA, CB, LB>(k, y, x, tbase + lv * CPL + CPL);
        }
        if (lv < nlev) {
            tm_level<SK, COMPACT, real, QA, CB, LB>(k, x, y, tbase + lv * CPL);
            odd = true;
        }
    }
    if (odd) {
#pragma unroll
        for (int q = 0; q < QA; ++q)
#pragma unroll
            for (int cb = 0; cb < CB; ++cb) x[q][cb] = y[q][cb];
    }
}

// nlev: substeps this pass fuses (<= TmCfg::TMAX); mom: also reduce the S9 moments.  Local-step mode (LOC):
// configuration c takes clamp(n_steps[c] - done, 0, nlev) steps of its own size dt_c[c]; `kp` then carries the factors
// per unit dt; `list` as in mm_coef.cuh.
template <typename real, int NXI, int NETA, int CB, int P, int D, int WARPS, int MINB, bool MF, bool LOC, bool PF = false>
__global__ void __launch_bounds__(WARPS * 32, MINB)
    substep_tm_kernel(const __grid_constant__ KParams<real> kp, const real *__restrict__ in, real *__restrict__ out,
                      double *__restrict__ force, double *__restrict__ torque, int nlev_pass, int mom,
                      const int32_t *__restrict__ n_steps, const real *__restrict__ dt_c, int32_t done,
                      const int32_t *__restrict__ list, const int32_t *__restrict__ list_count,
                      double *__restrict__ fline)
{
    using Cfg = TmCfg<real, NXI, NETA, CB, P, D, WARPS, MINB>;
    using Co = typename Cfg::Co;
    constexpr int LB = Co::LB, G = Co::G, QA = Co::QA, PLANE = Co::PLANE, NK = Co::NK, VW = Co::VW;
    constexpr int CPL = Cfg::CPL, NKP = Cfg::NKP;
    using V128 = CVec<real, VW>;
    constexpr int OX = 0, OE = (QA + 1) * CB, OC = OE + QA * (CB + 1);   // offsets of h0x, h0e, c0m among the constants

    extern __shared__ __align__(128) unsigned char smem_raw[];
    real *kap_s = reinterpret_cast<real *>(smem_raw);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    real *ring = reinterpret_cast<real *>(smem_raw + Co::TABLE_BYTES + (size_t)warp * Co::WARP_BYTES);
    uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw + Co::TABLE_BYTES + (size_t)WARPS * Co::WARP_BYTES) + warp * D;
    uint32_t *tm_slot = reinterpret_cast<uint32_t *>(smem_raw + Co::SMEM_BYTES);

    for (int i = threadIdx.x; i < PLANE; i += WARPS * 32) kap_s[i] = kp.kappa[i];
    if (lane == 0) {
#pragma unroll
        for (int d = 0; d < D; ++d) mbar_init(&full[d], 1);
        mbar_fence_init();
    }
    if (warp == 0) tm_alloc(tm_slot, Cfg::TC);
    tm_fence_before_sync();
    __syncthreads();
    tm_fence_after_sync();
    const uint32_t tm_cta = *tm_slot;
    // this warp's block: its lane quarter (a warp reaches only lanes 32 (warp % 4) .. +31), its share of the columns;
    // first the per-configuration constants, then the carries of levels 0, 1, ...
    const uint32_t tm_k = tm_cta + ((uint32_t)((warp & 3) * 32) << 16) + (uint32_t)((warp >> 2) * Cfg::WCOLS);
    const uint32_t tm_p = tm_k + Cfg::KCOLS;

    // ---- lane's patch and configuration-independent constants
    const int g = lane / LB, lb = lane - g * LB;
    const int a0 = g * QA, b0 = lb * CB;
    const bool is_g0 = (g == 0), is_gtop = (g == G - 1), is_l0 = (lb == 0), is_lr = (lb == LB - 1);
    constexpr bool loc = LOC;   // compile time: in the global mode the level count stays a kernel argument (uniform)
    real maskf[QA][CB], xiq[QA], etab[CB];
#pragma unroll
    for (int q = 0; q < QA; ++q) {
        xiq[q] = -kp.R + (real(a0 + q) + real(0.5)) * kp.dxi;
#pragma unroll
        for (int cb = 0; cb < CB; ++cb) maskf[q][cb] = kp.inside[(a0 + q) * NETA + b0 + cb] ? real(1) : real(0);
    }
#pragma unroll
    for (int cb = 0; cb < CB; ++cb) etab[cb] = -kp.R + (real(b0 + cb) + real(0.5)) * kp.deta;
    unsigned short *nod = reinterpret_cast<unsigned short *>(smem_raw + ((Cfg::SMEM_BYTES + 15) / 16) * 16) +
                          (size_t)warp * kp.ns * (NXI + NETA);   // MF: this warp's node tables (host adds the bytes)

    const int ns = kp.ns;
    const int64_t inner = (int64_t)ns * PLANE;
    const int CH = (ns + P - 1) / P;
    const int64_t gw = (int64_t)blockIdx.x * WARPS + warp, nw = (int64_t)gridDim.x * WARPS;
    const int64_t nact = (loc && list) ? (int64_t)*list_count : kp.nc;   // configurations this pass visits
    const int64_t my_n = gw < nact ? (nact - gw + nw - 1) / nw : 0;
    const int64_t total = my_n * CH;

    int64_t pk = 0;   // producer state (lane 0): next chunk to request
    int pch = 0, pslot = 0;
    auto issue = [&]() {   // lane 0 only: TMA bulk copy of the next stream chunk into its ring slot
        const int64_t c = (loc && list) ? (int64_t)list[gw + pk * nw] : gw + pk * nw;
        const int planes = min(P, ns - pch * P);
        const uint32_t bytes = (uint32_t)(planes * PLANE * sizeof(real));
        mbar_expect_tx(&full[pslot], bytes);
        tma_load_1d(ring + (size_t)pslot * P * PLANE, in + c * inner + (int64_t)pch * P * PLANE, bytes, &full[pslot]);
        if (++pslot == D) pslot = 0;
        if (++pch == CH) { pch = 0; ++pk; }
    };
    if (lane == 0)
        for (int64_t i = 0; i < total && i < D; ++i) issue();

    TmCoef<real, QA, CB> co;
    real hbx = 0, hbe = 0, ct = 0, st = 0, dtc = real(1);
    int nlev = nlev_pass;
    bool last_pass = true;
    real FX = 0, FY = 0, TQ = 0;

    // MF: co.src of s-plane jj = mask dt k_on M_f(node of the cell's anchor), through this warp's node tables
    auto gather = [&](int jj) {
        const unsigned short *nj = nod + jj * (NXI + NETA);
        int nodx[QA], nody[CB];
#pragma unroll
        for (int q = 0; q < QA; ++q) nodx[q] = (int)nj[a0 + q] * kp.ny;
#pragma unroll
        for (int cb = 0; cb < CB; ++cb) nody[cb] = (int)nj[NXI + b0 + cb];
#pragma unroll
        for (int q = 0; q < QA; ++q)
#pragma unroll
            for (int cb = 0; cb < CB; ++cb)
                co.src[q][cb] = maskf[q][cb] * (kp.dt_kon * dtc * __ldg(&kp.Mf_r[nodx[q] + nody[cb]]));
    };

    int64_t k = 0, c = 0;
    int ch = 0, slot = 0;
    uint32_t phase = 0;
    real *optr = out;   // this lane's first cell of the plane being stored
    for (int64_t i = 0; i < total; ++i) {
        if (ch == 0) {
            // ---- per configuration (S2-S4, S6 folded; everything that does not depend on s)
            c = (loc && list) ? (int64_t)list[gw + k * nw] : gw + k * nw;
            optr = out + c * inner + a0 * NETA + b0;
            const int kth = (int)(c % kp.ntheta);
            ct = kp.cos_t[kth];
            st = kp.sin_t[kth];
            const real U = kp.U[c], Vv = kp.V[c], Om = kp.Om[c];
            if (MF) {
                const int iy = (int)((c / kp.ntheta) % kp.ny), ix = (int)(c / ((int64_t)kp.ntheta * kp.ny));
                __syncwarp();   // the previous configuration's planes are done with the tables
                if (kp.node_x) {
                    // the context's tables: rows (ix, itheta) and (iy, itheta), ns x NXI and ns x NETA entries, copied 8
                    // entries at a time into the interleaved per-warp table
                    constexpr int VX = NXI / 8, VY = NETA / 8;
                    static_assert(NXI % 8 == 0 && NETA % 8 == 0, "vector copy of the node tables");
                    const uint4 *sx = reinterpret_cast<const uint4 *>(kp.node_x + ((int64_t)ix * kp.ntheta + kth) * kp.ns * NXI);
                    const uint4 *sy = reinterpret_cast<const uint4 *>(kp.node_y + ((int64_t)iy * kp.ntheta + kth) * kp.ns * NETA);
                    for (int e = lane; e < kp.ns * VX; e += 32) {
                        const int jj = e / VX, part = e - jj * VX;
                        *reinterpret_cast<uint4 *>(nod + jj * (NXI + NETA) + part * 8) = __ldg(sx + e);
                    }
                    for (int e = lane; e < kp.ns * VY; e += 32) {
                        const int jj = e / VY, part = e - jj * VY;
                        *reinterpret_cast<uint4 *>(nod + jj * (NXI + NETA) + NXI + part * 8) = __ldg(sy + e);
                    }
                } else {
                const double theta = 2.0 * 3.14159265358979323846264338327950288 * (double)kth / (double)kp.ntheta;
                const double mf_ct = cos(theta), mf_st = sin(theta);
                const double mf_tx = __ddiv_rn((double)ix, (double)kp.nx), mf_ty = __ddiv_rn((double)iy, (double)kp.ny);
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
                }
                __syncwarp();
            }
            if (loc) {
                dtc = dt_c[c];
                const int owed = n_steps[c] - done;
                nlev = owed < 0 ? 0 : (owed > nlev_pass ? nlev_pass : owed);
                last_pass = owed <= nlev_pass;
            }
            const real hdx = real(0.5) * kp.dt_dxi * dtc, hde = real(0.5) * kp.dt_deta * dtc;
            const real dsrc = kp.dt_src * dtc;
            hbx = -hdx * Om * st;   // d/ds_j of h_xi   (S4: A_xi = U + w cos - s Omega sin)
            hbe = hde * Om * ct;    // d/ds_j of h_eta  (S4: A_eta = V + w sin + s Omega cos)
            // kc[OX + fq*CB + cb]     = h0x: (dt/2dxi)  A_xi  at s = 0 on the xi faces below rows a0 .. a0+QA       (S4)
            // kc[OE + q*(CB+1) + fb]  = h0e: (dt/2deta) A_eta at s = 0 on the eta faces left of columns b0 .. b0+CB
            // kc[OC + q*CB + cb]      = c0m: mask (1 - dt W/ds - dt kappa - [h_t - h_b] - [h_r - h_l])
            real kc[NKP];
#pragma unroll
            for (int e = NK; e < NKP; ++e) kc[e] = real(0);
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
                    const real cs = kp.dt_ds * dtc * walk_speed(kp.v0, kp.kload, ct, st, xiq[q], etab[cb]);
                    const real lin = (kc[OX + (q + 1) * CB + cb] - kc[OX + q * CB + cb]) +
                                     (kc[OE + q * (CB + 1) + cb + 1] - kc[OE + q * (CB + 1) + cb]);
                    const real c0 = real(1) - cs - kp.dt * dtc * kap_s[(a0 + q) * NETA + b0 + cb] - lin;
                    co.csm[q][cb] = maskf[q][cb] * cs;
                    co.src[q][cb] = maskf[q][cb] * dsrc;
                    kc[OC + q * CB + cb] = maskf[q][cb] * c0;
                }
            }
            tm_wait_st();   // the previous configuration's last carries have landed
            tm_st<NKP>(tm_k, kc);
            {
                // zero inflow at s_lo (S5): the carry into plane 0 is the source alone (MF: its own, gathered), at every level
                if constexpr (MF) gather(0);
                real p0[QA * CB];
#pragma unroll
                for (int q = 0; q < QA; ++q)
#pragma unroll
                    for (int cb = 0; cb < CB; ++cb) p0[q * CB + cb] = co.src[q][cb];
                for (int lv = 0; lv < nlev; ++lv) tm_st<QA * CB>(tm_p + lv * CPL, p0);
            }
            FX = FY = TQ = real(0);
        }

        mbar_wait(&full[slot], phase);
        const real *sp = ring + (size_t)slot * P * PLANE + a0 * NETA + b0;   // this lane's first cell; advanced plane by plane
#pragma unroll 1
        for (int pl = 0; pl < P; ++pl) {
            const int j = ch * P + pl;
            if (j >= ns) break;   // ragged last chunk
            const real sj = kp.s_lo + (real(j) + real(0.5)) * kp.ds;
            // MF: the carry a plane sends downstream holds the source of the RECEIVING cell: while plane j is worked on,
            // co.src is the (gathered) source of plane j+1 (plane 0 received its own with the zero-inflow carry above)
            if constexpr (MF) gather(j + 1 < ns ? j + 1 : j);
            // ---- level-independent coefficients of this plane
            uint32_t zxm = 0, zxp = 0, zem = 0, zep = 0;   // OR of the bit patterns: 0 <=> the whole set is +0
            {
                real kl[NKP];
                tm_wait_st();   // kc, the plane-0 carries, the previous plane's carries
                tm_ld<NKP>(tm_k, kl);
                tm_wait_ld();
                real hx[QA + 1][CB], he[QA][CB + 1];
#pragma unroll
                for (int fq = 0; fq <= QA; ++fq)
#pragma unroll
                    for (int cb = 0; cb < CB; ++cb) hx[fq][cb] = fma(sj, hbx, kl[OX + fq * CB + cb]);
#pragma unroll
                for (int q = 0; q < QA; ++q)
#pragma unroll
                    for (int fb = 0; fb <= CB; ++fb) he[q][fb] = fma(sj, hbe, kl[OE + q * (CB + 1) + fb]);
                const bool endj = (j < kp.n_end) || (j >= ns - kp.n_end);   // enhanced end detachment (S6)
                const real endx = endj ? kp.dt_endx * dtc : real(0);
#pragma unroll
                for (int q = 0; q < QA; ++q)
#pragma unroll
                    for (int cb = 0; cb < CB; ++cb) {
                        const real sabs = (rabs(hx[q][cb]) + rabs(hx[q + 1][cb])) + (rabs(he[q][cb]) + rabs(he[q][cb + 1]));
                        const real pb = hx[q][cb] + rabs(hx[q][cb]);               // max(A,0) on the face below
                        const real nt = rabs(hx[q + 1][cb]) - hx[q + 1][cb];       // -min(A,0) on the face above
                        const real pl_ = he[q][cb] + rabs(he[q][cb]);
                        const real nr = rabs(he[q][cb + 1]) - he[q][cb + 1];
                        const real m = maskf[q][cb];
                        if constexpr (sizeof(real) == 4) co.c0j[q][cb] = fma(-m, sabs, kl[OC + q * CB + cb]);   // end planes: below
                        else co.c0j[q][cb] = fma(-m, fma(endx, kap_s[(a0 + q) * NETA + b0 + cb], sabs), kl[OC + q * CB + cb]);
                        co.cxm[q][cb] = m * pb; co.cxp[q][cb] = m * nt; co.cem[q][cb] = m * pl_; co.cep[q][cb] = m * nr;
                    }
                // enhanced end detachment (S6), fp32: on the n_end planes at either end only (uniform branch; the other planes
                // skip the loads of kappa and eight FMAs: configs[4] 2514 -> 2541 G/s; the fp64 kernel lost 2 % to the branch)
                if (sizeof(real) == 4 && endj) {
#pragma unroll
                    for (int q = 0; q < QA; ++q)
#pragma unroll
                        for (int cb = 0; cb < CB; ++cb)
                            co.c0j[q][cb] = fma(-maskf[q][cb] * endx, kap_s[(a0 + q) * NETA + b0 + cb], co.c0j[q][cb]);
                }
                // ghost cells beyond the box are 0 (S5): their coefficient is an exact 0 on the edge lanes
#pragma unroll
                for (int cb = 0; cb < CB; ++cb) {
                    co.cxm[0][cb] = is_g0 ? real(0) : co.cxm[0][cb];
                    co.cxp[QA - 1][cb] = is_gtop ? real(0) : co.cxp[QA - 1][cb];
                }
#pragma unroll
                for (int q = 0; q < QA; ++q) {
                    co.cem[q][0] = is_l0 ? real(0) : co.cem[q][0];
                    co.cep[q][CB - 1] = is_lr ? real(0) : co.cep[q][CB - 1];
                }
#pragma unroll
                for (int q = 0; q < QA; ++q)
#pragma unroll
                    for (int cb = 0; cb < CB; ++cb) {
                        zxm = rbits_or(zxm, co.cxm[q][cb]); zxp = rbits_or(zxp, co.cxp[q][cb]);
                        zem = rbits_or(zem, co.cem[q][cb]); zep = rbits_or(zep, co.cep[q][cb]);
                    }
            }
            real x[QA][CB];
#pragma unroll
            for (int q = 0; q < QA; ++q)
#pragma unroll
                for (int v4 = 0; v4 < CB / VW; ++v4) {
                    const V128 v = *reinterpret_cast<const V128 *>(sp + q * NETA + v4 * VW);
#pragma unroll
                    for (int e = 0; e < VW; ++e) x[q][v4 * VW + e] = v.v[e];
                }
            // ---- the levels: one of 9 straight-line variants, by which coefficient sets vanish on this plane
            {
                const int vx = __all_sync(0xffffffffu, zxm == 0) ? 1 : (__all_sync(0xffffffffu, zxp == 0) ? 2 : 0);
                const int ve = __all_sync(0xffffffffu, zem == 0) ? 1 : (__all_sync(0xffffffffu, zep == 0) ? 2 : 0);
#define MM_TM_VARIANT(SK_) tm_plane<SK_, MF, real, QA, CB, LB, CPL>(co, x, tm_p, nlev)
                switch (vx * 3 + ve) {
                case 0: MM_TM_VARIANT(0); break;
                case 1: MM_TM_VARIANT(4); break;
                case 2: MM_TM_VARIANT(8); break;
                case 3: MM_TM_VARIANT(1); break;
                case 4: MM_TM_VARIANT(5); break;
                case 5: MM_TM_VARIANT(9); break;
                case 6: MM_TM_VARIANT(2); break;
                case 7: MM_TM_VARIANT(6); break;
                default: MM_TM_VARIANT(10); break;
                }
#undef MM_TM_VARIANT
            }
            // ---- store the last level of plane j; S9 partial sums
#pragma unroll
            for (int q = 0; q < QA; ++q)
#pragma unroll
                for (int v4 = 0; v4 < CB / VW; ++v4) {
                    V128 v;
#pragma unroll
                    for (int e = 0; e < VW; ++e) v.v[e] = x[q][v4 * VW + e];
                    *reinterpret_cast<V128 *>(optr + q * NETA + v4 * VW) = v;
                }
            sp += PLANE;
            optr += PLANE;   // carried from plane to plane: the 64-bit address is not rebuilt (15 instructions) every plane
            if (mom) {
                // sum_ab xi_a m and sum_ab eta_b m over the lane's patch, with xi_a = xi_a0 + q dxi, eta_b = eta_b0 + cb
                // deta: S = sum m, fxp = xi_a0 S + dxi sum_q q rs_q, fyp = eta_b0 S + deta sum_cb cb cs_cb -- two
                // per-lane coordinates instead of QA + CB (which the compiler rematerialised on every plane)
                real rs[QA], cs[CB];
#pragma unroll
                for (int q = 0; q < QA; ++q) {
                    rs[q] = x[q][0];
#pragma unroll
                    for (int cb = 1; cb < CB; ++cb) rs[q] += x[q][cb];
                }
#pragma unroll
                for (int cb = 0; cb < CB; ++cb) {
                    cs[cb] = x[0][cb];
#pragma unroll
                    for (int q = 1; q < QA; ++q) cs[cb] += x[q][cb];
                }
                real S = rs[0], wq = real(0), wc = real(0);
#pragma unroll
                for (int q = 1; q < QA; ++q) { S += rs[q]; wq = fma(real(q), rs[q], wq); }
#pragma unroll
                for (int cb = 1; cb < CB; ++cb) wc = fma(real(cb), cs[cb], wc);
                const real fxp = fma(kp.dxi, wq, xiq[0] * S), fyp = fma(kp.deta, wc, etab[0] * S);
                FX += fxp;
                FY += fyp;
                TQ = fma(sj, ct * fyp - st * fxp, TQ);
                if (PF && last_pass) {   // PF: compiled only into the instances launched with a plane-force buffer
                    // NEXT-4: the spring force carried by this plane, f_j(c) = -k dxi deta sum_ab (xi_a, eta_b) m, is the
                    // pair of sums just formed: reduce both across the warp in one butterfly (lanes 0-15 gather the xi
                    // sum, lanes 16-31 the eta sum) and store them for mm_spread_force -- no separate read of the density
                    real a = (lane & 16) ? fyp : fxp;
                    const real b = (lane & 16) ? fxp : fyp;
                    a += __shfl_xor_sync(0xffffffffu, b, 16);
#pragma unroll
                    for (int o = 8; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
                    if ((lane & 15) == 0) fline[(c * ns + j) * 2 + (lane >> 4)] = kp.pf_scale * (double)a;   // a kernel parameter: no register held
                }
            }
        }
        // every lane has consumed this slot (its values fed the stores above): refill it
        __syncwarp();
        if (lane == 0 && i + D < total) issue();
        if (++slot == D) { slot = 0; phase ^= 1u; }

        if (++ch == CH) {
            if (mom && last_pass) {
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
    tm_wait_st();
    tm_fence_before_sync();
    __syncthreads();
    if (warp == 0) tm_dealloc(tm_cta, Cfg::TC);
}

}  // namespace mm
