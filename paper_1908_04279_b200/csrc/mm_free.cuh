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
    const unsigned short *tabx, *taby;   // NULL, or the context's anchor-node tables (node_table_kernel)
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
// PRIV (MODE 0): every CTA deposits into its OWN copy of the (x, y) table in shared memory (nx ny doubles, dynamic) with
// shared-memory atomics and adds it to the global table once at the end: the 8.6 G deposits of configs[4] then contend
// inside an SM only, and the global table sees nx ny atomics per CTA instead of one per cell (profiles/r02b_README.md).
template <typename real, int MODE, bool PRIV = false>
__global__ void __launch_bounds__(PRIV ? 1024 : 256) free_cells_kernel(const FreeGeom q, int64_t nc, real *__restrict__ dens,
                                                         const double *__restrict__ psi, double w, double *__restrict__ raw,
                                                         const double *__restrict__ factor, const int *__restrict__ any_capped,
                                                         unsigned long long * /*raw_fx: vector kernels only*/ = nullptr,
                                                         double /*inv_unit*/ = 1.0)
{
    if (MODE == 1 && *any_capped == 0) return;
    extern __shared__ double free_tab[];
    double *tab = raw;
    if (PRIV) {
        for (int i = threadIdx.x; i < q.nx * q.ny; i += blockDim.x) free_tab[i] = 0.0;
        __syncthreads();
        tab = free_tab;
    }
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
                    if (val != 0.0 && wp != 0.0) atomicAdd(&tab[n], wp * val);
                } else {
                    const double f = factor[n];
                    if (f != 1.0) *v = (real)((double)*v * f);
                }
            }
        }
    }
    if (PRIV) {
        __syncthreads();
        for (int i = threadIdx.x; i < q.nx * q.ny; i += blockDim.x)
            if (free_tab[i] != 0.0) atomicAdd(&raw[i], free_tab[i]);
    }
}

// Exact accumulation in shared memory.  Shared-memory atomics are native for 32-bit integers only (fp64 and 64-bit
// integer adds compile to compare-and-swap loops), so a private table holds every node as a 96-bit two's-complement
// fixed-point number in three 32-bit limbs, value = (L2:L1 2^-32 + L0 2^-64) * unit with unit = the power of two >=
// M_total: a deposit is 2 (rarely 3) native ATOMS.ADD, each returning the old limb so that exactly the add that wraps a
// limb carries into the next.  Integer adds commute: the table does not depend on the order of the deposits; its
// resolution (2^-64 unit per deposit, truncated) is far below the fp64 rounding of a node sum; range |sum| < 2^31 unit.
__device__ __forceinline__ void fx_deposit(uint32_t *L0, uint32_t *L1, uint32_t *L2, int n, double q /* value / unit */)
{
    const double t = q * 4294967296.0;                            // exact
    const long long i1 = __double2ll_rd(t);                       // floor: bits 2^-32 and up
    const uint32_t x0 = __double2uint_rd((t - (double)i1) * 4294967296.0);   // the next 32 bits, truncated
    const uint32_t x1 = (uint32_t)i1, x2 = (uint32_t)(i1 >> 32);
    const uint32_t o0 = atomicAdd(&L0[n], x0);
    const uint32_t t1 = x1 + ((o0 + x0 < o0) ? 1u : 0u);
    uint32_t c1 = (t1 < x1) ? 1u : 0u;                            // x1 = 2^32 - 1 with a carry in: carry out, nothing to add
    if (t1) { const uint32_t o1 = atomicAdd(&L1[n], t1); c1 |= (o1 + t1 < o1) ? 1u : 0u; }
    if (x2 | c1) atomicAdd(&L2[n], x2 + c1);
}

// the same out of line: the rare route of the vector kernel (a deposit of 2^19 units or more)
__device__ __noinline__ void fx_deposit_rare(uint32_t *L0, uint32_t *L1, uint32_t *L2, int n, double q)
{
    fx_deposit(L0, L1, L2, n, q);
}

// The anchor-node tables of a context for the coupled substep kernel (mm_tm.cuh): the x node depends on (ix, itheta, j,
// a) only, the y node on (iy, itheta, j, b), and the geometry never changes, so the fp64 evaluation (1600 instructions
// per lane and configuration in that kernel) is done once: tabx[((ix ntheta + itheta) ns + j) nxi + a],
// taby[((iy ntheta + itheta) ns + j) neta + b].  Same expression, operation by operation, as the inline evaluation
// (ties break alike).  The fp32 deposit pass below reads them too, one 16-bit load per lane and plane issued with the
// density loads (a look-up at the point of use, a dependent load in front of the atomics, measured 10.9 -> 12.2 ms on
// configs[4]; prefetched 9.7 ms).
__global__ void __launch_bounds__(256) node_table_kernel(const FreeGeom q, unsigned short *__restrict__ tabx, unsigned short *__restrict__ taby)
{
    const int64_t nxe = (int64_t)q.nx * q.ntheta * q.ns * q.nxi, nye = (int64_t)q.ny * q.ntheta * q.ns * q.neta;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < nxe + nye; e += (int64_t)gridDim.x * blockDim.x) {
        const bool isx = e < nxe;
        const int64_t i = isx ? e : e - nxe;
        const int no = isx ? q.nxi : q.neta, n = isx ? q.nx : q.ny;
        const int k = (int)(i % no);
        const int j = (int)((i / no) % q.ns);
        const int itheta = (int)((i / ((int64_t)no * q.ns)) % q.ntheta);
        const int row = (int)(i / ((int64_t)no * q.ns * q.ntheta));
        const double theta = 2.0 * 3.14159265358979323846264338327950288 * (double)itheta / (double)q.ntheta;
        const double cs = isx ? cos(theta) : sin(theta);
        const double base = __ddiv_rn((double)row, (double)n);
        const double off = __dadd_rn(-q.R, __dmul_rn(k + 0.5, isx ? q.dxi : q.deta));
        const double sj = __dadd_rn(q.s_lo, __dmul_rn(j + 0.5, q.ds));
        const double r = __dmul_rn(__dsub_rn(__dadd_rn(base, __dmul_rn(sj, cs)), off), (double)n);
        (isx ? tabx : taby)[i] = (unsigned short)wrap_floor(__dadd_rn(r, 0.5), n);
    }
}

// old = L[addr]; L[addr] += x -- skipped (old = 0) when x == 0; a predicated ATOMS, no branch around it
__device__ __forceinline__ uint32_t atoms_add_nz(uint32_t saddr, uint32_t x)
{
    uint32_t o;
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %2, 0;\n\tmov.u32 %0, 0;\n\t@p atom.shared.add.u32 %0, [%1], %2;\n\t}"
                 : "=r"(o) : "r"(saddr), "r"(x) : "memory");
    return o;
}
__device__ __forceinline__ void reds_add_nz(uint32_t saddr, uint32_t x)
{
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %1, 0;\n\t@p red.shared.add.u32 [%0], %1;\n\t}" :: "r"(saddr), "r"(x) : "memory");
}

// The same two passes for the BASELINE offset planes (16x16, 8x8; a plane tiles a warp with VW cells of one row per
// 64/128-bit access, NV accesses per lane): PL planes are in flight per lane before any is consumed -- one 4-byte load
// per lane and plane, as in the kernel above, leaves the pass bound by load latency -- the node of a cell is two table
// look-ups by shuffle (the index separates), and with PRIV the deposits go to the CTA's fixed-point table.
#ifndef MM_FREE_PRIV_PL
#define MM_FREE_PRIV_PL 4   // planes in flight per lane
#endif
#ifndef MM_FREE_PRIV_THREADS_F32
#define MM_FREE_PRIV_THREADS_F32 512   // 640 threads (96 registers): 12.8 ms on configs[4] instead of 11.2; 768 (80, spills): 19.3
#endif
template <typename real, int MODE, bool PRIV, int NXI, int NETA, int PL>
__global__ void __launch_bounds__(PRIV ? (sizeof(real) == 4 ? MM_FREE_PRIV_THREADS_F32 : 512) : 256) free_cells_vec_kernel(const FreeGeom q, int64_t nc, real *__restrict__ dens,
                                                                          const double *__restrict__ psi, double w,
                                                                          double *__restrict__ raw, const double *__restrict__ factor,
                                                                          const int *__restrict__ any_capped,
                                                                          unsigned long long *__restrict__ raw_fx = nullptr,
                                                                          double inv_unit = 1.0)
{
    constexpr int PLANE = NXI * NETA;
    constexpr int VW = (16 / (int)sizeof(real)) * 32 <= PLANE ? 16 / (int)sizeof(real) : PLANE / 32;   // cells per access
    constexpr int NV = PLANE / (32 * VW), LB = NETA / VW, RPV = 32 / LB;   // accesses per plane; lanes per row; rows per access
    static_assert(NXI <= 16 && NETA <= 16 && VW >= 1 && NV * 32 * VW == PLANE && NETA % VW == 0 && 32 % LB == 0, "plane must tile a warp");
    if (MODE == 1 && *any_capped == 0) return;
    struct alignas(sizeof(real) * VW) Vec { real v[VW]; };
    extern __shared__ double free_tab[];
    const int nn = q.nx * q.ny;
    // PRIV: the limb tables, rows padded to an odd stride -- the rows of a patch are ny apart in the global table, a
    // multiple of 32 banks on the BASELINE grids (8-way conflicts on every atomic otherwise)
    const int ldt = PRIV ? (q.ny | 1) : q.ny, nnp = q.nx * ldt;
    uint32_t *L0 = reinterpret_cast<uint32_t *>(free_tab), *L1 = L0 + nnp, *L2 = L1 + nnp;
    if (PRIV) {
        for (int i = threadIdx.x; i < 3 * nnp; i += blockDim.x) L0[i] = 0u;
        __syncthreads();
    }
    const int lane = threadIdx.x & 31;
    const int64_t warp0 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = ((int64_t)gridDim.x * blockDim.x) >> 5;
    const int k16 = lane & 15, arow = lane / LB, b0 = (lane % LB) * VW;
    const double off = lane < 16 ? __dadd_rn(-q.R, __dmul_rn(k16 + 0.5, q.dxi)) : __dadd_rn(-q.R, __dmul_rn(k16 + 0.5, q.deta));
    const int64_t inner = (int64_t)PLANE * q.ns;
    for (int64_t c = warp0; c < nc; c += nwarps) {
        const int itheta = (int)(c % q.ntheta);
        const int iy = (int)((c / q.ntheta) % q.ny), ix = (int)(c / ((int64_t)q.ntheta * q.ny));
        constexpr bool USE_TAB = sizeof(real) == 4;
        double cs = 0.0, base = 0.0;   // the inline node evaluation only
        if (!(USE_TAB && q.tabx)) {
            const double theta = 2.0 * 3.14159265358979323846264338327950288 * (double)itheta / (double)q.ntheta;
            cs = lane < 16 ? cos(theta) : sin(theta);
            base = lane < 16 ? __ddiv_rn((double)ix, (double)q.nx) : __ddiv_rn((double)iy, (double)q.ny);
        }
        const double nd = lane < 16 ? (double)q.nx : (double)q.ny;
        const double wp = MODE == 0 ? w * psi[c] : 0.0;
        if (MODE == 0 && wp == 0.0) continue;
        const double wps = wp * inv_unit * 4294967296.0;   // powers of two: wps * m rounds as wp * m
        real *mc = dens + c * inner + lane * VW;
        // with the context's tables the node of this lane (x node of row a = lane, or y node of column b = lane - 16)
        // is one 16-bit load per plane, issued with the density loads of the plane (a look-up at the point of use is a
        // dependent load in front of the atomics: slower than the inline evaluation).  fp32 contexts only: 10.9 -> 9.7 ms
        // on configs[4]; the fp64 pass, closer to its HBM roof and short of registers, got slower with it (3.6 -> 4.1 ms)
        const unsigned short *tab = nullptr;
        if (USE_TAB && q.tabx) {
            const int kk = k16 < (lane < 16 ? NXI : NETA) ? k16 : 0;
            tab = lane < 16 ? q.tabx + ((int64_t)ix * q.ntheta + itheta) * q.ns * NXI + kk
                            : q.taby + ((int64_t)iy * q.ntheta + itheta) * q.ns * NETA + kk;
        }
        const int tstride = lane < 16 ? NXI : NETA;
        for (int j0 = 0; j0 < q.ns; j0 += PL) {
            Vec v[PL][NV];
            int tnode[PL];
#pragma unroll
            for (int pl = 0; pl < PL; ++pl) {
#pragma unroll
                for (int k = 0; k < NV; ++k)
                    if (j0 + pl < q.ns) v[pl][k] = *reinterpret_cast<const Vec *>(mc + (int64_t)(j0 + pl) * PLANE + k * 32 * VW);
                if (USE_TAB) tnode[pl] = (tab && j0 + pl < q.ns) ? (int)tab[(j0 + pl) * tstride] : 0;
            }
#pragma unroll
            for (int pl = 0; pl < PL; ++pl) {
                const int j = j0 + pl;
                if (j >= q.ns) break;
                // lanes 0..15: x node of row a = lane (times ny); lanes 16..31: y node of column b = lane - 16; every
                // operation rounded separately, exactly the oracle's expression (ties)
                int my_node;
                if (USE_TAB && tab) {
                    my_node = lane < 16 ? tnode[pl] * ldt : tnode[pl];
                } else {
                    const double sj = __dadd_rn(q.s_lo, __dmul_rn(j + 0.5, q.ds));
                    const double r = __dmul_rn(__dsub_rn(__dadd_rn(base, __dmul_rn(sj, cs)), off), nd);
                    my_node = lane < 16 ? wrap_floor(__dadd_rn(r, 0.5), q.nx) * ldt : wrap_floor(__dadd_rn(r, 0.5), q.ny);
                }
                int nb[VW];
#pragma unroll
                for (int e = 0; e < VW; ++e) nb[e] = __shfl_sync(0xffffffffu, my_node, 16 + b0 + e);
                if (MODE == 0 && PRIV) {
                    // the NV * VW deposits of this lane's cells as three rounds of independent, unconditional atomics
                    // (limb 0 of every cell, then limb 1 with the carries, then -- rarely -- limb 2): one chain of
                    // returning ATOMS at a time leaves the pass bound by their latency, a branch around each by issue.
                    // The limbs come from two round-down additions of 1.5 * 2^52 (floor of |t| < 2^51 in the low mantissa
                    // bits) instead of three 64-bit conversions; a deposit outside that range takes fx_deposit.
                    constexpr int NB = NV * VW;
                    constexpr double MG = 6755399441055744.0;   // 1.5 * 2^52, bits 0x43380000'00000000
                    uint32_t n[NB];   // byte address of the node's limb 0 in shared memory
                    uint32_t x0[NB], x1[NB], x2[NB], bad = 0u;
                    const uint32_t sL0 = (uint32_t)__cvta_generic_to_shared(L0), limb = (uint32_t)nnp * 4u;
#pragma unroll
                    for (int k = 0; k < NV; ++k) {
                        const int na = __shfl_sync(0xffffffffu, my_node, k * RPV + arow);
#pragma unroll
                        for (int e = 0; e < VW; ++e) {
                            const int i = k * VW + e;
                            n[i] = sL0 + (uint32_t)(na + nb[e]) * 4u;
                            const double t = __dmul_rn(wps, (double)v[pl][k].v[e]);   // (w psi m / unit) 2^32, rounded as w psi m
                            const double tm = __dadd_rd(t, MG);
                            const double r = t - (tm - MG);                              // exact, in [0, 1)
                            x0[i] = (uint32_t)__double2loint(__fma_rd(r, 4294967296.0, MG));
                            x1[i] = (uint32_t)__double2loint(tm);
                            const uint32_t hi = (uint32_t)__double2hiint(tm);
                            x2[i] = hi - 0x43380000u;
                            bad |= hi ^ 0x43300000u;   // exponent field 0x433 <=> tm in [2^52, 2^53)
                        }
                    }
                    if (bad >> 20) {   // |t| >= 2^51 (a single deposit of 2^19 units or more) or not finite
#pragma unroll
                        for (int k = 0; k < NV; ++k)
#pragma unroll
                            for (int e = 0; e < VW; ++e) {
                                const double val = (double)v[pl][k].v[e];
                                if (val != 0.0) fx_deposit_rare(L0, L1, L2, (int)((n[k * VW + e] - sL0) >> 2), __dmul_rn(wp, val) * inv_unit);
                            }
                        continue;
                    }
                    uint32_t any2 = 0u;
#pragma unroll
                    for (int i = 0; i < NB; ++i) {
                        uint32_t o;
                        asm volatile("atom.shared.add.u32 %0, [%1], %2;" : "=r"(o) : "r"(n[i]), "r"(x0[i]) : "memory");
                        // x1 += carry of limb 0; x0 = carry out of that
                        asm("{\n\t.reg .u32 t;\n\tadd.cc.u32 t, %2, %3;\n\taddc.cc.u32 %0, %0, 0;\n\taddc.u32 %1, 0, 0;\n\t}"
                            : "+r"(x1[i]), "=r"(x0[i]) : "r"(o), "r"(x0[i]));
                    }
#pragma unroll
                    for (int i = 0; i < NB; ++i) {
                        uint32_t o;
                        asm volatile("atom.shared.add.u32 %0, [%1], %2;" : "=r"(o) : "r"(n[i] + limb), "r"(x1[i]) : "memory");
                        asm("{\n\t.reg .u32 t;\n\tadd.cc.u32 t, %1, %2;\n\taddc.u32 %0, %0, %3;\n\t}"
                            : "+r"(x2[i]) : "r"(o), "r"(x1[i]), "r"(x0[i]));
                        any2 |= x2[i];
                    }
                    if (any2) {
#pragma unroll
                        for (int i = 0; i < NB; ++i) reds_add_nz(n[i] + 2u * limb, x2[i]);
                    }
                    continue;
                }
#pragma unroll
                for (int k = 0; k < NV; ++k) {
                    const int na = __shfl_sync(0xffffffffu, my_node, k * RPV + arow);
                    bool dirty = false;
#pragma unroll
                    for (int e = 0; e < VW; ++e) {
                        const int n = na + nb[e];
                        if (MODE == 0) {
                            const double val = (double)v[pl][k].v[e];
                            if (val != 0.0) {
                                if (PRIV) fx_deposit(L0, L1, L2, n, __dmul_rn(wp, val) * inv_unit);
                                else atomicAdd(&raw[n], wp * val);
                            }
                        } else {
                            const double f = factor[n];
                            if (f != 1.0) { v[pl][k].v[e] = (real)((double)v[pl][k].v[e] * f); dirty = true; }
                        }
                    }
                    if (MODE == 1 && dirty) *reinterpret_cast<Vec *>(mc + (int64_t)j * PLANE + k * 32 * VW) = v[pl][k];
                }
            }
        }
    }
    if (PRIV) {
        // add this CTA's table to the global one: 128-bit fixed point, {low 64 fraction bits, signed integer part}
        __syncthreads();
        for (int i = threadIdx.x; i < nn; i += blockDim.x) {
            const int ip = (i / q.ny) * ldt + i % q.ny;
            const unsigned long long lo = ((unsigned long long)L1[ip] << 32) | L0[ip];
            long long hi = (long long)(int32_t)L2[ip];
            if (lo) { const unsigned long long o = atomicAdd(&raw_fx[2 * i], lo); hi += (o + lo < o) ? 1 : 0; }
            if (hi) atomicAdd(&raw_fx[2 * i + 1], (unsigned long long)hi);
        }
    }
}

// Per node: cap, factor, M_b,coarse, M_f.
// raw_fx != NULL: the sums arrive as 128-bit fixed point in units of `unit` (see fx_deposit)
__global__ void free_cap_kernel(int nn, double m_total, const double *__restrict__ raw, double *__restrict__ factor,
                                double *__restrict__ Mbc, double *__restrict__ Mf, int *__restrict__ any_capped,
                                const unsigned long long *__restrict__ raw_fx = nullptr, double unit = 1.0,
                                float *__restrict__ Mf_f32 = nullptr)
{
    for (int n = blockIdx.x * blockDim.x + threadIdx.x; n < nn; n += gridDim.x * blockDim.x) {
        const double r = raw_fx ? ((double)(long long)raw_fx[2 * n + 1] + (double)raw_fx[2 * n] * 5.421010862427522e-20) * unit : raw[n];
        const bool over = r > m_total;
        factor[n] = over ? m_total / r : 1.0;
        const double capped = over ? m_total : r;
        Mbc[n] = capped;
        Mf[n] = m_total - capped;
        if (Mf_f32) Mf_f32[n] = (float)(m_total - capped);
        if (over) *any_capped = 1;
    }
}

}  // namespace mm
