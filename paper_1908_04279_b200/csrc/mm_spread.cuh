// mm_spread.cuh -- SURVEY.md 8(f) NEXT-4: motor-force spreading onto the fluid grid (Eq. 10):
//     F_2(x) = F iiint p delta(y + (l/L) s p - x) Psi M_b ds dr0 dy dtheta.
// Readings Q34-Q37: the force carried by plane j of configuration c is the S9 spring force before the sum
// over j, f_j(c) = -k dxi deta sum_ab (xi_a, eta_b) m[c,j,a,b]; c = (ix, iy, itheta) sits at the node (ix/nx, iy/ny)
// of the periodic unit square and its head at X = x_c + s_j p_c; the delta is Peskin's 4-point kernel per direction;
//     F2[g] = dtheta ds sum_{c,j} Psi_c f_j(c) phi((X - X_g)_x / h_x) phi((X - X_g)_y / h_y).
// Two kernels: the plane forces (one HBM read of the density, one warp per configuration, no atomics), then the
// spreading of Nc*Ns point forces (16 nodes each) with fp64 atomic adds -- the paper's own structure ("independent
// GPU threads ... limiting the use of atomic operations to the final reduction").  Macro cadence.
#pragma once
#include "mm_common.cuh"

namespace mm {

// f_j(c) for every plane: fl[c][j][2] (fp64).  One warp per configuration; lanes stride over the plane, VW
// contiguous elements per load (VW = 1: any plane size).  fp32 contexts: fp32 within a lane, fp64 across lanes.
template <typename real, int VW>
__global__ void __launch_bounds__(256) plane_force_kernel(const __grid_constant__ KParams<real> kp,
                                                          const real *__restrict__ dens, double *__restrict__ fl)
{
    struct alignas(sizeof(real) * VW) Vec { real v[VW]; };
    const int plane = kp.nxi * kp.neta, nvec = plane / VW;
    const int lane = threadIdx.x & 31;
    const int64_t warp0 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = ((int64_t)gridDim.x * blockDim.x) >> 5;
    const double scale = kp.mom_scale / (double)kp.ds;   // -k dxi deta
    for (int64_t c = warp0; c < kp.nc; c += nwarps) {
        const Vec *mc = reinterpret_cast<const Vec *>(dens + c * (int64_t)plane * kp.ns);
        for (int j = 0; j < kp.ns; ++j) {
            real px = 0, py = 0;
            for (int iv = lane; iv < nvec; iv += 32) {
                const Vec v = mc[(int64_t)j * nvec + iv];
#pragma unroll
                for (int e = 0; e < VW; ++e) {
                    const int i = iv * VW + e;
                    const int a = i / kp.neta, b = i - a * kp.neta;
                    px = fma(-kp.R + (real(a) + real(0.5)) * kp.dxi, v.v[e], px);
                    py = fma(-kp.R + (real(b) + real(0.5)) * kp.deta, v.v[e], py);
                }
            }
            const double fx = warp_sum((double)px), fy = warp_sum((double)py);
            if (lane == 0) {
                fl[(c * kp.ns + j) * 2 + 0] = scale * fx;
                fl[(c * kp.ns + j) * 2 + 1] = scale * fy;
            }
        }
    }
}

__device__ __forceinline__ double peskin4(double r)
{
    const double a = fabs(r);
    if (a <= 1.0) return (3.0 - 2.0 * a + sqrt(1.0 + 4.0 * a - 4.0 * a * a)) / 8.0;
    if (a <= 2.0) return (5.0 - 2.0 * a - sqrt(-7.0 + 12.0 * a - 4.0 * a * a)) / 8.0;
    return 0.0;
}

// One thread per (c, j, u): the four nodes of stencil column u, both components: 8 fp64 atomic adds.
__global__ void __launch_bounds__(256) spread_kernel(int64_t nc, int ns, int nx, int ny, int ntheta, double s_lo, double ds,
                                                     const double *__restrict__ psi, const double *__restrict__ fl,
                                                     double *__restrict__ F2)
{
    const int64_t total = nc * ns * 4;
    const double dtheta = 2.0 * 3.14159265358979323846264338327950288 / (double)ntheta;
    for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (int64_t)gridDim.x * blockDim.x) {
        const int u = (int)(t & 3) - 1;
        const int64_t cj = t >> 2;
        const int64_t c = cj / ns;
        const int j = (int)(cj - c * ns);
        const double w0 = dtheta * ds * psi[c];
        if (w0 == 0.0) continue;
        const int itheta = (int)(c % ntheta);
        const int iy = (int)((c / ntheta) % ny), ix = (int)(c / ((int64_t)ntheta * ny));
        const double theta = 2.0 * 3.14159265358979323846264338327950288 * (double)itheta / (double)ntheta;
        const double sj = s_lo + (j + 0.5) * ds;
        const double gx = ((double)ix / nx + sj * cos(theta)) * nx, gy = ((double)iy / ny + sj * sin(theta)) * ny;
        const double bx = floor(gx), by = floor(gy);
        const double wx = peskin4(gx - (bx + u));
        long jx = ((long)bx + u) % nx;
        if (jx < 0) jx += nx;
        const double fx = fl[cj * 2], fy = fl[cj * 2 + 1];
#pragma unroll
        for (int v = -1; v <= 2; ++v) {
            const double w = w0 * wx * peskin4(gy - (by + v));
            long jy = ((long)by + v) % ny;
            if (jy < 0) jy += ny;
            atomicAdd(&F2[(jx * ny + jy) * 2 + 0], w * fx);
            atomicAdd(&F2[(jx * ny + jy) * 2 + 1], w * fy);
        }
    }
}

// ---- spreading as a GATHER (default).  The head of (ix, iy, itheta, j) sits at node coordinates (ix + t_x, iy + t_y)
// with t = s_j p(theta) (nx, ny): for a fixed pair (itheta, j) the stencil -- its integer offset floor(t) and its 4 x 4
// weights -- is the same for every (ix, iy), so
//     F2[g] = sum_{theta,j} sum_{u,v} w_{theta,j}(u, v) G_{theta,j}[g - floor(t) - (u, v)],   G = dtheta ds Psi f_j,
// 2048 shifted 4 x 4 stencils over 128 x 128 fields at configs[4] instead of 1.07 G atomic adds, and a sum in a fixed
// order.  Three kernels: (1) scale and transpose the plane forces to G[tj][node] (tj = itheta ns + j), so that the
// nodes a warp reads are contiguous; (2) one thread per target node and chunk of SPREAD_CH pairs tj; (3) the chunks
// summed in order.
constexpr int SPREAD_CH = 32;

__global__ void __launch_bounds__(256) spread_transpose_kernel(int nn, int ntheta, int ns, double w, const double *__restrict__ psi,
                                                               const double2 *__restrict__ fl, double2 *__restrict__ G)
{
    __shared__ double2 tile[32][33];
    const int nt = ntheta * ns;
    const int n0 = blockIdx.x * 32, tj0 = blockIdx.y * 32;
    for (int r = threadIdx.y; r < 32; r += 8) {   // rows: nodes; columns: tj (contiguous in fl)
        const int node = n0 + r, tj = tj0 + threadIdx.x;
        if (node < nn && tj < nt) {
            const double2 f = fl[(int64_t)node * nt + tj];
            const double ws = w * psi[(int64_t)node * ntheta + tj / ns];
            tile[r][threadIdx.x] = make_double2(ws * f.x, ws * f.y);
        }
    }
    __syncthreads();
    for (int r = threadIdx.y; r < 32; r += 8) {   // rows: tj; columns: nodes (contiguous in G)
        const int tj = tj0 + r, node = n0 + threadIdx.x;
        if (node < nn && tj < nt) G[(int64_t)tj * nn + node] = tile[threadIdx.x][r];
    }
}

__global__ void __launch_bounds__(256) spread_gather_kernel(int nx, int ny, int ntheta, int ns, double s_lo, double ds,
                                                            const double2 *__restrict__ G, double2 *__restrict__ part)
{
    __shared__ double wgt[SPREAD_CH][16];
    __shared__ int off[SPREAD_CH][2];
    const int nn = nx * ny, nt = ntheta * ns;
    const int tj0 = blockIdx.y * SPREAD_CH;
    const int ntj = min(SPREAD_CH, nt - tj0);
    if ((int)threadIdx.x < ntj) {   // the stencil of pair tj: offset reduced to [0, n), weights phi(frac - u) phi(frac - v)
        const int tj = tj0 + threadIdx.x, itheta = tj / ns, j = tj - itheta * ns;
        const double theta = 2.0 * 3.14159265358979323846264338327950288 * (double)itheta / (double)ntheta;
        const double sj = s_lo + (j + 0.5) * ds;
        const double tx = sj * cos(theta) * nx, ty = sj * sin(theta) * ny;
        const double bx = floor(tx), by = floor(ty);
        double wx[4], wy[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) { wx[u] = peskin4(tx - (bx + (u - 1))); wy[u] = peskin4(ty - (by + (u - 1))); }
#pragma unroll
        for (int u = 0; u < 4; ++u)
#pragma unroll
            for (int v = 0; v < 4; ++v) wgt[threadIdx.x][u * 4 + v] = wx[u] * wy[v];
        long ox = (long)bx % nx, oy = (long)by % ny;
        off[threadIdx.x][0] = (int)(ox < 0 ? ox + nx : ox);
        off[threadIdx.x][1] = (int)(oy < 0 ? oy + ny : oy);
    }
    __syncthreads();
    const int node = blockIdx.x * 256 + threadIdx.x;
    if (node >= nn) return;
    const int gx = node / ny, gy = node - gx * ny;
    double ax = 0.0, ay = 0.0;
    for (int t = 0; t < ntj; ++t) {
        const double2 *Gt = G + (int64_t)(tj0 + t) * nn;
        // the source of stencil point (u, v) is the node g - offset - (u, v): start at u = v = -1, step down with wrap
        int sx = gx - off[t][0] + 1, sy0 = gy - off[t][1] + 1;
        sx = sx < 0 ? sx + nx : (sx >= nx ? sx - nx : sx);
        sy0 = sy0 < 0 ? sy0 + ny : (sy0 >= ny ? sy0 - ny : sy0);
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            int sy = sy0;
#pragma unroll
            for (int v = 0; v < 4; ++v) {
                const double2 g = Gt[sx * ny + sy];
                const double w = wgt[t][u * 4 + v];
                ax = fma(w, g.x, ax);
                ay = fma(w, g.y, ay);
                sy = sy == 0 ? ny - 1 : sy - 1;
            }
            sx = sx == 0 ? nx - 1 : sx - 1;
        }
    }
    part[(int64_t)blockIdx.y * nn + node] = make_double2(ax, ay);
}

__global__ void __launch_bounds__(256) spread_sum_kernel(int nn, int nchunks, const double2 *__restrict__ part, double2 *__restrict__ F2)
{
    const int node = blockIdx.x * 256 + threadIdx.x;
    if (node >= nn) return;
    double ax = 0.0, ay = 0.0;
    for (int k = 0; k < nchunks; ++k) {
        const double2 p = part[(int64_t)k * nn + node];
        ax += p.x;
        ay += p.y;
    }
    F2[node] = make_double2(ax, ay);
}

}  // namespace mm
