/* oracle/mm_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU statement of the bound-motor microscale substep of Cook & Shinar
 * (arxiv 1908.04279), in the re-parametrised form BASELINE.json `north_star` names:
 * density m over configuration c=(x,y,theta) x arc length s x stalk offset (xi,eta).
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may build, load or call this file.  It shares no code with paper_1908_04279_b200/.
 *
 * The method is an explicit iteration, so the oracle IS the algorithm, step by step, as
 * literal loops in flux-difference form, in the order of SURVEY.md section 8(c) S1..S9:
 *   - motor equation  d_t M_b + d_s M_b = -k_off M_b + k_on M_f 1_{D_rc}   PAPER.md:60 (Eq. 4)
 *   - capture-radius restriction |x + s p - r0| <= r_c
 *   - per-unit explicit update, units independent                          PAPER.md:91, Alg. 2
 *   - motor force / reduction per unit                                     PAPER.md:80-81 (Eq. 10), Alg. 2 l.14 PAPER.md:206-208
 *   - force-dependent walking speed, head-relative-to-tail advection in (xi,eta), Bell
 *     detachment, end detachment, spring-force moments: BASELINE.json north_star (1)-(3).
 * The paper prints no discretisation; every reading (Q1..Q23) is listed in DESIGN.md.
 *
 * Parity pins (tests/test_oracle_pins.py): C1 mass conservation, C1b discrete mass budget,
 * C2 pure detachment closed form, C3 exact shift at CFL=1, C4 steady-state recursion,
 * C5 brute-force/analytic moments on 2x2x2x4x3x3, C6 single-cell delta column, C7 point
 * symmetry, C8 independence/additivity, C9 positivity/affinity; the NEXT-row functions further down by R1-R7
 * (RK2 + Superbee), L1-L5 (local time step; L5: with the coupled source), F1-F5 (force spreading), N1-N7 (free-motor
 * coupling; N6: which node a cell's coupled source is read from, one-hot tables against the exact-rational anchor map;
 * N7: Alg. 2's cadence, mmo_run_alg2).  No function is unpinned.
 *
 * Second scheme (flag MMO_RK2_SUPERBEE): the paper's own integrator --
 * Runge-Kutta 2 through the half step (Alg. 2 l.9-10: "Compute M_b(t^* + dt^* / 2)",
 * "Compute M_b(t^* + dt^*)"; "We instead use Runge-Kutta 2, which only requires the M_b array at
 * t^{n+1} and t^n") with the Superbee flux limiter in the arclength dimension
 * ("applies a Superbee flux limiter"; "The Superbee flux limiter operates
 * in the arclength s dimension ... neighborhood access pattern of (s-2,s-1,s,s+1,s+2)").  The paper
 * prints neither formula; the readings (Q27-Q30) are: midpoint RK2 as a method of lines,
 *     m* = m^n + (dt/2) L(m^n),   m^{n+1} = m^n + dt L(m*),
 * L(m) = -div F(m) + src - kappa m, both stages masked to the disc; the s flux on face j+1/2 is
 * W (m_j + sigma_j / 2) with the Superbee-limited slope in its division-free form
 *     sigma_j = maxmod( minmod(2a, b), minmod(a, 2b) ),  a = m_j - m_{j-1},  b = m_{j+1} - m_j
 * (= phi(r) b with phi(r) = max(0, min(2r,1), min(r,2)), r = a/b); ghosts beyond both ends of s
 * are 0 as in S5; (xi, eta) stay first-order upwind.  Pins R1-R7 in tests/test_oracle_rk2_pins.py.
 *
 * Parallelism: `#pragma omp parallel for` over configurations only (they never interact).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct { int32_t nx, ny, ntheta, ns, nxi, neta; } mmo_grid;

typedef struct {
    double v0, f_stall, k_spring, k_on, k_off0, f_detach, end_detach_mult, m_free, R;
    double s_lo, s_hi;
    int32_t n_end_cells;
    uint32_t flags;
} mmo_params;

#define MMO_S_PERIODIC 1u
#define MMO_OFFSET_PERIODIC_NOMASK 2u
#define MMO_RK2_SUPERBEE 8u   /* bit 2 (4u) is the product's CHECK_DT flag; unused here */

static const double MMO_PI = 3.14159265358979323846264338327950288;

/* S1: exact integer disc test  xi_a^2 + eta_b^2 <= R^2  at cell centres */
static int inside(const mmo_grid *g, const mmo_params *p, int a, int b)
{
    if (p->flags & MMO_OFFSET_PERIODIC_NOMASK) return 1;
    int64_t u = 2 * (int64_t)a + 1 - g->nxi, v = 2 * (int64_t)b + 1 - g->neta;
    int64_t nx2 = (int64_t)g->nxi * g->nxi, ne2 = (int64_t)g->neta * g->neta;
    return u * u * ne2 + v * v * nx2 <= nx2 * ne2;
}

/* S3: walking speed, linear force-velocity law clamped below at 0 (Q5, Q6) */
static double walk_speed(const mmo_params *p, double ct, double st, double xi, double eta)
{
    double load = p->k_spring * (xi * ct + eta * st) / p->f_stall;
    double f = 1.0 - load;
    return p->v0 * (f > 0.0 ? f : 0.0);
}

static double dmax(double a, double b) { return a > b ? a : b; }
static double dmin(double a, double b) { return a < b ? a : b; }

/* Superbee-limited slope (division-free form; LeVeque's maxmod/minmod statement of the limiter the
 * paper names at PAPER.md:89, 175).  a = backward difference, b = forward difference. */
static double minmod(double a, double b)
{
    if (a * b <= 0.0) return 0.0;
    return a > 0.0 ? dmin(a, b) : dmax(a, b);
}
static double maxmod(double a, double b)
{
    if (a * b <= 0.0) return 0.0;
    return a > 0.0 ? dmax(a, b) : dmin(a, b);
}
static double superbee_slope(double a, double b) { return maxmod(minmod(2.0 * a, b), minmod(a, 2.0 * b)); }

/* One explicit stage (S2..S7) of ONE configuration:
 *     mnew = inside ? mbase + dt * L(m) : 0,    L(m) = -div F(m) + src - kappa m.
 * Forward Euler (the north_star scheme) is the single stage mbase = m.  RK2 calls it twice
 * (mbase = m^n both times; m = m^n with dt/2, then m = m* with dt).  `limited` switches the s flux
 * from first-order upwind to the Superbee-limited one.
 * m, mbase, mnew: [ns][nxi][neta], b fastest.  scratch: 3 flux arrays (sizes below). */
/* Nearest node of the periodic (x, y) grid to the anchor (tail) of cell (c, j, a, b) -- SURVEY.md 8(f) NEXT-2,
 * reading Q38/Q39: the tail is the head minus the stalk offset, r0 = x_c + s_j p_c - (xi_a, eta_b). */
static size_t anchor_node(const mmo_grid *g, int ix, int iy, double ct, double st, double sj, double xi, double eta)
{
    double rx = ((double)ix / g->nx + sj * ct - xi) * g->nx, ry = ((double)iy / g->ny + sj * st - eta) * g->ny;
    long nx_ = (long)floor(rx + 0.5) % g->nx, ny_ = (long)floor(ry + 0.5) % g->ny;
    if (nx_ < 0) nx_ += g->nx;
    if (ny_ < 0) ny_ += g->ny;
    return (size_t)nx_ * g->ny + (size_t)ny_;
}

static void stage_config(const mmo_grid *g, const mmo_params *p, int itheta,
                         double U, double V, double Om, double dt,
                         const double *mbase, const double *m, double *mnew, int limited,
                         double *Fs, double *Fxi, double *Feta,
                         const double *Mf, int ix, int iy)   /* Mf != NULL: source k_on M_f(r0) (Eq. 4 with Eq. 6) */
{
    const int ns = g->ns, nxi = g->nxi, neta = g->neta;
    const int per_s = (p->flags & MMO_S_PERIODIC) != 0;
    const int per_o = (p->flags & MMO_OFFSET_PERIODIC_NOMASK) != 0;
    const double R = p->R;
    const double ds = (p->s_hi - p->s_lo) / ns, dxi = 2.0 * R / nxi, deta = 2.0 * R / neta;
    /* S1/S2 */
    const double theta = 2.0 * MMO_PI * (double)itheta / (double)g->ntheta;
    const double ct = cos(theta), st = sin(theta);
#define M(j, a, b) m[((size_t)(j) * nxi + (a)) * neta + (b)]
    /* S5, s-faces.  Fs index jf = 0..ns  is the face s_{jf - 1/2}; upwind cell is jf-1 (W >= 0). */
#define FS(jf, a, b) Fs[((size_t)(jf) * nxi + (a)) * neta + (b)]
    for (int a = 0; a < nxi; ++a)
        for (int b = 0; b < neta; ++b) {
            double xi = -R + (a + 0.5) * dxi, eta = -R + (b + 0.5) * deta;
            double W = walk_speed(p, ct, st, xi, eta);            /* S4: W[c,a,b] */
            if (!limited) {
                for (int jf = 1; jf <= ns; ++jf) FS(jf, a, b) = W * M(jf - 1, a, b);
            } else {
                /* Superbee in s: face jf takes cell j = jf-1 plus half its limited slope */
                for (int jf = 1; jf <= ns; ++jf) {
                    int j = jf - 1;
                    double mc = M(j, a, b);
                    double mm1 = j >= 1 ? M(j - 1, a, b) : (per_s ? M(ns - 1, a, b) : 0.0);
                    double mp1 = j + 1 < ns ? M(j + 1, a, b) : (per_s ? M(0, a, b) : 0.0);
                    FS(jf, a, b) = W * (mc + 0.5 * superbee_slope(mc - mm1, mp1 - mc));
                }
            }
            FS(0, a, b) = per_s ? FS(ns, a, b) : 0.0;             /* zero inflow at s = s_lo (Q9) */
        }
    /* S5, xi-faces.  index af = 0..nxi is the face xi_{af - 1/2} = -R + af*dxi. */
#define FXI(j, af, b) Fxi[((size_t)(j) * (nxi + 1) + (af)) * neta + (b)]
    for (int j = 0; j < ns; ++j) {
        double sj = p->s_lo + (j + 0.5) * ds;
        for (int af = 0; af <= nxi; ++af)
            for (int b = 0; b < neta; ++b) {
                if (per_o && af == nxi) { FXI(j, af, b) = FXI(j, 0, b); continue; }  /* ONE wrapped face */
                double xif = -R + af * dxi, eta = -R + (b + 0.5) * deta;
                double A = U + walk_speed(p, ct, st, xif, eta) * ct - sj * Om * st;   /* S4: A_xi */
                double mL, mR;
                if (per_o) {
                    mL = M(j, (af - 1 + nxi) % nxi, b);
                    mR = M(j, af % nxi, b);
                } else {
                    mL = af >= 1 ? M(j, af - 1, b) : 0.0;        /* ghost = 0 (Q10) */
                    mR = af < nxi ? M(j, af, b) : 0.0;
                }
                FXI(j, af, b) = dmax(A, 0.0) * mL + dmin(A, 0.0) * mR;
            }
    }
    /* S5, eta-faces.  index bf = 0..neta is the face eta_{bf - 1/2} = -R + bf*deta. */
#define FETA(j, a, bf) Feta[((size_t)(j) * nxi + (a)) * (neta + 1) + (bf)]
    for (int j = 0; j < ns; ++j) {
        double sj = p->s_lo + (j + 0.5) * ds;
        for (int a = 0; a < nxi; ++a)
            for (int bf = 0; bf <= neta; ++bf) {
                if (per_o && bf == neta) { FETA(j, a, bf) = FETA(j, a, 0); continue; }
                double xi = -R + (a + 0.5) * dxi, etaf = -R + bf * deta;
                double A = V + walk_speed(p, ct, st, xi, etaf) * st + sj * Om * ct;   /* S4: A_eta */
                double mL, mR;
                if (per_o) {
                    mL = M(j, a, (bf - 1 + neta) % neta);
                    mR = M(j, a, bf % neta);
                } else {
                    mL = bf >= 1 ? M(j, a, bf - 1) : 0.0;
                    mR = bf < neta ? M(j, a, bf) : 0.0;
                }
                FETA(j, a, bf) = dmax(A, 0.0) * mL + dmin(A, 0.0) * mR;
            }
    }
    /* S6 + S7 */
    for (int j = 0; j < ns; ++j) {
        double E = (j < p->n_end_cells || j >= ns - p->n_end_cells) ? p->end_detach_mult : 1.0;  /* Q8 */
        for (int a = 0; a < nxi; ++a)
            for (int b = 0; b < neta; ++b) {
                double xi = -R + (a + 0.5) * dxi, eta = -R + (b + 0.5) * deta;
                double r = sqrt(xi * xi + eta * eta);
                double kappa = p->k_off0 * exp(p->k_spring * r / p->f_detach) * E;     /* Bell law (Q7) */
                int in = inside(g, p, a, b);
                double src = in ? p->k_on * p->m_free : 0.0;                           /* Q11 */
                if (Mf && in) {                                                        /* Q42: k_on M_f at the anchor's node */
                    double sj = p->s_lo + (j + 0.5) * ds;
                    src = p->k_on * Mf[anchor_node(g, ix, iy, ct, st, sj, xi, eta)];
                }
                double mc = M(j, a, b);
                double div = (FS(j + 1, a, b) - FS(j, a, b)) / ds
                           + (FXI(j, a + 1, b) - FXI(j, a, b)) / dxi
                           + (FETA(j, a, b + 1) - FETA(j, a, b)) / deta;
                double mb = mbase[((size_t)j * nxi + a) * neta + b];
                double mp = mb - dt * div + dt * (src - kappa * mc);
                mnew[((size_t)j * nxi + a) * neta + b] = in ? mp : 0.0;
            }
    }
#undef M
#undef FS
#undef FXI
#undef FETA
}

static size_t scratch_doubles(const mmo_grid *g)
{
    size_t ns = g->ns, nxi = g->nxi, neta = g->neta;
    return (ns + 1) * nxi * neta + ns * (nxi + 1) * neta + ns * nxi * (neta + 1) + 2 * ns * nxi * neta;
}

/* Advance configurations [0, n_configs) by n_sub substeps of size dt, in place.
 * m: [n_configs][ns][nxi][neta]; U,V,Om: [n_configs]; itheta0: theta index of the first
 * configuration is (c_first % ntheta) where c_first is the global index of m's first config. */
static int run_impl(const mmo_grid *g, const mmo_params *p, int64_t c_first, int64_t n_configs,
                    const double *U, const double *V, const double *Om,
                    double *m, int32_t n_sub, double dt, const double *Mf)
{
    const size_t inner = (size_t)g->ns * g->nxi * g->neta;
    int fail = 0;
#pragma omp parallel for schedule(static)
    for (int64_t c = 0; c < n_configs; ++c) {
        double *scr = (double *)malloc(sizeof(double) * scratch_doubles(g));
        if (!scr) { fail = 1; continue; }
        double *Fs = scr;
        double *Fxi = Fs + (size_t)(g->ns + 1) * g->nxi * g->neta;
        double *Feta = Fxi + (size_t)g->ns * (g->nxi + 1) * g->neta;
        double *tmp = Feta + (size_t)g->ns * g->nxi * (g->neta + 1);
        double *half = tmp + inner;
        double *cur = m + (size_t)c * inner;
        int itheta = (int)((c_first + c) % g->ntheta);
        int iy = (int)(((c_first + c) / g->ntheta) % g->ny), ix = (int)((c_first + c) / ((int64_t)g->ntheta * g->ny));
        for (int n = 0; n < n_sub; ++n) {
            if (p->flags & MMO_RK2_SUPERBEE) {
                /* Alg. 2 l.9: M_b at t + dt/2;  l.10: M_b at t + dt */
                stage_config(g, p, itheta, U[c], V[c], Om[c], 0.5 * dt, cur, cur, half, 1, Fs, Fxi, Feta, Mf, ix, iy);
                stage_config(g, p, itheta, U[c], V[c], Om[c], dt, cur, half, tmp, 1, Fs, Fxi, Feta, Mf, ix, iy);
            } else {
                stage_config(g, p, itheta, U[c], V[c], Om[c], dt, cur, cur, tmp, 0, Fs, Fxi, Feta, Mf, ix, iy);
            }
            memcpy(cur, tmp, sizeof(double) * inner);   /* "swap buffers" */
        }
        free(scr);
    }
    return fail ? -1 : 0;
}

int mmo_run(const mmo_grid *g, const mmo_params *p, int64_t c_first, int64_t n_configs,
            const double *U, const double *V, const double *Om,
            double *m, int32_t n_sub, double dt)
{
    return run_impl(g, p, c_first, n_configs, U, V, Om, m, n_sub, dt, NULL);
}

/* ---- free-motor coupling -----------------------------------------------------------------
 * Eq. 5: M_b,coarse = iiint M_b Psi ds dx dtheta (per r0);  Eq. 6: M_f = M - M_b,coarse;
 * Alg. 2 l.14-20: compute M_b,coarse(r0) (reduction); if M_total(r0) < M_b,coarse(r0): scale all
 * M_b of that r0 and set M_b,coarse = M_total; compute M_f(r0).  Readings Q38-Q42:
 *  - the anchor of cell (c,j,a,b) is r0 = x_c + s_j p_c - (xi_a, eta_b); it is binned to the NEAREST node of the
 *    periodic (x, y) grid, so that every cell belongs to exactly one r0 (the cap rescales "all M_b with that r0");
 *  - M_b,coarse[n] = dtheta ds dxi deta sum_{cells -> n} Psi_c m   (dx at fixed r0 is dxi deta; h_x h_y cancels);
 *  - M_total = params.m_free at every node; f[n] = min(1, M_total / M_b,coarse[n]) multiplies the cells of node n;
 *  - M_f[n] = M_total - min(M_b,coarse[n], M_total) >= 0 then feeds the source k_on M_f(r0) 1_disc of Eq. 4.
 * m: ALL configurations [nc][ns][nxi][neta], rescaled in place; Mbc, Mf: [nx][ny] (outputs, either may be NULL). */
int mmo_free_motors(const mmo_grid *g, const mmo_params *p, double *m, const double *psi, double *Mbc, double *Mf)
{
    const int ns = g->ns, nxi = g->nxi, neta = g->neta;
    const int64_t nc = (int64_t)g->nx * g->ny * g->ntheta;
    const size_t nn = (size_t)g->nx * g->ny, inner = (size_t)ns * nxi * neta;
    const double R = p->R;
    const double ds = (p->s_hi - p->s_lo) / ns, dxi = 2.0 * R / nxi, deta = 2.0 * R / neta;
    const double w = 2.0 * MMO_PI / (double)g->ntheta * ds * dxi * deta;
    double *acc = (double *)calloc(nn, sizeof(double));
    if (!acc) return -1;
    for (int pass = 0; pass < 2; ++pass) {              /* pass 0: coarse sums; pass 1: cap rescale */
        for (int64_t c = 0; c < nc; ++c) {
            int itheta = (int)(c % g->ntheta);
            int iy = (int)((c / g->ntheta) % g->ny), ix = (int)(c / ((int64_t)g->ntheta * g->ny));
            double theta = 2.0 * MMO_PI * (double)itheta / (double)g->ntheta;
            double ct = cos(theta), st = sin(theta);
            for (int j = 0; j < ns; ++j) {
                double sj = p->s_lo + (j + 0.5) * ds;
                for (int a = 0; a < nxi; ++a)
                    for (int b = 0; b < neta; ++b) {
                        double xi = -R + (a + 0.5) * dxi, eta = -R + (b + 0.5) * deta;
                        size_t n = anchor_node(g, ix, iy, ct, st, sj, xi, eta);
                        double *v = &m[(size_t)c * inner + ((size_t)j * nxi + a) * neta + b];
                        if (pass == 0) acc[n] += w * psi[c] * (*v);
                        else if (acc[n] > p->m_free) *v *= p->m_free / acc[n];
                    }
            }
        }
    }
    for (size_t n = 0; n < nn; ++n) {
        double capped = acc[n] > p->m_free ? p->m_free : acc[n];
        if (Mbc) Mbc[n] = capped;
        if (Mf) Mf[n] = p->m_free - capped;
    }
    free(acc);
    return 0;
}

/* mmo_run with the source k_on M_f(r0) of the given free-motor table (frozen over these substeps). */
int mmo_run_coupled(const mmo_grid *g, const mmo_params *p, int64_t c_first, int64_t n_configs,
                    const double *U, const double *V, const double *Om,
                    double *m, int32_t n_sub, double dt, const double *Mf)
{
    return run_impl(g, p, c_first, n_configs, U, V, Om, m, n_sub, dt, Mf);
}

/* Alg. 2 with the paper's cadence: the coarse reduction, the cap and M_f (l.14-20) sit INSIDE the
 * inner loop `while t* < t*_end` (l.4), i.e. they are redone after inner steps, not once per macro step.  Here: before
 * every `refresh`-th substep (substeps 0, refresh, 2 refresh, ...) mmo_free_motors is applied to the whole state (cap
 * rescale included) and the following substeps take their source from the new table.  refresh = 1 is the paper's loop;
 * refresh >= n_sub is one update followed by mmo_run_coupled.  m: ALL configurations; Mbc, Mf: the tables of the LAST
 * update (outputs, [nx][ny]).  Nothing new is computed here: the function composes mmo_free_motors and run_impl. */
int mmo_run_alg2(const mmo_grid *g, const mmo_params *p, const double *U, const double *V, const double *Om,
                 double *m, const double *psi, int32_t n_sub, double dt, int32_t refresh, double *Mbc, double *Mf)
{
    const int64_t nc = (int64_t)g->nx * g->ny * g->ntheta;
    if (refresh < 1 || !Mf) return -2;
    for (int32_t n = 0; n < n_sub; n += refresh) {
        int32_t k = n_sub - n < refresh ? n_sub - n : refresh;
        if (mmo_free_motors(g, p, m, psi, Mbc, Mf) != 0) return -1;
        if (run_impl(g, p, 0, nc, U, V, Om, m, k, dt, Mf) != 0) return -1;
    }
    return 0;
}

/* ---- local adaptive time step per independent unit ------------------------------------
 * "We instead compute a local dt* for each r0 at the beginning of each inner time step and update M_b at each r0
 * asynchronously"; Alg. 2 l.2-5: "Set t*_end = t + dt; for r0 in grid: while
 * t* < t*_end: compute adaptive dt*"; "the inner time step dt* restricted by the motor speed and binding/unbinding
 * rates in Eq. (4)".  The paper prints no formula; readings Q31-Q33:
 *  - the unit is the configuration c (this path's independent unit, as r0 is the paper's);
 *  - its stability rate is the S8 positivity rate maximised over the cells of the unit that are evolved
 *    (inside the disc):  lambda_c = max_{j,a,b} [ W/ds + (max(Axi[a+1/2],0) - min(Axi[a-1/2],0))/dxi
 *                                              + (max(Aeta[b+1/2],0) - min(Aeta[b-1/2],0))/deta + kappa_ab E_j ];
 *    the rates do not depend on m, so dt* is constant over the macro step;
 *  - n_c = max(1, ceil(dt lambda_c / cfl)) local steps of equal size dt*_c = dt / n_c (<= cfl / lambda_c), which
 *    land exactly on t + dt. */
int mmo_rate_bound(const mmo_grid *g, const mmo_params *p, int64_t c_first, int64_t n_configs,
                   const double *U, const double *V, const double *Om, double *lambda)
{
    const int ns = g->ns, nxi = g->nxi, neta = g->neta;
    const double R = p->R;
    const double ds = (p->s_hi - p->s_lo) / ns, dxi = 2.0 * R / nxi, deta = 2.0 * R / neta;
#pragma omp parallel for schedule(static)
    for (int64_t c = 0; c < n_configs; ++c) {
        int itheta = (int)((c_first + c) % g->ntheta);
        double theta = 2.0 * MMO_PI * (double)itheta / (double)g->ntheta;
        double ct = cos(theta), st = sin(theta);
        double lam = 0.0;
        for (int j = 0; j < ns; ++j) {
            double sj = p->s_lo + (j + 0.5) * ds;
            double E = (j < p->n_end_cells || j >= ns - p->n_end_cells) ? p->end_detach_mult : 1.0;
            for (int a = 0; a < nxi; ++a)
                for (int b = 0; b < neta; ++b) {
                    if (!inside(g, p, a, b)) continue;
                    double xi = -R + (a + 0.5) * dxi, eta = -R + (b + 0.5) * deta;
                    double W = walk_speed(p, ct, st, xi, eta);
                    double Axh = U[c] + walk_speed(p, ct, st, -R + (a + 1) * dxi, eta) * ct - sj * Om[c] * st;
                    double Axl = U[c] + walk_speed(p, ct, st, -R + a * dxi, eta) * ct - sj * Om[c] * st;
                    double Aeh = V[c] + walk_speed(p, ct, st, xi, -R + (b + 1) * deta) * st + sj * Om[c] * ct;
                    double Ael = V[c] + walk_speed(p, ct, st, xi, -R + b * deta) * st + sj * Om[c] * ct;
                    double r = sqrt(xi * xi + eta * eta);
                    double kappa = p->k_off0 * exp(p->k_spring * r / p->f_detach) * E;
                    double rate = W / ds + (dmax(Axh, 0.0) - dmin(Axl, 0.0)) / dxi
                                + (dmax(Aeh, 0.0) - dmin(Ael, 0.0)) / deta + kappa;
                    lam = dmax(lam, rate);
                }
        }
        lambda[c] = lam;
    }
    return 0;
}

/* Advance every configuration from t to t + dt with its own n_c equal local steps (see above); the scheme of each
 * local step is the one the flags select.  n_steps (may be NULL) receives n_c. */
static int advance_local_impl(const mmo_grid *g, const mmo_params *p, int64_t c_first, int64_t n_configs,
                              const double *U, const double *V, const double *Om,
                              double *m, double dt, double cfl, int32_t *n_steps, const double *Mf)
{
    const size_t inner = (size_t)g->ns * g->nxi * g->neta;
    double *lambda = (double *)malloc(sizeof(double) * (size_t)(n_configs > 0 ? n_configs : 1));
    if (!lambda) return -1;
    mmo_rate_bound(g, p, c_first, n_configs, U, V, Om, lambda);
    int fail = 0;
#pragma omp parallel for schedule(dynamic)
    for (int64_t c = 0; c < n_configs; ++c) {
        double need = ceil(dt * lambda[c] / cfl);
        int32_t n_c = need < 1.0 ? 1 : (int32_t)need;
        if (n_steps) n_steps[c] = n_c;
        if (run_impl(g, p, c_first + c, 1, U + c, V + c, Om + c, m + (size_t)c * inner, n_c, dt / (double)n_c, Mf) != 0)
            fail = 1;
    }
    free(lambda);
    return fail ? -1 : 0;
}

int mmo_advance_local(const mmo_grid *g, const mmo_params *p, int64_t c_first, int64_t n_configs,
                      const double *U, const double *V, const double *Om,
                      double *m, double dt, double cfl, int32_t *n_steps)
{
    return advance_local_impl(g, p, c_first, n_configs, U, V, Om, m, dt, cfl, n_steps, NULL);
}

/* Alg. 2 as ONE loop: the local steps of l.5 with the source k_on M_f(r0) of the given table (frozen
 * over the macro step, reading Q42).  The step count does not depend on the source (reading Q32: lambda_c is the S8
 * rate of advection and detachment), so n_c is the same as without the table. */
int mmo_advance_local_coupled(const mmo_grid *g, const mmo_params *p, int64_t c_first, int64_t n_configs,
                              const double *U, const double *V, const double *Om,
                              double *m, double dt, double cfl, int32_t *n_steps, const double *Mf)
{
    return advance_local_impl(g, p, c_first, n_configs, U, V, Om, m, dt, cfl, n_steps, Mf);
}

/* S9: per-configuration moments; force [n][2], torque [n]; optional (may be NULL) test-only
 * cancellation-free scales N0 = dV sum m, SF = k dV sum r m, Stau = k dV sum |s| r m. */
int mmo_moments(const mmo_grid *g, const mmo_params *p, int64_t c_first, int64_t n_configs,
                const double *m, double *force, double *torque,
                double *N0, double *SF, double *Stau)
{
    const int ns = g->ns, nxi = g->nxi, neta = g->neta;
    const double R = p->R, k = p->k_spring;
    const double ds = (p->s_hi - p->s_lo) / ns, dxi = 2.0 * R / nxi, deta = 2.0 * R / neta;
    const double dV = ds * dxi * deta;
    const size_t inner = (size_t)ns * nxi * neta;
#pragma omp parallel for schedule(static)
    for (int64_t c = 0; c < n_configs; ++c) {
        int itheta = (int)((c_first + c) % g->ntheta);
        double theta = 2.0 * MMO_PI * (double)itheta / (double)g->ntheta;
        double ct = cos(theta), st = sin(theta);
        double sx = 0.0, sy = 0.0, stq = 0.0, s0 = 0.0, sf = 0.0, sta = 0.0;
        const double *mc = m + (size_t)c * inner;
        for (int j = 0; j < ns; ++j) {
            double sj = p->s_lo + (j + 0.5) * ds;
            for (int a = 0; a < nxi; ++a)
                for (int b = 0; b < neta; ++b) {
                    double xi = -R + (a + 0.5) * dxi, eta = -R + (b + 0.5) * deta;
                    double v = mc[((size_t)j * nxi + a) * neta + b];
                    double r = sqrt(xi * xi + eta * eta);
                    sx += xi * v;
                    sy += eta * v;
                    stq += sj * (eta * ct - xi * st) * v;
                    s0 += v;
                    sf += r * v;
                    sta += fabs(sj) * r * v;
                }
        }
        force[2 * c + 0] = -k * dV * sx;
        force[2 * c + 1] = -k * dV * sy;
        torque[c] = -k * dV * stq;
        if (N0) N0[c] = dV * s0;
        if (SF) SF[c] = k * dV * sf;
        if (Stau) Stau[c] = k * dV * sta;
    }
    return 0;
}

/* ---- motor-force spreading onto the fluid grid ----------------------------------------
 * Eq. 10: F_2(x) = F iiint f ds dr0 dy dtheta, f = p delta(y + (l/L) s p - x) Psi M_b: the force the
 * bound motors exert is weighted by the filament density Psi and spread to the fluid point under the motor head
 * with a delta function; "use independent GPU threads to compute the integral ... limiting the use of atomic
 * operations to the final reduction".  The paper does not print the discrete delta or the quadrature;
 * readings Q34-Q37:
 *  - the force carried by plane j of configuration c is the spring force of S9 before the sum over j,
 *        f_j(c) = -k dxi deta sum_ab (xi_a, eta_b) m[c,j,a,b]      (so that ds sum_j f_j(c) = the S9 force);
 *  - configuration c = (ix, iy, itheta) sits at the node x_c = (ix/nx, iy/ny) of the periodic unit square; the head
 *    of plane j is at X = x_c + s_j p_c  (l/L = 1, Q4);
 *  - delta_h = Peskin's 4-point kernel phi in each direction, delta_h(r) = phi(r_x/h_x) phi(r_y/h_y) / (h_x h_y),
 *        phi(r) = (3 - 2|r| + sqrt(1 + 4|r| - 4 r^2))/8 for |r| <= 1, (5 - 2|r| - sqrt(-7 + 12|r| - 4 r^2))/8 for
 *        1 <= |r| <= 2, 0 beyond; the grid is periodic;
 *  - quadrature: F_2[g] = sum_c sum_j Psi_c f_j(c) delta_h(X_g - X_cj) ds (h_x h_y dtheta)
 *                       = dtheta ds sum_{c,j} Psi_c f_j(c) phi(.) phi(.).
 * F2: [nx][ny][2], ACCUMULATED into (the caller zeroes it); configurations [c_first, c_first + n_configs). */
static double peskin4(double r)
{
    double a = fabs(r);
    if (a <= 1.0) return (3.0 - 2.0 * a + sqrt(1.0 + 4.0 * a - 4.0 * a * a)) / 8.0;
    if (a <= 2.0) return (5.0 - 2.0 * a - sqrt(-7.0 + 12.0 * a - 4.0 * a * a)) / 8.0;
    return 0.0;
}

int mmo_spread_force(const mmo_grid *g, const mmo_params *p, int64_t c_first, int64_t n_configs,
                     const double *m, const double *psi, double *F2)
{
    const int ns = g->ns, nxi = g->nxi, neta = g->neta, nx = g->nx, ny = g->ny;
    const double R = p->R, k = p->k_spring;
    const double ds = (p->s_hi - p->s_lo) / ns, dxi = 2.0 * R / nxi, deta = 2.0 * R / neta;
    const double dtheta = 2.0 * MMO_PI / (double)g->ntheta;
    const size_t inner = (size_t)ns * nxi * neta;
    for (int64_t cc = 0; cc < n_configs; ++cc) {            /* serial: plain sums in a fixed order */
        int64_t c = c_first + cc;
        int itheta = (int)(c % g->ntheta);
        int iy = (int)((c / g->ntheta) % ny), ix = (int)(c / ((int64_t)g->ntheta * ny));
        double theta = 2.0 * MMO_PI * (double)itheta / (double)g->ntheta;
        double ct = cos(theta), st = sin(theta);
        const double *mc = m + (size_t)cc * inner;
        for (int j = 0; j < ns; ++j) {
            double sj = p->s_lo + (j + 0.5) * ds;
            double fx = 0.0, fy = 0.0;
            for (int a = 0; a < nxi; ++a)
                for (int b = 0; b < neta; ++b) {
                    double xi = -R + (a + 0.5) * dxi, eta = -R + (b + 0.5) * deta;
                    double v = mc[((size_t)j * nxi + a) * neta + b];
                    fx += xi * v;
                    fy += eta * v;
                }
            fx *= -k * dxi * deta;
            fy *= -k * dxi * deta;
            /* head position in grid units */
            double gx = ((double)ix / nx + sj * ct) * nx, gy = ((double)iy / ny + sj * st) * ny;
            double bx = floor(gx), by = floor(gy);
            for (int u = -1; u <= 2; ++u)
                for (int v = -1; v <= 2; ++v) {
                    double wx = peskin4(gx - (bx + u)), wy = peskin4(gy - (by + v));
                    long jx = ((long)bx + u) % nx, jy = ((long)by + v) % ny;
                    if (jx < 0) jx += nx;
                    if (jy < 0) jy += ny;
                    double w = dtheta * ds * psi[cc] * wx * wy;
                    F2[((size_t)jx * ny + jy) * 2 + 0] += w * fx;
                    F2[((size_t)jx * ny + jy) * 2 + 1] += w * fy;
                }
        }
    }
    return 0;
}

int mmo_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
