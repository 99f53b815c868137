/* mm_inputs/gen.c -- seeded synthetic inputs for the bound-motor microscale step.
 *
 * This module holds the INPUT RECIPE only (BASELINE.json
 * configs[0]: "initial density = U[0,1) (mt19937_64 seed 1) x exp(-(xi^2+eta^2)/(2(R/2)^2));
 * U,V ~ U[-0.5,0.5], Omega ~ U[-1,1] per (x,y,theta)").  It contains none of the
 * method's arithmetic (no fluxes, no rates, no moments) and is the one piece of code
 * that both the oracle-side tests and the CUDA-side harness may call.
 *
 * Generator: the 64-bit Mersenne Twister of Matsumoto & Nishimura (the algorithm that
 * C++ names std::mt19937_64), restated here from its published definition.
 * Real from raw: u = (g() >> 11) * 2^-53 in [0,1).
 *
 * Draw order (one engine per data set, seeded once):
 *   1. for c = 0..Nc-1:  U_c = u - 1/2, V_c = u - 1/2, Omega_c = omega_max*(2u - 1)
 *   2. for every cell in canonical order (c slowest, then j, a, b; b fastest; cells
 *      outside the disc included so the stream position is layout independent):
 *         m0 = u * exp(-(xi_a^2+eta_b^2)/(2 (R/2)^2)) * inside(a,b)
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>

#define NN 312
#define MM 156

typedef struct {
    uint64_t mt[NN];
    int idx;
} mmi_engine;

static void engine_seed(mmi_engine *g, uint64_t seed)
{
    g->mt[0] = seed;
    for (int i = 1; i < NN; ++i)
        g->mt[i] = 6364136223846793005ULL * (g->mt[i - 1] ^ (g->mt[i - 1] >> 62)) + (uint64_t)i;
    g->idx = NN;
}

static void engine_refill(mmi_engine *g)
{
    const uint64_t UM = 0xFFFFFFFF80000000ULL, LM = 0x7FFFFFFFULL, A = 0xB5026F5AA96619E9ULL;
    uint64_t *mt = g->mt;
    int i;
    for (i = 0; i < NN - MM; ++i) {
        uint64_t x = (mt[i] & UM) | (mt[i + 1] & LM);
        mt[i] = mt[i + MM] ^ (x >> 1) ^ ((x & 1ULL) ? A : 0ULL);
    }
    for (; i < NN - 1; ++i) {
        uint64_t x = (mt[i] & UM) | (mt[i + 1] & LM);
        mt[i] = mt[i + (MM - NN)] ^ (x >> 1) ^ ((x & 1ULL) ? A : 0ULL);
    }
    {
        uint64_t x = (mt[NN - 1] & UM) | (mt[0] & LM);
        mt[NN - 1] = mt[MM - 1] ^ (x >> 1) ^ ((x & 1ULL) ? A : 0ULL);
    }
    g->idx = 0;
}

static inline uint64_t engine_next(mmi_engine *g)
{
    if (g->idx >= NN) engine_refill(g);
    uint64_t x = g->mt[g->idx++];
    x ^= (x >> 29) & 0x5555555555555555ULL;
    x ^= (x << 17) & 0x71D67FFFEDA60000ULL;
    x ^= (x << 37) & 0xFFF7EEE000000000ULL;
    x ^= (x >> 43);
    return x;
}

static inline double engine_unit(mmi_engine *g)
{
    return (double)(engine_next(g) >> 11) * (1.0 / 9007199254740992.0);
}

/* ---- public C entry points (called through ctypes) ---------------------------- */

mmi_engine *mmi_open(uint64_t seed)
{
    mmi_engine *g = (mmi_engine *)malloc(sizeof(mmi_engine));
    if (g) engine_seed(g, seed);
    return g;
}

void mmi_close(mmi_engine *g) { free(g); }

uint64_t mmi_raw(mmi_engine *g) { return engine_next(g); }

void mmi_skip(mmi_engine *g, uint64_t n)
{
    for (uint64_t i = 0; i < n; ++i) (void)engine_next(g);
}

/* step 1 of the draw order: 3 consecutive draws per configuration */
void mmi_draw_velocities(mmi_engine *g, int64_t nc, double omega_max,
                         double *U, double *V, double *Om)
{
    for (int64_t c = 0; c < nc; ++c) {
        U[c] = engine_unit(g) - 0.5;
        V[c] = engine_unit(g) - 0.5;
        Om[c] = omega_max * (2.0 * engine_unit(g) - 1.0);
    }
}

/* exact integer disc test, xi_a^2 + eta_b^2 <= R^2 with cell centres
 * xi_a = -R + (a+1/2) 2R/nxi */
int mmi_inside(int a, int b, int nxi, int neta)
{
    int64_t p = 2 * (int64_t)a + 1 - nxi, q = 2 * (int64_t)b + 1 - neta;
    int64_t lhs = p * p * (int64_t)neta * neta + q * q * (int64_t)nxi * nxi;
    return lhs <= (int64_t)nxi * nxi * (int64_t)neta * neta;
}

/* step 2 of the draw order for n_configs consecutive configurations, continuing from
 * the engine's current position.  as_float != 0 writes float (round to nearest). */
int mmi_draw_density(mmi_engine *g, int64_t n_configs, int ns, int nxi, int neta,
                     double R, int mask_disc, int as_float, void *out)
{
    const int plane = nxi * neta;
    double *env = (double *)malloc(sizeof(double) * (size_t)plane);
    if (!env) return -1;
    const double dxi = 2.0 * R / nxi, deta = 2.0 * R / neta, sig = 0.5 * R;
    for (int a = 0; a < nxi; ++a)
        for (int b = 0; b < neta; ++b) {
            double xi = -R + (a + 0.5) * dxi, eta = -R + (b + 0.5) * deta;
            double e = exp(-(xi * xi + eta * eta) / (2.0 * sig * sig));
            if (mask_disc && !mmi_inside(a, b, nxi, neta)) e = 0.0;
            env[a * neta + b] = e;
        }
    const int64_t per_config = (int64_t)ns * plane;
    double *od = (double *)out;
    float *of = (float *)out;
    for (int64_t c = 0; c < n_configs; ++c)
        for (int j = 0; j < ns; ++j)
            for (int p = 0; p < plane; ++p) {
                double v = engine_unit(g) * env[p];
                int64_t i = c * per_config + (int64_t)j * plane + p;
                if (as_float) of[i] = (float)v; else od[i] = v;
            }
    free(env);
    return 0;
}
