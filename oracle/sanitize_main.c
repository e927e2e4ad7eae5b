/* ORACLE — TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 * Driver that calls every entry point of dbie_oracle.c on small seeded inputs; built together
 * with it under -fsanitize=address,undefined by tests/test_oracle_pins.py (SURVEY section 5:
 * "ASan/UBSan on the oracle").  Exit code 0 = no finding; the numbers are not checked here. */
#include "dbie_oracle.c"
#include <stdio.h>

static unsigned long long lcg = 13061122ULL;
static double rnd(void)
{
    lcg = lcg * 6364136223846793005ULL + 1442695040888963407ULL;
    return (double)(lcg >> 11) / 9007199254740992.0;
}
static double quad3(const double l[3]) { return l[0] * l[0] + 2 * l[1] * l[1] + 3 * l[2] * l[2] + l[0] * l[1]; }

int main(void)
{
    enum { NX = 7, NY = 6, M = 5 };
    double bx[NX * NY], by[NX * NY], bz[NX * NY], x[M], y[M], z[M], lam[3 * M];
    for (int k = 0; k < NX * NY; ++k) { bx[k] = rnd() - .5; by[k] = rnd() - .5; bz[k] = rnd() - .5; }
    for (int i = 0; i < M; ++i) { x[i] = NX * rnd(); y[i] = NY * rnd(); z[i] = 1.0 + 3 * rnd(); }
    for (int i = 0; i < 3 * M; ++i) lam[i] = 0.3 * rnd();
    z[M - 1] = -1.0; /* an invalid point goes through every path too */
    orc_boundary b = { NX, NY, 1.0, 0.0, 0.0, bx, by, bz, NULL, NULL };
    double B[3 * M], G[9 * M], out[9 * M], phi[M], l2[3 * M], resid[2 * M], margin[M];
    int iters[M], status[M], nfev[M];
    orc_eval(&b, M, x, y, z, lam, B, 2);
    orc_gradient(&b, M, x, y, z, lam, B, G, 2);
    for (int analytic = 0; analytic < 2; ++analytic) {
        orc_opts o = { 0, 1e-3, 1.0, 1.0, 1e-3, 1e-4, 0.05, 0.05, 1e-4, 1e-6, 40, 4, 3, 0.4, 1, analytic };
        orc_residual(&b, &o, M, x, y, z, lam, out, phi, 2);
        orc_solve_nm(&b, &o, M, x, y, z, B, l2, resid, iters, status, margin, nfev, phi, 2);
        orc_solve_grid(&b, &o, M, x, y, z, B, l2, resid, iters, status, margin, phi, 2);
        o.n_trial = 3; /* odd T: centre trial = incumbent */
        orc_solve_grid(&b, &o, M, x, y, z, B, l2, resid, iters, status, NULL, NULL, 1);
    }
    /* 9-node staging, odd and even node counts */
    const int nsx = orc_q9_count(NX), nsy = orc_q9_count(NY);
    double *xs = malloc(sizeof(double) * nsx), *ys = malloc(sizeof(double) * nsy);
    double *sx = malloc(sizeof(double) * nsx * nsy), *sy = malloc(sizeof(double) * nsx * nsy),
           *sz = malloc(sizeof(double) * nsx * nsy);
    if (orc_q9_stage(&b, xs, ys, sx, sy, sz) != 0) return 2;
    orc_boundary b9 = { nsx, nsy, 1.0, 0.0, 0.0, sx, sy, sz, xs, ys };
    orc_eval(&b9, M, x, y, z, lam, B, 1);
    free(xs); free(ys); free(sx); free(sy); free(sz);
    /* generic Nelder-Mead driver */
    double sim[12] = { .05, .05, .05, .1, .05, .05, .05, .1, .05, .05, .05, .1 }, trace[3 * 31], fs[12], ff[4], mg;
    int it, nf, st;
    orc_nm_generic(quad3, sim, 1e-7, 1e-9, 30, trace, fs, ff, &it, &nf, &st, &mg);
    printf("sanitize_main ok (%d threads max)\n", orc_max_threads());
    return 0;
}
