/* ===========================================================================
 * ORACLE — TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, obviously-correct CPU implementation of the DBIE hot path of
 * Wang, Yan & Tan (arXiv 1306.1122; /root/reference/PAPER.md), written from
 * the paper.  It shares no code, header, table or constant with the CUDA path
 * (paper_1306_1122_b200/csrc, include/dbie.h) and is used only by tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs.
 *
 * What each function follows:
 *   orc_eval            Eq. 6 discretised as the nodal sum of
 *                       Eq. 16, midpoint rule (reading A-1).
 *   orc_residual        Eq. 8, 9, Eq. 13 frozen-lambda forward
 *                       differences with delta = 1e-3 px,
 *                       Eq. 14 J = curl B.
 *   orc_solve_nm        Downhill Simplex of Nelder & Mead with the
 *                       stopping rule Eq. 10-12.
 *   orc_solve_grid      BASELINE.json config 5 reading (">= 8 trial lambda per
 *                       component per iteration"); NOT in the paper
 *                       (reading O-4).
 *   orc_gradient        O-5 (NOT the paper's default): the nine
 *                       dB_p/dx_j as a second sum over the same pixels, from
 *                       d/dr[n(lambda r)/r^3] = lambda^2 cos(lambda r)/r^2
 *                       - 3 n(lambda r)/r^4 ("possible if the function f_i can be
 *                       calculated analytically").  With
 *                       opts.analytic = 1 orc_residual / orc_solve_nm take J and
 *                       div B from it instead of Eq. 13's differences.
 *   orc_q9_stage        O-6: Eq. 15's 9-node element quadrature
 *                        as a tensor grid of weighted sources;
 *                       every function above then runs on it unchanged.
 *   orc_nm_generic      the same Nelder-Mead driver on a caller-supplied
 *                       objective, so tests can pin it against SciPy (pin S-1).
 *
 * Pins (tests/test_oracle_pins.py): K-1..K-10, S-1..S-4 of DESIGN.md.  The
 * agreement with the paper's OWN numerical output (its element quadrature,
 * thresholds, initial simplex) is "parity unpinned": the paper prints no
 * worked example of Eq. 6.
 *
 * Arithmetic: IEEE double, libm sqrt/sin/cos, products formed in double, sums
 * accumulated in long double (x87 80-bit) in pixel-index order k = 0..N-1.
 * Build: gcc -O2 -ffp-contract=off -fopenmp (never -ffast-math).
 * ======================================================================== */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_PI 3.14159265358979323846264338327950288

typedef struct {
    int nx, ny;                 /* boundary grid, pixel k = iy*nx + ix              */
    double h, x0, y0;           /* pixel size; corner of pixel (0,0)                */
    const double *bx, *by, *bz; /* N = nx*ny each                                   */
    const double *xs, *ys;      /* NULL: sources are the pixel centres (reading A-1).
                                   Else explicit source abscissae xs[nx], ys[ny] of a
                                   tensor grid of weighted sources (O-6, orc_q9_stage) */
} orc_boundary;

typedef struct {
    int method;                 /* 0 = NM, 1 = GRID (informational)                 */
    double delta;               /* FD step as a fraction of h (1e-3)   */
    double cell;                /* d in g_i as a fraction of h (reading A-6)        */
    double w_g;                 /* Phi = f + w_g g (reading A-7)                    */
    double eps_f, eps_g;        /* Eq. 12 thresholds (reading A-8)                  */
    double lam0, step;          /* initial simplex, units 1/h (reading A-9)         */
    double xtol, ftol;          /* simplex tolerances (xtol in 1/h)                 */
    int maxiter;
    int n_trial, n_level;       /* GRID: T, number of levels                        */
    double lam_max;             /* GRID: window [0, lam_max/h]                      */
    int use_eq12;               /* 1: Eq. 12 early exit enabled                     */
    int analytic;               /* 1: analytic gradient of Eq. 6 instead of the
                                   finite differences of Eq. 13 (O-5)               */
} orc_opts;

/* ---------------------------------------------------------------- O-6 ---- */
/* 9-node element quadrature (Eq. 15: "the boundary has
 * been subdivided into N_e 9-nodes elements with boundary data known over each node,
 * N_k(xi, eta) is the shape function, J the Jacobian").  Reading (the paper gives neither
 * the node placement nor the Gauss order): nodes = pixel centres; an element spans
 * 3 x 3 nodes (2h x 2h), biquadratic Lagrange shape functions
 *     N_-1 = xi (xi - 1)/2,  N_0 = 1 - xi^2,  N_+1 = xi (xi + 1)/2   per direction,
 * 3 x 3 Gauss-Legendre points xi = -sqrt(3/5), 0, +sqrt(3/5), weights 5/9, 8/9, 5/9,
 * Jacobian h^2.  When the node count in a direction is even, the last element re-uses the
 * last three nodes and is integrated over its outer half xi in [0, 1] only.  The integral
 * over the boundary is from the first to the last node (the outer half pixel, where the
 * field is assumed to vanish anyway, is dropped).
 * Eq. 15 then reads  B_i = sum over Gauss points g of  K(r_ig) * [w_g sum_j N_j(g) B_j],
 * i.e. the SAME sum as Eq. 16 over a tensor grid of weighted sources.  This function
 * builds that grid: xs[nsx], ys[nsy] and the weighted values (in units of the pixel
 * area h^2, so the prefactor z h^2/2pi of Eq. 6 is unchanged).  nsx = 3 ceil((nx-1)/2). */
static int q9_axis(int n, double c0, double h, double *pos, double *wq, int *base, double (*shape)[3])
{
    /* one direction: for every Gauss abscissa its position, weight, first node and N_a */
    const double g[3] = { -sqrt(0.6), 0.0, sqrt(0.6) }, w[3] = { 5.0 / 9.0, 8.0 / 9.0, 5.0 / 9.0 };
    const int ne = (n - 1 + 1) / 2; /* ceil((n-1)/2) */
    for (int e = 0; e < ne; ++e) {
        const int half = (2 * e + 2 > n - 1);      /* even n: the last element, outer half only */
        const int i0 = half ? n - 3 : 2 * e;
        const double xc = c0 + (i0 + 1 + 0.5) * h; /* centre node of the element */
        for (int q = 0; q < 3; ++q) {
            const double xi = half ? 0.5 + 0.5 * g[q] : g[q];
            const int k = 3 * e + q;
            pos[k] = xc + xi * h;
            wq[k] = half ? 0.5 * w[q] : w[q];
            base[k] = i0;
            shape[k][0] = xi * (xi - 1.0) / 2.0;
            shape[k][1] = 1.0 - xi * xi;
            shape[k][2] = xi * (xi + 1.0) / 2.0;
        }
    }
    return 3 * ne;
}

int orc_q9_count(int n) { return n < 3 ? 0 : 3 * ((n - 1 + 1) / 2); }

/* in: nodal boundary b (nx, ny >= 3).  out: xs[nsx], ys[nsy], sx/sy/sz[nsy*nsx].  Returns 0. */
int orc_q9_stage(const orc_boundary *b, double *xs, double *ys, double *sx, double *sy, double *sz)
{
    if (b->nx < 3 || b->ny < 3) return 1;
    const int nsx = orc_q9_count(b->nx), nsy = orc_q9_count(b->ny);
    double *wx = malloc(sizeof(double) * nsx), *wy = malloc(sizeof(double) * nsy);
    int *bx0 = malloc(sizeof(int) * nsx), *by0 = malloc(sizeof(int) * nsy);
    double (*Nx)[3] = malloc(sizeof(double[3]) * nsx), (*Ny)[3] = malloc(sizeof(double[3]) * nsy);
    q9_axis(b->nx, b->x0, b->h, xs, wx, bx0, Nx);
    q9_axis(b->ny, b->y0, b->h, ys, wy, by0, Ny);
    for (int gy = 0; gy < nsy; ++gy)
        for (int gx = 0; gx < nsx; ++gx) {
            double v[3] = { 0.0, 0.0, 0.0 };
            for (int bb = 0; bb < 3; ++bb)
                for (int a = 0; a < 3; ++a) {
                    const long k = (long)(by0[gy] + bb) * b->nx + bx0[gx] + a;
                    const double N = Ny[gy][bb] * Nx[gx][a];
                    v[0] += N * b->bx[k]; v[1] += N * b->by[k]; v[2] += N * b->bz[k];
                }
            const double w = wy[gy] * wx[gx];
            const long o = (long)gy * nsx + gx;
            sx[o] = w * v[0]; sy[o] = w * v[1]; sz[o] = w * v[2];
        }
    free(wx); free(wy); free(bx0); free(by0); free(Nx); free(Ny);
    return 0;
}

/* ---------------------------------------------------------------- O-1 ---- */
/* B_p(i) = (z_i h^2 / 2 pi) * sum_k [theta sin theta + cos theta] / r^3 * B_p0[k],
 * theta = |lambda_p| r,  r = sqrt((x_k-x_i)^2 + (y_k-y_i)^2 + z_i^2).   Eq. 6/16. */
static void eval_point(const orc_boundary *b, double xi, double yi, double zi,
                       const double lam[3], double B[3])
{
    long double s0 = 0.0L, s1 = 0.0L, s2 = 0.0L;
    const double l0 = fabs(lam[0]), l1 = fabs(lam[1]), l2 = fabs(lam[2]);
    if (!(zi > 0.0) || !isfinite(xi) || !isfinite(yi) || !isfinite(zi) ||
        !isfinite(l0) || !isfinite(l1) || !isfinite(l2)) {
        B[0] = B[1] = B[2] = NAN;
        return;
    }
    for (int iy = 0; iy < b->ny; ++iy) {
        const double yk = b->ys ? b->ys[iy] : b->y0 + (iy + 0.5) * b->h;
        const double dy = yk - yi;
        for (int ix = 0; ix < b->nx; ++ix) {
            const double xk = b->xs ? b->xs[ix] : b->x0 + (ix + 0.5) * b->h;
            const double dx = xk - xi;
            const double r2 = dx * dx + dy * dy + zi * zi;
            const double r = sqrt(r2);
            const double r3 = r2 * r;
            const long k = (long)iy * b->nx + ix;
            double th, a;
            th = l0 * r; a = (th * sin(th) + cos(th)) / r3; s0 += (long double)(a * b->bx[k]);
            th = l1 * r; a = (th * sin(th) + cos(th)) / r3; s1 += (long double)(a * b->by[k]);
            th = l2 * r; a = (th * sin(th) + cos(th)) / r3; s2 += (long double)(a * b->bz[k]);
        }
    }
    const long double c = (long double)zi * (long double)b->h * (long double)b->h /
                          (2.0L * (long double)ORC_PI);
    B[0] = (double)(c * s0);
    B[1] = (double)(c * s1);
    B[2] = (double)(c * s2);
}

void orc_eval(const orc_boundary *b, long M, const double *x, const double *y,
              const double *z, const double *lam /* 3*M, lam[p*M+i] */,
              double *B /* 3*M */, int nthreads)
{
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
#pragma omp parallel for schedule(dynamic, 4)
    for (long i = 0; i < M; ++i) {
        double l[3] = { lam[i], lam[M + i], lam[2 * M + i] }, Bi[3];
        eval_point(b, x[i], y[i], z[i], l, Bi);
        B[i] = Bi[0]; B[M + i] = Bi[1]; B[2 * M + i] = Bi[2];
    }
}

/* ---------------------------------------------------------------- O-2 ---- */
/* out[0..2] = B(r_i); out[3] = f (Eq. 8); out[4] = g (Eq. 9); out[5..7] = J
 * (Eq. 14); out[8] = div B.  Returns Phi = f + w_g g, or NaN for an invalid
 * point (z <= 0, non-finite input, |B| = 0).                                  */
static double residual_from_stencil(const double B0[3], const double Bx[3],
                                    const double By[3], const double Bz[3],
                                    double delta_abs, double d_abs, double w_g,
                                    double out[9])
{
    double G[3][3]; /* G[p][j] = dB_p/dx_j, forward difference, Eq. 13 */
    for (int p = 0; p < 3; ++p) {
        G[p][0] = (Bx[p] - B0[p]) / delta_abs;
        G[p][1] = (By[p] - B0[p]) / delta_abs;
        G[p][2] = (Bz[p] - B0[p]) / delta_abs;
    }
    const double Jx = G[2][1] - G[1][2];
    const double Jy = G[0][2] - G[2][0];
    const double Jz = G[1][0] - G[0][1];
    const double div = G[0][0] + G[1][1] + G[2][2];
    const double nB = sqrt(B0[0] * B0[0] + B0[1] * B0[1] + B0[2] * B0[2]);
    const double nJ = sqrt(Jx * Jx + Jy * Jy + Jz * Jz);
    const double cx = Jy * B0[2] - Jz * B0[1];
    const double cy = Jz * B0[0] - Jx * B0[2];
    const double cz = Jx * B0[1] - Jy * B0[0];
    const double nC = sqrt(cx * cx + cy * cy + cz * cz);
    out[0] = B0[0]; out[1] = B0[1]; out[2] = B0[2];
    out[5] = Jx; out[6] = Jy; out[7] = Jz; out[8] = div;
    if (!(nB > 0.0) || !isfinite(nB)) {
        out[3] = out[4] = NAN;
        return NAN;
    }
    const double f = (nJ <= 1e-300) ? 0.0 : nC / (nJ * nB);
    const double g = fabs(div) * (d_abs / 6.0) / nB;
    out[3] = f; out[4] = g;
    return f + w_g * g;
}

/* ---------------------------------------------------------------- O-5 ---- */
/* Analytic gradient (PAPER.md:92 allows it, Eq. 13 is the default).
 * With K(r) = n(lambda r)/r^3, n = theta sin theta + cos theta, theta = lambda r:
 *   dK/dr = lambda^2 cos(theta)/r^2 - 3 n/r^4,   D(r) := (dK/dr)/r,
 *   r^2 = (x_k-x_i)^2 + (y_k-y_i)^2 + z_i^2  =>  dr/dx_i = -(x_k-x_i)/r, dr/dz_i = z_i/r,
 *   B_p    = (z h^2/2pi) sum_k K B_p0
 *   dB_p/dx = -(z h^2/2pi) sum_k D (x_k-x_i) B_p0      (same for y)
 *   dB_p/dz =  (h^2/2pi) [ sum_k K B_p0 + z^2 sum_k D B_p0 ].
 * G[p][j] = dB_p/dx_j.                                                        */
static void eval_point_grad(const orc_boundary *b, double xi, double yi, double zi,
                            const double lam[3], double B[3], double G[3][3])
{
    long double s0[3] = { 0, 0, 0 }, sx[3] = { 0, 0, 0 }, sy[3] = { 0, 0, 0 }, sd[3] = { 0, 0, 0 };
    const double l[3] = { fabs(lam[0]), fabs(lam[1]), fabs(lam[2]) };
    if (!(zi > 0.0) || !isfinite(xi) || !isfinite(yi) || !isfinite(zi) ||
        !isfinite(l[0]) || !isfinite(l[1]) || !isfinite(l[2])) {
        for (int p = 0; p < 3; ++p) { B[p] = NAN; G[p][0] = G[p][1] = G[p][2] = NAN; }
        return;
    }
    for (int iy = 0; iy < b->ny; ++iy) {
        const double yk = b->ys ? b->ys[iy] : b->y0 + (iy + 0.5) * b->h;
        const double dy = yk - yi;
        for (int ix = 0; ix < b->nx; ++ix) {
            const double xk = b->xs ? b->xs[ix] : b->x0 + (ix + 0.5) * b->h;
            const double dx = xk - xi;
            const double r2 = dx * dx + dy * dy + zi * zi;
            const double r = sqrt(r2);
            const double r3 = r2 * r, r5 = r3 * r2;
            const long k = (long)iy * b->nx + ix;
            const double b0[3] = { b->bx[k], b->by[k], b->bz[k] };
            for (int p = 0; p < 3; ++p) {
                const double th = l[p] * r, sn = sin(th), cs = cos(th);
                const double n = th * sn + cs;
                const double K = n / r3;
                const double D = l[p] * l[p] * cs / r3 - 3.0 * n / r5;
                s0[p] += (long double)(K * b0[p]);
                sx[p] += (long double)(D * dx * b0[p]);
                sy[p] += (long double)(D * dy * b0[p]);
                sd[p] += (long double)(D * b0[p]);
            }
        }
    }
    const long double c1 = (long double)b->h * (long double)b->h / (2.0L * (long double)ORC_PI);
    const long double c = (long double)zi * c1;
    for (int p = 0; p < 3; ++p) {
        B[p] = (double)(c * s0[p]);
        G[p][0] = (double)(-c * sx[p]);
        G[p][1] = (double)(-c * sy[p]);
        G[p][2] = (double)(c1 * (s0[p] + (long double)zi * (long double)zi * sd[p]));
    }
}

/* Eq. 14, 8, 9 from a given gradient: the tail of residual_from_stencil, same formulas. */
static double residual_from_gradient(const double B0[3], const double G[3][3], double d_abs,
                                     double w_g, double out[9])
{
    const double Jx = G[2][1] - G[1][2];
    const double Jy = G[0][2] - G[2][0];
    const double Jz = G[1][0] - G[0][1];
    const double div = G[0][0] + G[1][1] + G[2][2];
    const double nB = sqrt(B0[0] * B0[0] + B0[1] * B0[1] + B0[2] * B0[2]);
    const double nJ = sqrt(Jx * Jx + Jy * Jy + Jz * Jz);
    const double cx = Jy * B0[2] - Jz * B0[1];
    const double cy = Jz * B0[0] - Jx * B0[2];
    const double cz = Jx * B0[1] - Jy * B0[0];
    const double nC = sqrt(cx * cx + cy * cy + cz * cz);
    out[0] = B0[0]; out[1] = B0[1]; out[2] = B0[2];
    out[5] = Jx; out[6] = Jy; out[7] = Jz; out[8] = div;
    if (!(nB > 0.0) || !isfinite(nB)) {
        out[3] = out[4] = NAN;
        return NAN;
    }
    const double f = (nJ <= 1e-300) ? 0.0 : nC / (nJ * nB);
    const double g = fabs(div) * (d_abs / 6.0) / nB;
    out[3] = f; out[4] = g;
    return f + w_g * g;
}

void orc_gradient(const orc_boundary *b, long M, const double *x, const double *y,
                  const double *z, const double *lam /* 3*M */, double *B /* 3*M */,
                  double *G /* 9*M: G[(p*3+j)*M + i] = dB_p/dx_j */, int nthreads)
{
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
#pragma omp parallel for schedule(dynamic, 4)
    for (long i = 0; i < M; ++i) {
        double l[3] = { lam[i], lam[M + i], lam[2 * M + i] }, Bi[3], Gi[3][3];
        eval_point_grad(b, x[i], y[i], z[i], l, Bi, Gi);
        for (int p = 0; p < 3; ++p) {
            B[p * M + i] = Bi[p];
            for (int j = 0; j < 3; ++j) G[(p * 3 + j) * M + i] = Gi[p][j];
        }
    }
}

typedef struct {
    const orc_boundary *b;
    double xi, yi, zi;
    double delta_abs, d_abs, w_g;
    long nfev;
    int analytic;
} point_ctx;

/* objective of the per-point search: lambda triple -> Phi; aux = (B, f, g, J, div) */
static double point_objective(const double lam[3], void *user, double aux[9])
{
    point_ctx *c = (point_ctx *)user;
    double B0[3], Bx[3], By[3], Bz[3];
    c->nfev++;
    if (c->analytic) { /* O-5: one evaluation position, exact derivatives */
        double G[3][3];
        eval_point_grad(c->b, c->xi, c->yi, c->zi, lam, B0, G);
        return residual_from_gradient(B0, G, c->d_abs, c->w_g, aux);
    }
    /* Eq. 13: the same lambda triple at r_i and at its delta-neighbours */
    eval_point(c->b, c->xi, c->yi, c->zi, lam, B0);
    eval_point(c->b, c->xi + c->delta_abs, c->yi, c->zi, lam, Bx);
    eval_point(c->b, c->xi, c->yi + c->delta_abs, c->zi, lam, By);
    eval_point(c->b, c->xi, c->yi, c->zi + c->delta_abs, lam, Bz);
    return residual_from_stencil(B0, Bx, By, Bz, c->delta_abs, c->d_abs, c->w_g, aux);
}

void orc_residual(const orc_boundary *b, const orc_opts *o, long M, const double *x,
                  const double *y, const double *z, const double *lam /* 3*M */,
                  double *out /* 9*M: out[q*M+i], q as in residual_from_stencil */,
                  double *phi /* M */, int nthreads)
{
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
#pragma omp parallel for schedule(dynamic, 1)
    for (long i = 0; i < M; ++i) {
        point_ctx c = { b, x[i], y[i], z[i], o->delta * b->h, o->cell * b->h, o->w_g, 0, o->analytic };
        double l[3] = { lam[i], lam[M + i], lam[2 * M + i] }, aux[9];
        phi[i] = point_objective(l, &c, aux);
        for (int q = 0; q < 9; ++q) out[q * M + i] = aux[q];
    }
}

/* ---------------------------------------------------------------- O-3 ---- */
/* Nelder & Mead (1965) in the Lagarias et al. (1998) ordering, coefficients
 * rho = 1, chi = 2, psi = 1/2, sigma = 1/2 (reading A-9).  The vertex formulas
 * are written as (1+rho) xbar - rho x_worst etc. so that the sequence can be
 * pinned against SciPy's non-adaptive Nelder-Mead bit for bit (pin S-1).      */
typedef double (*orc_objective)(const double lam[3], void *user, double aux[9]);

typedef struct {
    double V[4][3], F[4], aux[4][9];
    int iters, status, nfev;
    double margin; /* smallest |a-b| over every comparison a<b taken (protocol P-4) */
} nm_state;

static double as_inf(double v) { return isnan(v) ? INFINITY : v; }

static void note_margin(nm_state *s, double a, double b)
{
    double d = fabs(a - b);
    if (isfinite(d) && d < s->margin) s->margin = d;
}

static void nm_sort(nm_state *s)
{
    /* stable insertion sort, ascending Phi; ties keep the earlier index first */
    for (int i = 1; i < 4; ++i) {
        double v[3], f = s->F[i], a[9];
        memcpy(v, s->V[i], sizeof v); memcpy(a, s->aux[i], sizeof a);
        int j = i - 1;
        while (j >= 0 && s->F[j] > f) {
            memcpy(s->V[j + 1], s->V[j], sizeof v);
            memcpy(s->aux[j + 1], s->aux[j], sizeof a);
            s->F[j + 1] = s->F[j];
            --j;
        }
        memcpy(s->V[j + 1], v, sizeof v); memcpy(s->aux[j + 1], a, sizeof a);
        s->F[j + 1] = f;
    }
    for (int i = 0; i < 4; ++i)
        for (int j = i + 1; j < 4; ++j) note_margin(s, s->F[i], s->F[j]);
}

static void nm_replace_worst(nm_state *s, const double v[3], double f, const double a[9])
{
    memcpy(s->V[3], v, 3 * sizeof(double));
    memcpy(s->aux[3], a, 9 * sizeof(double));
    s->F[3] = f;
}

static void nm_minimise(orc_objective obj, void *user, const double V0[4][3],
                        double xtol_abs, double ftol, int maxiter, int use_eq12,
                        double eps_f, double eps_g, nm_state *s,
                        double *trace /* (maxiter+1)*3 best vertex per iteration, or NULL */)
{
    s->iters = 0; s->nfev = 0; s->status = 2; s->margin = INFINITY;
    for (int j = 0; j < 4; ++j) {
        memcpy(s->V[j], V0[j], 3 * sizeof(double));
        s->F[j] = as_inf(obj(s->V[j], user, s->aux[j]));
        s->nfev++;
    }
    nm_sort(s);
    if (trace) memcpy(trace, s->V[0], 3 * sizeof(double));
    while (s->iters < maxiter) {
        /* Eq. 12: f <= eps_f and g <= eps_g at the best vertex */
        if (use_eq12) {
            note_margin(s, s->aux[0][3], eps_f);
            note_margin(s, s->aux[0][4], eps_g);
            if (s->aux[0][3] <= eps_f && s->aux[0][4] <= eps_g) { s->status = 0; return; }
        }
        double dx = 0.0, df = 0.0;
        for (int j = 1; j < 4; ++j) {
            for (int p = 0; p < 3; ++p) dx = fmax(dx, fabs(s->V[j][p] - s->V[0][p]));
            df = fmax(df, fabs(s->F[0] - s->F[j]));
        }
        note_margin(s, df, ftol);
        if (dx <= xtol_abs && df <= ftol) { s->status = 1; return; }

        double xbar[3], xr[3], xt[3], ar[9], at[9], fr, ft;
        for (int p = 0; p < 3; ++p) xbar[p] = ((s->V[0][p] + s->V[1][p]) + s->V[2][p]) / 3.0;
        for (int p = 0; p < 3; ++p) xr[p] = 2.0 * xbar[p] - 1.0 * s->V[3][p];
        fr = as_inf(obj(xr, user, ar)); s->nfev++;
        int shrink = 0;
        note_margin(s, fr, s->F[0]);
        if (fr < s->F[0]) {
            for (int p = 0; p < 3; ++p) xt[p] = 3.0 * xbar[p] - 2.0 * s->V[3][p];
            ft = as_inf(obj(xt, user, at)); s->nfev++;
            note_margin(s, ft, fr);
            if (ft < fr) nm_replace_worst(s, xt, ft, at);
            else nm_replace_worst(s, xr, fr, ar);
        } else {
            note_margin(s, fr, s->F[2]);
            if (fr < s->F[2]) {
                nm_replace_worst(s, xr, fr, ar);
            } else {
                note_margin(s, fr, s->F[3]);
                if (fr < s->F[3]) { /* outside contraction */
                    for (int p = 0; p < 3; ++p) xt[p] = 1.5 * xbar[p] - 0.5 * s->V[3][p];
                    ft = as_inf(obj(xt, user, at)); s->nfev++;
                    note_margin(s, ft, fr);
                    if (ft <= fr) nm_replace_worst(s, xt, ft, at);
                    else shrink = 1;
                } else {            /* inside contraction */
                    for (int p = 0; p < 3; ++p) xt[p] = 0.5 * xbar[p] + 0.5 * s->V[3][p];
                    ft = as_inf(obj(xt, user, at)); s->nfev++;
                    note_margin(s, ft, s->F[3]);
                    if (ft < s->F[3]) nm_replace_worst(s, xt, ft, at);
                    else shrink = 1;
                }
                if (shrink) {
                    for (int j = 1; j < 4; ++j) {
                        for (int p = 0; p < 3; ++p)
                            s->V[j][p] = s->V[0][p] + 0.5 * (s->V[j][p] - s->V[0][p]);
                        s->F[j] = as_inf(obj(s->V[j], user, s->aux[j])); s->nfev++;
                    }
                }
            }
        }
        nm_sort(s);
        s->iters++;
        if (trace) memcpy(trace + 3 * s->iters, s->V[0], 3 * sizeof(double));
    }
    s->status = 2;
}

/* generic driver for pin S-1 (objective supplied by the test) */
typedef double (*orc_objective3)(const double lam[3]);
static double generic_adapter(const double lam[3], void *user, double aux[9])
{
    for (int q = 0; q < 9; ++q) aux[q] = 0.0;
    return ((orc_objective3)user)(lam);
}
void orc_nm_generic(orc_objective3 fn, const double *simplex /* 4*3 */, double xtol,
                    double ftol, int maxiter, double *trace /* (maxiter+1)*3 */,
                    double *final_simplex /* 12 */, double *final_f /* 4 */,
                    int *iters, int *nfev, int *status, double *margin /* 1 or NULL */)
{
    nm_state s;
    double V0[4][3];
    memcpy(V0, simplex, sizeof V0);
    nm_minimise(generic_adapter, (void *)fn, V0, xtol, ftol, maxiter, 0, 0.0, 0.0, &s, trace);
    memcpy(final_simplex, s.V, sizeof s.V);
    memcpy(final_f, s.F, sizeof s.F);
    *iters = s.iters; *nfev = s.nfev; *status = s.status;
    if (margin) *margin = s.margin;
}

void orc_solve_nm(const orc_boundary *b, const orc_opts *o, long M, const double *x,
                  const double *y, const double *z,
                  double *B /* 3*M */, double *lam /* 3*M, >= 0 */,
                  double *resid /* 2*M: f, g */, int *iters, int *status,
                  double *margin /* M or NULL */, int *nfev /* M or NULL */,
                  double *phi /* M or NULL */, int nthreads)
{
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
#pragma omp parallel for schedule(dynamic, 1)
    for (long i = 0; i < M; ++i) {
        point_ctx c = { b, x[i], y[i], z[i], o->delta * b->h, o->cell * b->h, o->w_g, 0, o->analytic };
        nm_state s;
        double V0[4][3];
        const double l0 = o->lam0 / b->h, st = o->step / b->h;
        for (int j = 0; j < 4; ++j)
            for (int p = 0; p < 3; ++p) V0[j][p] = l0;
        for (int j = 1; j < 4; ++j) V0[j][j - 1] = l0 + st;
        int invalid = !(z[i] > 0.0) || !isfinite(x[i]) || !isfinite(y[i]) || !isfinite(z[i]);
        if (!invalid) {
            nm_minimise(point_objective, &c, V0, o->xtol / b->h, o->ftol, o->maxiter,
                        o->use_eq12, o->eps_f, o->eps_g, &s, NULL);
            if (!isfinite(s.F[0])) invalid = 1;
        }
        if (invalid) {
            for (int p = 0; p < 3; ++p) { B[p * M + i] = NAN; lam[p * M + i] = NAN; }
            resid[i] = resid[M + i] = NAN;
            iters[i] = 0; status[i] = 3;
            if (margin) margin[i] = 0.0;
            if (nfev) nfev[i] = 0;
            if (phi) phi[i] = NAN;
            continue;
        }
        for (int p = 0; p < 3; ++p) {
            B[p * M + i] = s.aux[0][p];
            lam[p * M + i] = fabs(s.V[0][p]);
        }
        resid[i] = s.aux[0][3]; resid[M + i] = s.aux[0][4];
        iters[i] = s.iters; status[i] = s.status;
        if (margin) margin[i] = s.margin;
        if (nfev) nfev[i] = s.nfev;
        if (phi) phi[i] = s.F[0];
    }
}

/* ---------------------------------------------------------------- O-4 ---- */
/* GRID search: T trial values per component per level, using separability
 * (B_p depends on lambda_p only).  BASELINE.json config 5 reading,
 * not in the paper.                                                          */
void orc_solve_grid(const orc_boundary *b, const orc_opts *o, long M, const double *x,
                    const double *y, const double *z,
                    double *B, double *lam, double *resid, int *iters, int *status,
                    double *margin /* M or NULL */, double *phi /* M or NULL */,
                    int nthreads)
{
    const int T = o->n_trial;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
#pragma omp parallel for schedule(dynamic, 1)
    for (long i = 0; i < M; ++i) {
        const double da = o->delta * b->h, dc = o->cell * b->h;
        const double Lmax = o->lam_max / b->h;
        /* S[t][s][p]: component p at stencil position s (0, +x, +y, +z) for trial t;
         * slot T is the incumbent */
        double (*S)[4][3] = malloc(sizeof(double[4][3]) * (T + 1));
        /* O-5 (opts.analytic): per candidate value B and the analytic gradient instead of the stencil */
        double (*Bt)[3] = malloc(sizeof(double[3]) * (T + 1));
        double (*Gt)[3][3] = malloc(sizeof(double[3][3]) * (T + 1));
        double *lt = malloc(sizeof(double) * 3 * (T + 1)); /* lt[p*(T+1)+t] */
        double lo[3] = { 0.0, 0.0, 0.0 }, W = Lmax;
        double best_phi = INFINITY, best_aux[9], mrg = INFINITY;
        int have_inc = 0, st = 2, lev = 0;
        int invalid = !(z[i] > 0.0) || !isfinite(x[i]) || !isfinite(y[i]) || !isfinite(z[i]);
        for (lev = 0; lev < o->n_level && !invalid; ++lev) {
            for (int t = 0; t < T; ++t) {
                double l[3];
                for (int p = 0; p < 3; ++p) {
                    l[p] = lo[p] + W * (double)t / (double)(T - 1);
                    lt[p * (T + 1) + t] = l[p];
                }
                if (o->analytic) { eval_point_grad(b, x[i], y[i], z[i], l, Bt[t], Gt[t]); continue; }
                eval_point(b, x[i], y[i], z[i], l, S[t][0]);
                eval_point(b, x[i] + da, y[i], z[i], l, S[t][1]);
                eval_point(b, x[i], y[i] + da, z[i], l, S[t][2]);
                eval_point(b, x[i], y[i], z[i] + da, l, S[t][3]);
            }
            const int C = have_inc ? T + 1 : T;
            int bt[3] = { -1, -1, -1 };
            double lev_best = INFINITY, lev_second = INFINITY, lev_aux[9];
            for (int tx = 0; tx < C; ++tx)
                for (int ty = 0; ty < C; ++ty)
                    for (int tz = 0; tz < C; ++tz) {
                        const int tt[3] = { tx, ty, tz };
                        double P0[3], Px[3], Py[3], Pz[3], aux[9];
                        double ph;
                        if (o->analytic) { /* the stencil table S is not filled in this mode */
                            double Gc[3][3];
                            for (int p = 0; p < 3; ++p) {
                                P0[p] = Bt[tt[p]][p];
                                for (int j = 0; j < 3; ++j) Gc[p][j] = Gt[tt[p]][p][j];
                            }
                            ph = as_inf(residual_from_gradient(P0, Gc, dc, o->w_g, aux));
                        } else {
                            for (int p = 0; p < 3; ++p) {
                                P0[p] = S[tt[p]][0][p]; Px[p] = S[tt[p]][1][p];
                                Py[p] = S[tt[p]][2][p]; Pz[p] = S[tt[p]][3][p];
                            }
                            ph = as_inf(residual_from_stencil(P0, Px, Py, Pz, da, dc,
                                                              o->w_g, aux));
                        }
                        if (ph < lev_best) { /* strict: ties keep the lexicographically first */
                            lev_second = lev_best;
                            lev_best = ph; bt[0] = tx; bt[1] = ty; bt[2] = tz;
                            memcpy(lev_aux, aux, sizeof aux);
                        } else if (ph < lev_second) lev_second = ph;
                    }
            if (bt[0] < 0) { invalid = 1; break; }
            if (isfinite(lev_second - lev_best) && lev_second - lev_best < mrg)
                mrg = lev_second - lev_best;
            /* the argmin becomes the incumbent (slot T) */
            double inc[4][3], il[3];
            for (int p = 0; p < 3; ++p) il[p] = lt[p * (T + 1) + bt[p]];
            if (!o->analytic) {
                for (int p = 0; p < 3; ++p)
                    for (int s = 0; s < 4; ++s) inc[s][p] = S[bt[p]][s][p];
                memcpy(S[T], inc, sizeof inc);
            } else
                for (int p = 0; p < 3; ++p) {
                    Bt[T][p] = Bt[bt[p]][p];
                    for (int j = 0; j < 3; ++j) Gt[T][p][j] = Gt[bt[p]][p][j];
                }
            for (int p = 0; p < 3; ++p) lt[p * (T + 1) + T] = il[p];
            have_inc = 1;
            best_phi = lev_best; memcpy(best_aux, lev_aux, sizeof lev_aux);
            if (o->use_eq12 && best_aux[3] <= o->eps_f && best_aux[4] <= o->eps_g) {
                st = 0; ++lev; break;
            }
            /* next window centred on the incumbent, clipped to [0, Lmax] */
            const double Wn = 2.0 * W / (double)(T - 1);
            for (int p = 0; p < 3; ++p) {
                double l = il[p] - 0.5 * Wn;
                if (l < 0.0) l = 0.0;
                if (l + Wn > Lmax) l = Lmax - Wn;
                lo[p] = l;
            }
            W = Wn;
            st = 1;
        }
        if (invalid || !isfinite(best_phi)) {
            for (int p = 0; p < 3; ++p) { B[p * M + i] = NAN; lam[p * M + i] = NAN; }
            resid[i] = resid[M + i] = NAN; iters[i] = 0; status[i] = 3;
            if (margin) margin[i] = 0.0;
            if (phi) phi[i] = NAN;
        } else {
            for (int p = 0; p < 3; ++p) {
                B[p * M + i] = best_aux[p];
                lam[p * M + i] = fabs(lt[p * (T + 1) + T]);
            }
            resid[i] = best_aux[3]; resid[M + i] = best_aux[4];
            iters[i] = lev; status[i] = st;
            if (margin) margin[i] = mrg;
            if (phi) phi[i] = best_phi;
        }
        free(S); free(lt); free(Bt); free(Gt);
    }
}

int orc_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
