// dbie_nm.cuh — per-point arithmetic of the lambda search:
//   residual_from_sums : Eq. 13 forward differences -> J (Eq. 14), div B, f (Eq. 8), g (Eq. 9),
//                        Phi = f + w_g g
//   nm_advance         : Downhill Simplex of Nelder & Mead as a resumable state
//                        machine: one call consumes the objective value of the one outstanding
//                        trial point and either finishes the point (Eq. 10-12)
//                        or names the next trial point.  Lagarias et al. ordering, coefficients
//                        rho=1, chi=2, psi=1/2, sigma=1/2 (reading A-9).
// Every product and sum is a separately rounded IEEE operation (no FMA contraction): the
// decisions are chains of floating-point comparisons, and the formulas below are the ones
// DESIGN.md section 3 (O-2, O-3) fixes.  __host__ __device__ so the host test shim
// (host_shim.cpp, tests/test_device_math_host.py) can drive the same code against SciPy.
#pragma once
#include <math.h>

#if defined(__CUDACC__)
#define DBIE_NM_HD __host__ __device__ __forceinline__
#else
#define DBIE_NM_HD inline
#endif

namespace dbie {

#if defined(__CUDA_ARCH__)
DBIE_NM_HD double mul_(double a, double b) { return __dmul_rn(a, b); }
DBIE_NM_HD double add_(double a, double b) { return __dadd_rn(a, b); }
DBIE_NM_HD double sub_(double a, double b) { return __dsub_rn(a, b); }
DBIE_NM_HD double div_(double a, double b) { return __ddiv_rn(a, b); }
DBIE_NM_HD double sqrt_(double a) { return __dsqrt_rn(a); }
#else
// host build: compiled with -ffp-contract=off
DBIE_NM_HD double mul_(double a, double b) { return a * b; }
DBIE_NM_HD double add_(double a, double b) { return a + b; }
DBIE_NM_HD double sub_(double a, double b) { return a - b; }
DBIE_NM_HD double div_(double a, double b) { return a / b; }
DBIE_NM_HD double sqrt_(double a) { return sqrt(a); }
#endif

struct NMConsts {
    double delta_abs;   // finite-difference step, length units
    double d_abs;       // cell size d in g_i (reading A-6)
    double w_g;         // Phi = f + w_g g (reading A-7)
    double eps_f, eps_g;
    double xtol_abs, ftol;
    double lam0_abs, step_abs;
    double h2_over_2pi;  // h^2 / (2 pi): Eq. 6 prefactor without z_i
    int maxiter, use_eq12;
    int analytic;        // 1: sums are those of the analytic gradient (O-5), not of the Eq. 13 stencil
};

struct Residual {
    double B[3], f, g, J[3], div, phi;
};

DBIE_NM_HD double norm3_(double a, double b, double c) {
    return sqrt_(add_(add_(mul_(a, a), mul_(b, b)), mul_(c, c)));
}

// Gradient G[p][j] = dB_p/dx_j (Eq. 13 forward differences) and B at r_i -> J (Eq. 14), div B,
// f (Eq. 8), g (Eq. 9), Phi.  Split from the differencing so that GRID mode can form each
// component's three differences once per trial value (they depend on lambda_p only).
DBIE_NM_HD Residual residual_from_gradient(const double G[3][3], const double B0[3], const NMConsts& k) {
    Residual r;
    r.J[0] = sub_(G[2][1], G[1][2]);
    r.J[1] = sub_(G[0][2], G[2][0]);
    r.J[2] = sub_(G[1][0], G[0][1]);
    r.div = add_(add_(G[0][0], G[1][1]), G[2][2]);
    for (int p = 0; p < 3; ++p) r.B[p] = B0[p];
    const double nB = norm3_(r.B[0], r.B[1], r.B[2]);
    const double nJ = norm3_(r.J[0], r.J[1], r.J[2]);
    const double cx = sub_(mul_(r.J[1], r.B[2]), mul_(r.J[2], r.B[1]));
    const double cy = sub_(mul_(r.J[2], r.B[0]), mul_(r.J[0], r.B[2]));
    const double cz = sub_(mul_(r.J[0], r.B[1]), mul_(r.J[1], r.B[0]));
    const double nC = norm3_(cx, cy, cz);
    if (!(nB > 0.0) || !isfinite(nB)) {
        r.f = r.g = r.phi = NAN;
        return r;
    }
    r.f = (nJ <= 1e-300) ? 0.0 : div_(nC, mul_(nJ, nB));                 // Eq. 8
    r.g = div_(mul_(fabs(r.div), div_(k.d_abs, 6.0)), nB);               // Eq. 9, dV/dsigma = d/6
    r.phi = add_(r.f, mul_(k.w_g, r.g));
    return r;
}

// B at the four stencil positions -> f, g, J, div, Phi.  Bs[s][p], s: 0 = r_i, 1 = +delta x,
// 2 = +delta y, 3 = +delta z, all with the same lambda triple (Eq. 13).
DBIE_NM_HD Residual residual_from_stencil(const double Bs[4][3], const NMConsts& k) {
    double G[3][3];  // G[p][j] = dB_p/dx_j
    for (int p = 0; p < 3; ++p)
        for (int j = 0; j < 3; ++j) G[p][j] = div_(sub_(Bs[j + 1][p], Bs[0][p]), k.delta_abs);
    return residual_from_gradient(G, Bs[0], k);
}

// raw sums S[s*3+p] (Eq. 16 without the prefactor) -> B at the stencil -> residual
DBIE_NM_HD Residual residual_from_sums(const double S[12], double z, const NMConsts& k) {
    double Bs[4][3];
    const double c0 = mul_(z, k.h2_over_2pi);
    const double c3 = mul_(add_(z, k.delta_abs), k.h2_over_2pi);
    for (int s = 0; s < 4; ++s)
        for (int p = 0; p < 3; ++p) Bs[s][p] = mul_(s == 3 ? c3 : c0, S[s * 3 + p]);
    return residual_from_stencil(Bs, k);
}

// raw sums of the analytic-gradient mode (O-5): S[p] = sum K b_p, S[3+p] = sum D dx b_p,
// S[6+p] = sum D dy b_p, S[9+p] = sum D b_p  ->  B_p = c S[p], dB_p/dx = -c S[3+p], dB_p/dy = -c S[6+p],
// dB_p/dz = (h^2/2pi) (S[p] + z^2 S[9+p]), c = z h^2/2pi.
DBIE_NM_HD Residual residual_from_analytic_sums(const double S[12], double z, const NMConsts& k) {
    const double c = mul_(z, k.h2_over_2pi);
    const double zz = mul_(z, z);
    double G[3][3], B0[3];
    for (int p = 0; p < 3; ++p) {
        B0[p] = mul_(c, S[p]);
        G[p][0] = -mul_(c, S[3 + p]);
        G[p][1] = -mul_(c, S[6 + p]);
        G[p][2] = mul_(k.h2_over_2pi, add_(S[p], mul_(zz, S[9 + p])));
    }
    return residual_from_gradient(G, B0, k);
}

DBIE_NM_HD Residual residual_any(const double S[12], double z, const NMConsts& k) {
    return k.analytic ? residual_from_analytic_sums(S, z, k) : residual_from_sums(S, z, k);
}

enum NMPhase : int {
    NM_INIT0 = 0, NM_INIT1, NM_INIT2, NM_INIT3,
    NM_REFLECT, NM_EXPAND, NM_OUTSIDE, NM_INSIDE,
    NM_SHRINK1, NM_SHRINK2, NM_SHRINK3,
    NM_DONE
};

struct NMPoint {
    double V[4][3];   // simplex
    double F[4];      // Phi at the vertices (NaN stored as +inf)
    double A[4][5];   // (Bx, By, Bz, f, g) at the vertices
    double P[9];      // pending reflection point: x_r[3], Phi_r, (B, f, g)_r
    double cand[3];   // the trial point whose objective value is outstanding
    int phase, iters;
};

DBIE_NM_HD double as_inf_(double v) { return isnan(v) ? INFINITY : v; }

DBIE_NM_HD void nm_start(NMPoint& s, const NMConsts& k) {
    for (int j = 0; j < 4; ++j)
        for (int p = 0; p < 3; ++p) s.V[j][p] = k.lam0_abs;
    for (int j = 1; j < 4; ++j) s.V[j][j - 1] = add_(k.lam0_abs, k.step_abs);
    for (int j = 0; j < 4; ++j) {
        s.F[j] = INFINITY;
        for (int a = 0; a < 5; ++a) s.A[j][a] = NAN;
    }
    for (int a = 0; a < 9; ++a) s.P[a] = 0.0;
    for (int p = 0; p < 3; ++p) s.cand[p] = s.V[0][p];
    s.phase = NM_INIT0;
    s.iters = 0;
}

// stable insertion sort of the four vertices by Phi ascending (ties keep the earlier index)
DBIE_NM_HD void nm_sort_(NMPoint& s) {
    for (int i = 1; i < 4; ++i) {
        double v[3], a[5];
        const double f = s.F[i];
        for (int p = 0; p < 3; ++p) v[p] = s.V[i][p];
        for (int q = 0; q < 5; ++q) a[q] = s.A[i][q];
        int j = i - 1;
        while (j >= 0 && s.F[j] > f) {
            for (int p = 0; p < 3; ++p) s.V[j + 1][p] = s.V[j][p];
            for (int q = 0; q < 5; ++q) s.A[j + 1][q] = s.A[j][q];
            s.F[j + 1] = s.F[j];
            --j;
        }
        for (int p = 0; p < 3; ++p) s.V[j + 1][p] = v[p];
        for (int q = 0; q < 5; ++q) s.A[j + 1][q] = a[q];
        s.F[j + 1] = f;
    }
}

DBIE_NM_HD void nm_set_vertex_(NMPoint& s, int j, const double v[3], double f, const double a[5]) {
    for (int p = 0; p < 3; ++p) s.V[j][p] = v[p];
    for (int q = 0; q < 5; ++q) s.A[j][q] = a[q];
    s.F[j] = f;
}

DBIE_NM_HD void nm_centroid_(const NMPoint& s, double xbar[3]) {
    for (int p = 0; p < 3; ++p) xbar[p] = div_(add_(add_(s.V[0][p], s.V[1][p]), s.V[2][p]), 3.0);
}

// c1 * xbar + c2 * V3 written as the oracle writes it: (1+rho) xbar - rho V3 etc.
DBIE_NM_HD void nm_trial_(NMPoint& s, double c1, double c2, bool minus) {
    double xbar[3];
    nm_centroid_(s, xbar);
    for (int p = 0; p < 3; ++p) {
        const double a = mul_(c1, xbar[p]), b = mul_(c2, s.V[3][p]);
        s.cand[p] = minus ? sub_(a, b) : add_(a, b);
    }
}

// Consume the objective value of s.cand.  Returns -1 when another evaluation (of the new
// s.cand) is needed, else the final status 0 (Eq. 12 met), 1 (simplex tolerance), 2 (maxiter).
DBIE_NM_HD int nm_advance(NMPoint& s, double phi_raw, const double a[5], const NMConsts& k) {
    const double phi = as_inf_(phi_raw);
    bool end_iter = false, shrink = false;
    switch (s.phase) {
        case NM_INIT0: case NM_INIT1: case NM_INIT2: case NM_INIT3: {
            const int j = s.phase - NM_INIT0;
            nm_set_vertex_(s, j, s.cand, phi, a);
            if (j < 3) {
                for (int p = 0; p < 3; ++p) s.cand[p] = s.V[j + 1][p];
                s.phase = NM_INIT0 + j + 1;
                return -1;
            }
            nm_sort_(s);
            break;   // to the top of the iteration loop
        }
        case NM_REFLECT: {
            if (phi < s.F[0]) {
                for (int p = 0; p < 3; ++p) s.P[p] = s.cand[p];
                s.P[3] = phi;
                for (int q = 0; q < 5; ++q) s.P[4 + q] = a[q];
                nm_trial_(s, 3.0, 2.0, true);            // expansion: xbar + rho chi (xbar - V3)
                s.phase = NM_EXPAND;
                return -1;
            } else if (phi < s.F[2]) {
                nm_set_vertex_(s, 3, s.cand, phi, a);
                end_iter = true;
            } else if (phi < s.F[3]) {
                for (int p = 0; p < 3; ++p) s.P[p] = s.cand[p];
                s.P[3] = phi;
                for (int q = 0; q < 5; ++q) s.P[4 + q] = a[q];
                nm_trial_(s, 1.5, 0.5, true);            // outside contraction
                s.phase = NM_OUTSIDE;
                return -1;
            } else {
                nm_trial_(s, 0.5, 0.5, false);           // inside contraction
                s.phase = NM_INSIDE;
                return -1;
            }
            break;
        }
        case NM_EXPAND: {
            if (phi < s.P[3]) nm_set_vertex_(s, 3, s.cand, phi, a);
            else nm_set_vertex_(s, 3, &s.P[0], s.P[3], &s.P[4]);
            end_iter = true;
            break;
        }
        case NM_OUTSIDE: {
            if (phi <= s.P[3]) { nm_set_vertex_(s, 3, s.cand, phi, a); end_iter = true; }
            else shrink = true;
            break;
        }
        case NM_INSIDE: {
            if (phi < s.F[3]) { nm_set_vertex_(s, 3, s.cand, phi, a); end_iter = true; }
            else shrink = true;
            break;
        }
        case NM_SHRINK1: case NM_SHRINK2: {
            const int j = s.phase - NM_SHRINK1 + 1;
            for (int q = 0; q < 5; ++q) s.A[j][q] = a[q];
            s.F[j] = phi;
            for (int p = 0; p < 3; ++p) s.cand[p] = s.V[j + 1][p];
            s.phase += 1;
            return -1;
        }
        case NM_SHRINK3: {
            for (int q = 0; q < 5; ++q) s.A[3][q] = a[q];
            s.F[3] = phi;
            end_iter = true;
            break;
        }
        default:
            return 2;
    }
    if (shrink) {
        for (int j = 1; j < 4; ++j)
            for (int p = 0; p < 3; ++p)
                s.V[j][p] = add_(s.V[0][p], mul_(0.5, sub_(s.V[j][p], s.V[0][p])));
        for (int p = 0; p < 3; ++p) s.cand[p] = s.V[1][p];
        s.phase = NM_SHRINK1;
        return -1;
    }
    if (end_iter) {
        nm_sort_(s);
        s.iters += 1;
    }
    // top of the iteration loop (Eq. 10-12)
    if (s.iters >= k.maxiter) { s.phase = NM_DONE; return 2; }
    if (k.use_eq12 && s.A[0][3] <= k.eps_f && s.A[0][4] <= k.eps_g) { s.phase = NM_DONE; return 0; }
    double dx = 0.0, df = 0.0;
    for (int j = 1; j < 4; ++j) {
        for (int p = 0; p < 3; ++p) dx = fmax(dx, fabs(sub_(s.V[j][p], s.V[0][p])));
        df = fmax(df, fabs(sub_(s.F[0], s.F[j])));
    }
    if (dx <= k.xtol_abs && df <= k.ftol) { s.phase = NM_DONE; return 1; }
    nm_trial_(s, 2.0, 1.0, true);                        // reflection: xbar + rho (xbar - V3)
    s.phase = NM_REFLECT;
    return -1;
}

}  // namespace dbie
