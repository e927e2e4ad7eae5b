// host_shim.cpp — CPU build of the __host__ __device__ arithmetic of the CUDA path
// (dbie_math.cuh, dbie_nm.cuh) so that the not-gpu tests can check it against mpmath / SciPy.
// This is NOT a CPU fallback: it exposes single functions to tests, it is not linked into
// libdbie_b200.so, and no product entry point calls it.  The only host/device difference is the
// reciprocal-sqrt seed (MUFU.RSQ64H on the device, a float-rounded 1/sqrt here).
// Built with g++ -O2 -ffp-contract=off; explicit fma() calls map to libm fma (correctly rounded).
#include "dbie_math.cuh"
#include "dbie_math_f32.cuh"
#include "dbie_nm.cuh"

static const dbie::TrigRef kTr{dbie::kTrigTabHost, 0u};   // the same table the kernels copy into shared memory

extern "C" {

void shim_sincos(long n, const double* th, double* s, double* c) {
    for (long i = 0; i < n; ++i) dbie::sincos_pos(th[i], kTr, s[i], c[i]);
}
void shim_kernel_n(long n, const double* th, double* out) {
    for (long i = 0; i < n; ++i) out[i] = dbie::kernel_n(th[i], kTr);
}
void shim_kernel_n_reduced(long n, const double* th, double* out) {   // reading A-12 (eval-only flag)
    for (long i = 0; i < n; ++i) out[i] = dbie::kernel_n<true>(th[i], kTr);
}
void shim_kernel_n_cos(long n, const double* th, double* nv, double* cv) {
    for (long i = 0; i < n; ++i) dbie::kernel_n_cos(th[i], kTr, nv[i], cv[i]);
}
void shim_kernel_n_near(long n, const double* th, const double* s0, const double* c0, const double* eps, double* out) {
    for (long i = 0; i < n; ++i) out[i] = dbie::kernel_n_near(th[i], s0[i], c0[i], eps[i]);
}
void shim_rsqrt(long n, const double* a, double* out) {
    for (long i = 0; i < n; ++i) out[i] = dbie::rsqrt_full(a[i]);
}
// one interaction exactly as the kernel's inner loop forms it: returns the three terms
// n(lam_p r) * (1/r^3 * B_p0)
void shim_interaction(double dx, double dy, double z, const double lam[3], const double b0[3], double out[3]) {
    const double cc = fma(dy, dy, z * z);
    const double r2 = fma(dx, dx, cc);
    const double y = dbie::rsqrt_full(r2);
    const double rr = r2 * y;
    const double w = (y * y) * y;
    for (int p = 0; p < 3; ++p) out[p] = dbie::kernel_n(fabs(lam[p]) * rr, kTr) * (w * b0[p]);
}

// fp32 kernel value n(theta) on the table path (the SFU variant is device only)
void shim_kernel_n_f32(long n, const float* th, float* out) {
    static const dbie::TrigRefF trf{dbie::kTrigTabHostF, 0u};
    for (long i = 0; i < n; ++i) out[i] = dbie::kernel_n_f32<false>(th[i], trf);
}

typedef double (*shim_objective)(const double*);

// Drive the resumable Nelder-Mead state machine on a caller-supplied objective (pin against
// SciPy).  simplex: 4x3 initial vertices.  Returns the final status.
int shim_nm_generic(shim_objective fn, const double* simplex, double xtol, double ftol, int maxiter,
                    double* trace /* (maxiter+1)*3 */, double* final_simplex /* 12 */, double* final_f /* 4 */,
                    int* iters, int* nfev) {
    dbie::NMConsts k;
    k.delta_abs = 1.0; k.d_abs = 1.0; k.w_g = 1.0; k.eps_f = 0.0; k.eps_g = 0.0;
    k.xtol_abs = xtol; k.ftol = ftol; k.lam0_abs = 0.0; k.step_abs = 1.0; k.h2_over_2pi = 1.0;
    k.maxiter = maxiter; k.use_eq12 = 0; k.analytic = 0;
    dbie::NMPoint p;
    dbie::nm_start(p, k);
    for (int j = 0; j < 4; ++j)
        for (int c = 0; c < 3; ++c) p.V[j][c] = simplex[j * 3 + c];
    for (int c = 0; c < 3; ++c) p.cand[c] = p.V[0][c];
    const double a[5] = {0, 0, 0, 1.0, 1.0};
    int st = -1, nf = 0, last_iters = -1;
    while (st < 0) {
        const double f = fn(p.cand);
        ++nf;
        st = dbie::nm_advance(p, f, a, k);
        if (trace && p.phase >= dbie::NM_REFLECT && p.iters != last_iters) {
            // a new iteration starts (or the search ended): record the best vertex
            for (int c = 0; c < 3; ++c) trace[3 * p.iters + c] = p.V[0][c];
            last_iters = p.iters;
        }
    }
    for (int j = 0; j < 4; ++j) {
        for (int c = 0; c < 3; ++c) final_simplex[j * 3 + c] = p.V[j][c];
        final_f[j] = p.F[j];
    }
    *iters = p.iters;
    *nfev = nf;
    return st;
}

// residual of Eq. 8, 9, 13, 14 from B at the four stencil positions: out = f, g, Jx, Jy, Jz, div, phi
void shim_residual(const double* Bs /* 4x3 */, double delta_abs, double d_abs, double w_g, double* out) {
    dbie::NMConsts k{};
    k.delta_abs = delta_abs; k.d_abs = d_abs; k.w_g = w_g;
    double B[4][3];
    for (int s = 0; s < 4; ++s)
        for (int p = 0; p < 3; ++p) B[s][p] = Bs[s * 3 + p];
    const dbie::Residual r = dbie::residual_from_stencil(B, k);
    out[0] = r.f; out[1] = r.g; out[2] = r.J[0]; out[3] = r.J[1]; out[4] = r.J[2]; out[5] = r.div; out[6] = r.phi;
}

}  // extern "C"
