// dbie_trace.cu — field-line and current-line tracing (PAPER.md:201-249 shows lines of B and
// of J = curl B, Eq. 14, without saying how they were integrated; reading T-1).
//
//   dr/ds = sigma v(r)/|v(r)|,  v = B or J,  classical RK4 in arc length at a fixed step ds:
//   k1 = u(r_n), k2 = u(r_n + ds/2 k1), k3 = u(r_n + ds/2 k2), k4 = u(r_n + ds k3),
//   r_{n+1} = r_n + ds/6 (k1 + 2 k2 + 2 k3 + k4).
//
// v at a stage point comes from the library's own entry points on the line heads (dbie_solve -> B and lambda,
// dbie_residual -> J, dbie_eval at a fixed lambda): nothing is interpolated.  The kernels here do only the
// bookkeeping between those calls: consume a stage's v, place the next stage point, accept the step, apply
// the stop rules.  A line that has stopped (or is stopped within the current step) hands z = -1 to the field
// evaluation, which treats it as an invalid point and spends nothing on it in the lambda solve.
// Every operation is separately rounded (compiled with -fmad=false, explicit _rn intrinsics), in the order the
// update is written above.
#include <cuda_runtime.h>
#include <math.h>

#include "dbie_internal.h"
#include "dbie_solver_common.cuh"

namespace dbie {

__device__ __forceinline__ bool trace_inside(const TraceBox& b, double x, double y, double z) {
    return (x >= b.x0) && (x <= b.x1) && (y >= b.y0) && (y <= b.y1) && (z > b.z0) && (z <= b.z1);
}

// seeds -> state; path[(c*(S+1) + k)*L + i] = NaN except point 0 of a line that starts inside the region
__global__ void trace_init_kernel(TraceState t, TraceBox box, long long L, int S, const double* __restrict__ sx,
                                  const double* __restrict__ sy, const double* __restrict__ sz, double* path,
                                  int* npts, int* status) {
    const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= L) return;
    const double x = sx[i], y = sy[i], z = sz[i];
    const bool in = trace_inside(box, x, y, z) && isfinite(x) && isfinite(y) && isfinite(z);
    for (int c = 0; c < 3; ++c)
        for (int k = 0; k <= S; ++k) path[((long long)c * (S + 1) + k) * L + i] = qnan();
    t.r[i] = x; t.r[L + i] = y; t.r[2 * L + i] = z;
    t.alive[i] = in;
    t.good[i] = in;
    t.why[i] = 1;
    npts[i] = in ? 1 : 0;
    status[i] = in ? 0 : 1;
    if (in) {
        path[(0LL * (S + 1)) * L + i] = x;
        path[(1LL * (S + 1)) * L + i] = y;
        path[(2LL * (S + 1)) * L + i] = z;
    }
    t.px[i] = x; t.py[i] = y; t.pz[i] = in ? z : -1.0;   // stage point 0 of step 0
}

// consume v of stage `stage` (0..3) of step `step`, place the next stage point or accept the step
__global__ void trace_stage_kernel(TraceState t, TraceBox box, long long L, int S, int step, int stage, int direction,
                                   double ds, const double* __restrict__ v, long long ldv, double* path, int* npts,
                                   int* status) {
    const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= L) return;
    if (!t.alive[i]) return;                       // its stage point stays at z = -1
    bool good = t.good[i] != 0;
    int why = t.why[i];
    const double rx = t.r[i], ry = t.r[L + i], rz = t.r[2 * L + i];
    double u[3] = {0.0, 0.0, 0.0};
    if (good) {
        const double v0 = v[i], v1 = v[ldv + i], v2 = v[2 * ldv + i];
        const double n = __dsqrt_rn(__dadd_rn(__dadd_rn(__dmul_rn(v0, v0), __dmul_rn(v1, v1)), __dmul_rn(v2, v2)));
        if (!(isfinite(n) && n > 0.0)) {
            good = false;
            why = 2;
        } else {
            const double sg = (double)direction;
            u[0] = __ddiv_rn(__dmul_rn(sg, v0), n);
            u[1] = __ddiv_rn(__dmul_rn(sg, v1), n);
            u[2] = __ddiv_rn(__dmul_rn(sg, v2), n);
            for (int c = 0; c < 3; ++c) t.k[((long long)stage * 3 + c) * L + i] = u[c];
        }
    }
    if (stage < 3) {
        double px = rx, py = ry, pz = -1.0;
        if (good) {
            const double cf = (stage < 2) ? __dmul_rn(0.5, ds) : ds;
            px = __dadd_rn(rx, __dmul_rn(cf, u[0]));
            py = __dadd_rn(ry, __dmul_rn(cf, u[1]));
            pz = __dadd_rn(rz, __dmul_rn(cf, u[2]));
            if (!trace_inside(box, px, py, pz)) {
                good = false;
                why = 1;
                px = rx; py = ry; pz = -1.0;
            }
        }
        t.px[i] = px; t.py[i] = py; t.pz[i] = pz;
        t.good[i] = good;
        t.why[i] = why;
        return;
    }
    // stage 3: r_{n+1} = r_n + ds/6 (((k1 + 2 k2) + 2 k3) + k4)
    double nx = rx, ny = ry, nz = rz;
    if (good) {
        const double w = __ddiv_rn(ds, 6.0);
        double rn[3];
        const double r0[3] = {rx, ry, rz};
        for (int c = 0; c < 3; ++c) {
            const double k1 = t.k[(0LL * 3 + c) * L + i], k2 = t.k[(1LL * 3 + c) * L + i];
            const double k3 = t.k[(2LL * 3 + c) * L + i], k4 = u[c];
            const double sum = __dadd_rn(__dadd_rn(__dadd_rn(k1, __dmul_rn(2.0, k2)), __dmul_rn(2.0, k3)), k4);
            rn[c] = __dadd_rn(r0[c], __dmul_rn(w, sum));
        }
        nx = rn[0]; ny = rn[1]; nz = rn[2];
        if (!(trace_inside(box, nx, ny, nz) && isfinite(nx) && isfinite(ny) && isfinite(nz))) {
            good = false;
            why = 1;
        }
    }
    if (good) {
        t.r[i] = nx; t.r[L + i] = ny; t.r[2 * L + i] = nz;
        path[(0LL * (S + 1) + step + 1) * L + i] = nx;
        path[(1LL * (S + 1) + step + 1) * L + i] = ny;
        path[(2LL * (S + 1) + step + 1) * L + i] = nz;
        npts[i] = step + 2;
        t.px[i] = nx; t.py[i] = ny; t.pz[i] = nz;       // stage point 0 of the next step
        t.good[i] = 1;
    } else {
        status[i] = why;
        t.alive[i] = 0;
        t.good[i] = 0;
        t.pz[i] = -1.0;
    }
    t.why[i] = 1;
}

__global__ void trace_fill_kernel(double* dst, long long n, double v0, double v1, double v2, long long L) {
    const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i < n) dst[i] = (i < L) ? v0 : (i < 2 * L ? v1 : v2);
}

cudaError_t launch_trace_init(const TraceState& t, const TraceBox& box, long long L, int S, const double* sx,
                              const double* sy, const double* sz, double* path, int* npts, int* status,
                              cudaStream_t st) {
    if (L <= 0) return cudaSuccess;
    trace_init_kernel<<<(unsigned)((L + 127) / 128), 128, 0, st>>>(t, box, L, S, sx, sy, sz, path, npts, status);
    return cudaGetLastError();
}

cudaError_t launch_trace_stage(const TraceState& t, const TraceBox& box, long long L, int S, int step, int stage,
                               int direction, double ds, const double* v, long long ldv, double* path, int* npts,
                               int* status, cudaStream_t st) {
    if (L <= 0) return cudaSuccess;
    trace_stage_kernel<<<(unsigned)((L + 127) / 128), 128, 0, st>>>(t, box, L, S, step, stage, direction, ds, v, ldv,
                                                                    path, npts, status);
    return cudaGetLastError();
}

cudaError_t launch_trace_fill_lambda(double* lam, long long L, const double l[3], cudaStream_t st) {
    if (L <= 0) return cudaSuccess;
    trace_fill_kernel<<<(unsigned)((3 * L + 255) / 256), 256, 0, st>>>(lam, 3 * L, l[0], l[1], l[2], L);
    return cudaGetLastError();
}

}  // namespace dbie
