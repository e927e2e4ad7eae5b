// dbie_solver.cu — the batched on-device lambda optimiser.
//
// The paper runs the Downhill Simplex iteration on the CPU and crosses the PCIe bus for every
// objective evaluation.  Here every field point carries a resumable Nelder-Mead
// state (dbie_nm.cuh) with exactly ONE outstanding trial lambda triple per pass; a pass is
//     interaction kernel over the active list (4 stencil positions per point, Eq. 13)
//  -> solve_step_kernel: chunk sums -> B at the stencil -> f, g, Phi (Eq. 8, 9, 14) -> simplex
//     decision -> next trial triple, or the point's final outputs -> compacted next active list.
// The host only enqueues passes; list lengths live in device memory.
#include <cuda_runtime.h>
#include <math.h>

#include "dbie_internal.h"
#include "dbie_nm.cuh"
#include "dbie_solver_common.cuh"

namespace dbie {

__device__ void load_point(const SolveArrays& s, long long M, long long i, NMPoint& p) {
    for (int j = 0; j < 4; ++j) {
        for (int c = 0; c < 3; ++c) p.V[j][c] = s.V[(j * 3 + c) * M + i];
        p.F[j] = s.F[j * M + i];
        for (int a = 0; a < 5; ++a) p.A[j][a] = s.aux[(j * 5 + a) * M + i];
    }
    for (int a = 0; a < 9; ++a) p.P[a] = s.pend[a * M + i];
    for (int c = 0; c < 3; ++c) p.cand[c] = s.cand[c * M + i];
    p.phase = s.phase[i];
    p.iters = s.iters[i];
}

__device__ void store_point(const SolveArrays& s, long long M, long long i, const NMPoint& p) {
    for (int j = 0; j < 4; ++j) {
        for (int c = 0; c < 3; ++c) s.V[(j * 3 + c) * M + i] = p.V[j][c];
        s.F[j * M + i] = p.F[j];
        for (int a = 0; a < 5; ++a) s.aux[(j * 5 + a) * M + i] = p.A[j][a];
    }
    for (int a = 0; a < 9; ++a) s.pend[a * M + i] = p.P[a];
    for (int c = 0; c < 3; ++c) s.cand[c * M + i] = p.cand[c];
    s.phase[i] = p.phase;
    s.iters[i] = p.iters;
}

__global__ void solve_init_kernel(SolveArrays s, NMConsts k, long long M, long long ldo,
                                  const double* __restrict__ x,
                                  const double* __restrict__ y, const double* __restrict__ z, double* B,
                                  double* lam, double* resid, int* iters, int* status) {
    const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    bool keep = false;
    if (i < M) {
        const double xi = x[i], yi = y[i], zi = z[i];
        const bool invalid = !(zi > 0.0) || !isfinite(xi) || !isfinite(yi) || !isfinite(zi);
        if (invalid) {
            write_invalid(ldo, i, B, lam, resid, iters, status);
            s.phase[i] = NM_DONE;
        } else {
            NMPoint p;
            nm_start(p, k);
            store_point(s, M, i, p);
            keep = true;
        }
    }
    warp_append(keep, (int)i, s.act[0], &s.nact[0]);
}

// pass `pass` consumes list pass&1 and builds list (pass+1)&1
__global__ void solve_step_kernel(SolveArrays s, NMConsts k, int nchunks, int pass, long long M,
                                  long long ldo,
                                  const double* __restrict__ z, const double* __restrict__ part,
                                  long long cap, double* B, double* lam, double* resid, int* iters,
                                  int* status, unsigned long long* nevals) {
    const int cur = pass & 1;
    const unsigned n = s.nact[cur];
    const unsigned j = blockIdx.x * blockDim.x + threadIdx.x;
    if (blockIdx.x * blockDim.x >= n) return;   // whole block idle (uniform)
    if (j == 0 && nevals) atomicAdd(nevals, (unsigned long long)n);
    bool keep = false;
    int id = 0;
    if (j < n) {
        id = s.act[cur][j];
        const NMConsts& c = k;
        double S[12];
        for (int q = 0; q < 12; ++q) {
            double sum = part[(long long)q * cap + j];
            for (int ch = 1; ch < nchunks; ++ch) sum = __dadd_rn(sum, part[((long long)ch * 12 + q) * cap + j]);
            S[q] = sum;
        }
        const Residual r = residual_any(S, z[id], c);
        const double a[5] = {r.B[0], r.B[1], r.B[2], r.f, r.g};
        NMPoint p;
        load_point(s, M, id, p);
        const int st = nm_advance(p, r.phi, a, c);
        store_point(s, M, id, p);
        if (st < 0) {
            keep = true;
        } else if (!isfinite(p.F[0])) {
            write_invalid(ldo, id, B, lam, resid, iters, status);
        } else {
            for (int q = 0; q < 3; ++q) {
                B[q * ldo + id] = p.A[0][q];
                lam[q * ldo + id] = fabs(p.V[0][q]);
            }
            resid[id] = p.A[0][3];
            resid[ldo + id] = p.A[0][4];
            iters[id] = p.iters;
            status[id] = st;
        }
    }
    warp_append(keep, id, s.act[cur ^ 1], &s.nact[cur ^ 1]);
}

// one objective evaluation per point at given lambda (dbie_residual)
__global__ void residual_finalize_kernel(NMConsts k, int nchunks, long long M, long long ldo,
                                         const double* __restrict__ z,
                                         const double* __restrict__ part, long long cap, double* out,
                                         double* phi) {
    const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= M) return;
    const NMConsts& c = k;
    double S[12];
    for (int q = 0; q < 12; ++q) {
        double sum = part[(long long)q * cap + i];
        for (int ch = 1; ch < nchunks; ++ch) sum = __dadd_rn(sum, part[((long long)ch * 12 + q) * cap + i]);
        S[q] = sum;
    }
    const double zi = z[i];
    Residual r = residual_any(S, zi, c);
    const bool invalid = !(zi > 0.0) || !isfinite(zi);
    const double v[9] = {r.B[0], r.B[1], r.B[2], r.f, r.g, r.J[0], r.J[1], r.J[2], r.div};
    for (int q = 0; q < 9; ++q) out[q * ldo + i] = invalid ? qnan() : v[q];
    if (phi) phi[i] = invalid ? qnan() : r.phi;
}

cudaError_t launch_solve_init(const SolveArrays& s, const NMConsts& k, long long M, long long ldo,
                              const double* x,
                              const double* y, const double* z, double* B, double* lam, double* resid,
                              int* iters, int* status, cudaStream_t st) {
    if (M <= 0) return cudaSuccess;
    const unsigned grid = (unsigned)((M + 127) / 128);
    solve_init_kernel<<<grid, 128, 0, st>>>(s, k, M, ldo, x, y, z, B, lam, resid, iters, status);
    return cudaGetLastError();
}

cudaError_t launch_solve_step(const SolveArrays& s, const NMConsts& k, const BoundaryView& bd, int pass,
                              long long M, long long ldo, const double* z, const double* part,
                              long long cap, double* B, double* lam, double* resid, int* iters,
                              int* status, unsigned long long* nevals, cudaStream_t st) {
    if (M <= 0) return cudaSuccess;
    const unsigned grid = (unsigned)((M + 127) / 128);   // blocks past the device-side count exit at once
    solve_step_kernel<<<grid, 128, 0, st>>>(s, k, bd.nchunks, pass, M, ldo, z, part, cap, B, lam, resid, iters,
                                            status, nevals);
    return cudaGetLastError();
}

cudaError_t launch_residual_finalize(const BoundaryView& bd, const NMConsts& k, long long M,
                                     long long ldo, const double* z, const double* part, long long cap, double* out,
                                     double* phi, cudaStream_t st) {
    if (M <= 0) return cudaSuccess;
    const unsigned grid = (unsigned)((M + 127) / 128);
    residual_finalize_kernel<<<grid, 128, 0, st>>>(k, bd.nchunks, M, ldo, z, part, cap, out, phi);
    return cudaGetLastError();
}

}  // namespace dbie
