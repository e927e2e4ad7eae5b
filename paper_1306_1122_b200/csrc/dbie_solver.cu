// dbie_solver.cu — the batched on-device lambda optimiser.
//
// The paper runs the Downhill Simplex iteration on the CPU and crosses the PCIe bus for every
// objective evaluation.  Here every field point carries a resumable Nelder-Mead
// state (dbie_nm.cuh) with exactly ONE outstanding trial lambda triple per pass.  This file holds
// the set-up kernel of the search (initial simplex, invalid points, first active list) and the
// epilogue of dbie_residual; the passes themselves run inside one cooperative launch
// (dbie_solve_fused.cu).  Compiled with -fmad=false.
#include <cuda_runtime.h>
#include <math.h>

#include "dbie_internal.h"
#include "dbie_nm.cuh"
#include "dbie_solver_common.cuh"

namespace dbie {

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

cudaError_t launch_residual_finalize(const BoundaryView& bd, const NMConsts& k, long long M,
                                     long long ldo, const double* z, const double* part, long long cap, double* out,
                                     double* phi, cudaStream_t st) {
    if (M <= 0) return cudaSuccess;
    const unsigned grid = (unsigned)((M + 127) / 128);
    residual_finalize_kernel<<<grid, 128, 0, st>>>(k, bd.nchunks, M, ldo, z, part, cap, out, phi);
    return cudaGetLastError();
}

}  // namespace dbie
