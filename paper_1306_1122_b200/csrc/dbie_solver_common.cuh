// dbie_solver_common.cuh — device helpers shared by the two lambda-search drivers
// (dbie_solver.cu: Nelder-Mead; dbie_grid.cu: GRID): NaN constant, warp-aggregated list append
// and the outputs of an invalid point.
#pragma once
#include <cuda_runtime.h>

#include "dbie_internal.h"
#include "dbie_nm.cuh"

namespace dbie {

static __device__ __forceinline__ double qnan() { return __longlong_as_double(0x7ff8000000000000LL); }

// append `id` to the list when `keep`; one atomic per warp, order inside a warp preserved
static __device__ __forceinline__ void warp_append(bool keep, int id, int* list, unsigned* counter) {
    const unsigned mask = __ballot_sync(0xffffffffu, keep);
    if (mask == 0) return;
    const int lane = threadIdx.x & 31;
    const int leader = __ffs(mask) - 1;
    unsigned base = 0;
    if (lane == leader) base = atomicAdd(counter, (unsigned)__popc(mask));
    base = __shfl_sync(0xffffffffu, base, leader);
    if (keep) list[base + __popc(mask & ((1u << lane) - 1u))] = id;
}

// outputs are addressed [q*ldo + i]: ldo is the caller's total point count (batched calls pass
// pointers already offset to the batch)
static __device__ void write_invalid(long long ldo, long long i, double* B, double* lam, double* resid, int* iters,
                              int* status) {
    for (int c = 0; c < 3; ++c) {
        B[c * ldo + i] = qnan();
        lam[c * ldo + i] = qnan();
    }
    resid[i] = qnan();
    resid[ldo + i] = qnan();
    iters[i] = 0;
    status[i] = 3;
}

// Per-point optimiser state <-> registers.  The loads go through L2 (__ldcg): in the fused solver the state
// was written earlier in the same launch, possibly by another SM.
static __device__ __forceinline__ void load_point(const SolveArrays& s, long long M, long long i, NMPoint& p) {
    for (int j = 0; j < 4; ++j) {
        for (int c = 0; c < 3; ++c) p.V[j][c] = __ldcg(s.V + (j * 3 + c) * M + i);
        p.F[j] = __ldcg(s.F + j * M + i);
        for (int a = 0; a < 5; ++a) p.A[j][a] = __ldcg(s.aux + (j * 5 + a) * M + i);
    }
    for (int a = 0; a < 9; ++a) p.P[a] = __ldcg(s.pend + a * M + i);
    for (int c = 0; c < 3; ++c) p.cand[c] = __ldcg(s.cand + c * M + i);
    p.phase = __ldcg(s.phase + i);
    p.iters = __ldcg(s.iters + i);
}

static __device__ __forceinline__ void store_point(const SolveArrays& s, long long M, long long i, const NMPoint& p) {
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

}  // namespace dbie
