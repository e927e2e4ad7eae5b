// dbie_solver_common.cuh — device helpers shared by the two lambda-search drivers
// (dbie_solver.cu: Nelder-Mead; dbie_grid.cu: GRID): NaN constant, warp-aggregated list append
// and the outputs of an invalid point.
#pragma once
#include <cuda_runtime.h>

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

}  // namespace dbie
