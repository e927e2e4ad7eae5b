// dbie_solve_fused.cu — the whole per-point Nelder-Mead search in ONE cooperative launch.
//
// The paper crosses the PCIe bus for every objective evaluation and names that as the bottleneck to remove
// (PAPER.md:124).  Round 1 of this build kept the data on the device but still had the host enqueue two
// launches per pass (interaction kernel, step kernel) with the chunk partial sums written to and re-read from
// scratch in between.  Here a persistent grid (one CTA per resident slot, cudaLaunchCooperativeKernel) loops
// over the passes itself:
//
//   pass:  n = length of the active list (device memory)            -> n == 0: every CTA leaves
//          work items from an atomic counter, two shapes chosen from n alone:
//            thread per point  (n large)  128 points x a range of canonical chunks; interact_item, the same
//                                         inner loops as dbie_residual;
//            warp per point    (n small)  4 points x one chunk; the 32 lanes of a warp take 32 consecutive
//                                         pixels, their 12 terms go through shared memory to 12 "chain" lanes
//                                         which add them in pixel order.  Same operations in the same order,
//                                         so the sums are bit-identical to the thread-per-point shape, at
//                                         ~1/10 of its latency for a handful of points.
//          the CTA that finishes the LAST chunk range of a point block adds the chunk sums in chunk order
//          (A4), forms B at the stencil -> J, div B, f, g, Phi (A5; Eq. 8, 9, 13, 14), advances the simplex
//          (A6) and appends the survivors to the next list (A7).  A CTA that covered all chunks itself (large
//          n) never writes the partial sums at all.
//          grid-wide barrier.
//
// The decisions are those of the resumable state machine nm_advance (dbie_nm.cuh, separately rounded IEEE operations);
// results do not depend on the batch, the shape or the CTA that happened to finish last.
// This unit is compiled like dbie_interact.cu (FMA contraction on): the interaction arithmetic must be the
// same instruction sequence as in dbie_residual; the search itself uses __dmul_rn / __dadd_rn throughout.
#include <cooperative_groups.h>
#include <cuda_runtime.h>
#include <math.h>

#include "dbie_interact_fp64.cuh"
#include "dbie_internal.h"
#include "dbie_nm.cuh"
#include "dbie_solver_common.cuh"

namespace cg = cooperative_groups;

namespace dbie {

constexpr int kFusedThreads = 128, kFusedMinB = 2;
constexpr int kFusedWarps = kFusedThreads / 32;
constexpr int kStageRow = 33;   // 32 pixels + 1 pad: the chain lanes' reads hit distinct banks
constexpr size_t kFusedSmem = kTrigTableBytes                                        // angle table (dbie_math.cuh)
                              + sizeof(double4) * 2 * kTilePx                        // boundary tiles
                              + sizeof(double) * kFusedWarps * 24 * kStageRow        // factor pairs of 32 pixels
                              + 64;                                                  // mbarriers, scalars

// chunk sums of a thread that covered every chunk itself stay in registers; otherwise they go to the scratch
struct FusedSink {
    const InteractParams& p;
    bool whole;
    double run[12];
    template <int NA>
    __device__ __forceinline__ void operator()(const ItemCtx& ic, int c, const double (&acc)[NA][3]) {
        static_assert(NA == 4, "12 sums per slot");
        if (whole) {
#pragma unroll
            for (int kd = 0; kd < 4; ++kd)
#pragma unroll
                for (int q = 0; q < 3; ++q)
                    run[kd * 3 + q] = (c == 0) ? acc[kd][q] : __dadd_rn(run[kd * 3 + q], acc[kd][q]);
        } else if (ic.live) {
#pragma unroll
            for (int kd = 0; kd < 4; ++kd)
#pragma unroll
                for (int q = 0; q < 3; ++q) p.part[((long long)c * 12 + kd * 3 + q) * p.cap + ic.slot] = acc[kd][q];
        }
    }
};

// A5 + A6 for one point: sums -> residual -> simplex decision -> state or final outputs.  True: still active.
static __device__ bool nm_consume(const FusedParams& P, int id, const double (&S)[12]) {
    const Residual r = residual_any(S, P.ip.z[id], P.k);
    const double a[5] = {r.B[0], r.B[1], r.B[2], r.f, r.g};
    NMPoint pt;
    load_point(P.s, P.count, id, pt);
    const int st = nm_advance(pt, r.phi, a, P.k);
    store_point(P.s, P.count, id, pt);
    if (st < 0) return true;
    if (!isfinite(pt.F[0])) {
        write_invalid(P.ldo, id, P.B, P.lam, P.resid, P.iters, P.status);
    } else {
        for (int q = 0; q < 3; ++q) {
            P.B[q * P.ldo + id] = pt.A[0][q];
            P.lam[q * P.ldo + id] = fabs(pt.V[0][q]);
        }
        P.resid[id] = pt.A[0][3];
        P.resid[P.ldo + id] = pt.A[0][4];
        P.iters[id] = pt.iters;
        P.status[id] = st;
    }
    return false;
}

// The warp-per-point shape: warp w of the CTA owns slot grp*4 + w; lanes = 32 consecutive pixels of a row.
template <int MODE>
__device__ __forceinline__ void interact_item_warp(const InteractParams& p, const TrigRef& tr, double4 (*tile)[kTilePx],
                                                   uint64_t* full, unsigned& it, double* stage, long long n,
                                                   long long grp, int c0, int c1) {
    const int tid = threadIdx.x, lane = tid & 31, wib = tid >> 5;
    const BoundaryView& bd = p.bd;
    const long long slot0 = grp * kFusedWarps + wib;
    const bool live = slot0 < n;
    const long long slot = live ? slot0 : n - 1;
    const long long id = (long long)__ldcg(p.act + slot);
    const double xi = p.x[id], yi = p.y[id], zi = p.z[id];
    const double z2 = zi * zi;
    const double xi1 = __dadd_rn(xi, p.delta_abs), yi2 = __dadd_rn(yi, p.delta_abs);
    const double zi3 = __dadd_rn(zi, p.delta_abs), z23 = zi3 * zi3;
    double lam[3], lam2[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        lam[c] = fabs(__ldcg(p.lam + c * p.ldlam + id));
        lam2[c] = lam[c] * lam[c];
    }
    const bool small_eps = fmax(fmax(lam[0], lam[1]), lam[2]) * p.delta_abs <= kNearEpsMax;
    double* stA = stage + (size_t)wib * 24 * kStageRow;   // [12][33]
    double* stB = stA + 12 * kStageRow;
    double acc = 0.0;                                      // chain lane k < 12 owns sum k = kind*3 + component

    const int u0 = chunk_first_unit(bd, c0), u1 = chunk_first_unit(bd, c1);   // as in interact_item
    const int t0 = unit_tile(bd, u0), t1 = unit_tile(bd, u1 - 1) + 1;
    int c = c0;
    int u_chunk_end = chunk_first_unit(bd, c + 1);
    if (tid == 0) {
        const TileDesc d = tile_desc(bd, t0);
        mbar_expect_tx(&full[it & 1], (unsigned)d.npx * 32u);
        bulk_g2s(&tile[it & 1][0], bd.rec + d.px0, (unsigned)d.npx * 32u, &full[it & 1]);
    }
    for (int t = t0; t < t1; ++t, ++it) {
        if (tid == 0 && t + 1 < t1) {
            const TileDesc dn = tile_desc(bd, t + 1);
            const unsigned sn = (it + 1) & 1;
            mbar_expect_tx(&full[sn], (unsigned)dn.npx * 32u);
            bulk_g2s(&tile[sn][0], bd.rec + dn.px0, (unsigned)dn.npx * 32u, &full[sn]);
        }
        const TileDesc d = tile_desc(bd, t);
        mbar_wait(&full[it & 1], (it >> 1) & 1);
        const double4* __restrict__ rp = &tile[it & 1][0];
        for (int row = 0; row < d.nrows; ++row, rp += d.ncols) {
            const int unit = (bd.segs_per_row == 1) ? d.row0 + row : t;
            if (unit < u0 || unit >= u1) continue;   // a row of a neighbouring chunk in a shared tile
            const double yk = __ldg(bd.yk + d.row0 + row);
            const double dy = yk - yi;
            const double cc = fma(dy, dy, z2);
            const double dy2 = yk - yi2;
            const double cc2 = fma(dy2, dy2, z2), cc3 = fma(dy, dy, z23);
            for (int j0 = 0; j0 < d.ncols; j0 += 32) {
                const int j = j0 + lane;
                if (j < d.ncols) {
                    double fa[4][3], fb[4][3];
                    if (MODE == MODE_STENCIL4) {
                        if (small_eps) stencil4_terms<true>(tr, rp[j], xi, xi1, cc, cc2, cc3, lam, fa, fb);
                        else stencil4_terms<false>(tr, rp[j], xi, xi1, cc, cc2, cc3, lam, fa, fb);
                    } else {
                        analytic_terms(tr, rp[j], xi, dy, cc, lam, lam2, fa, fb);
                    }
#pragma unroll
                    for (int kd = 0; kd < 4; ++kd)
#pragma unroll
                        for (int q = 0; q < 3; ++q) {
                            stA[(kd * 3 + q) * kStageRow + lane] = fa[kd][q];
                            stB[(kd * 3 + q) * kStageRow + lane] = fb[kd][q];
                        }
                }
                __syncwarp();
                if (lane < 12) {   // the accumulation of the thread-per-point loop, pixel by pixel
                    const int cnt = (d.ncols - j0 < 32) ? (d.ncols - j0) : 32;
                    const double* a = stA + lane * kStageRow;
                    const double* b = stB + lane * kStageRow;
                    for (int jj = 0; jj < cnt; ++jj) acc = fma(a[jj], b[jj], acc);
                }
                __syncwarp();
            }
            if (unit + 1 == u_chunk_end) {
                if (live && lane < 12) p.part[((long long)c * 12 + lane) * p.cap + slot] = acc;
                acc = 0.0;
                ++c;
                u_chunk_end = chunk_first_unit(bd, c + 1);
            }
        }
        __syncthreads();
    }
}

template <int MODE, int UNR>
__global__ void __launch_bounds__(kFusedThreads, kFusedMinB) solve_nm_fused_kernel(const __grid_constant__ FusedParams P) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double4(*tile)[kTilePx] = reinterpret_cast<double4(*)[kTilePx]>(smem_raw + kTrigTableBytes);
    double* stage = reinterpret_cast<double*>(smem_raw + kTrigTableBytes + sizeof(double4) * 2 * kTilePx);
    uint64_t* full = reinterpret_cast<uint64_t*>(stage + kFusedWarps * 24 * kStageRow);
    long long* next_item = reinterpret_cast<long long*>(full + 2);
    int* is_last = reinterpret_cast<int*>(next_item + 1);

    cg::grid_group grid = cg::this_grid();
    const int tid = threadIdx.x, lane = tid & 31, wib = tid >> 5;
    if (tid == 0) {
        mbar_init(&full[0], 1);
        mbar_init(&full[1], 1);
        mbar_fence_init();
    }
    const TrigRef tr = trig_fill(smem_raw, tid, kFusedThreads);
    __syncthreads();

    const InteractParams& ip = P.ip;
    const int NCH = ip.bd.nchunks;
    unsigned it = 0;
    for (int pass = 0; pass < P.maxpass; ++pass) {
        const int cur = pass & 1, r0 = pass % 3, r1 = (pass + 1) % 3, r2 = (pass + 2) % 3;
        const long long n = (long long)*(volatile const unsigned*)(P.nact3 + r0);
        if (P.trace && blockIdx.x == 0 && tid == 0 && pass < P.trace_cap) {   // diagnostic (dbie_profile): pass timeline
            unsigned long long now;
            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(now));
            P.trace[2 * pass] = (unsigned long long)n;
            P.trace[2 * pass + 1] = now;
        }
        if (n == 0) break;   // the same value in every CTA: nobody writes slot r0 during this pass
        if (blockIdx.x == 0 && tid == 0) {
            P.nact3[r2] = 0u;
            P.work3[r2] = 0u;
            atomicAdd(P.nevals, (unsigned long long)n);
        }
        InteractParams q = ip;
        q.act = P.s.act[cur];
        int* next_list = P.s.act[cur ^ 1];
        unsigned* next_count = P.nact3 + r1;
        const long long ngrp = (n + kFusedWarps - 1) / kFusedWarps;

        if (ngrp * NCH > P.warp_items_max) {
            // ---------------- thread per point: 128 points x a range of chunks
            // Schedule: as many whole rounds of the grid as the point blocks fill run with one item per block
            // covering ALL chunks (sums stay in registers); only the remaining blocks of the last, partial
            // round are split over chunk ranges, as finely as it takes to fill the grid once more.
            const long long nblk = (n + kFusedThreads - 1) / kFusedThreads;
            const long long G = gridDim.x;
            const long long nwhole = (nblk / G) * G;
            const long long rem = nblk - nwhole;
            int nsplit_t = 1;
            if (rem > 0) {   // smallest split minimising rounds x longest item, in chunks
                long long best = -1;
                for (int sc = 1; sc <= NCH; ++sc) {
                    const long long cost = ((rem * sc + G - 1) / G) * ((NCH + sc - 1) / sc);
                    if (best < 0 || cost < best) {
                        best = cost;
                        nsplit_t = sc;
                    }
                }
            }
            const long long nwork = nwhole + rem * nsplit_t;
            for (;;) {
                if (tid == 0) *next_item = (long long)atomicAdd(P.work3 + r0, 1u);
                __syncthreads();
                const long long w = *next_item;
                if (w >= nwork) break;
                long long blk = w;
                int nsplit = 1, sp = 0;
                if (w >= nwhole) {
                    nsplit = nsplit_t;
                    blk = nwhole + (w - nwhole) / nsplit;
                    sp = (int)((w - nwhole) % nsplit);
                }
                const int c0 = (int)(((long long)sp * NCH) / nsplit);
                const int c1 = (int)(((long long)(sp + 1) * NCH) / nsplit);
                FusedSink sink{q, nsplit == 1, {}};
                interact_item<MODE, 1, kFusedThreads, UNR>(q, tr, tile, full, it, n, 1, blk, c0, c1, sink);
                const long long slot = blk * kFusedThreads + tid;
                const bool live = slot < n;
                if (nsplit > 1) {
                    // the partial sums of this chunk range are in the scratch; the last CTA to get here consumes them
                    __threadfence();
                    __syncthreads();
                    if (tid == 0) {
                        const unsigned old = atomicAdd(P.done + blk, 1u);
                        const int last = old == (unsigned)(nsplit - 1);
                        if (last) P.done[blk] = 0u;   // next use is after the grid barrier
                        *is_last = last;
                    }
                    __syncthreads();
                    if (!*is_last) continue;
                    __threadfence();
                    if (live) {
#pragma unroll
                        for (int k = 0; k < 12; ++k) {
                            double sum = __ldcg(q.part + (long long)k * q.cap + slot);
                            for (int ch = 1; ch < NCH; ++ch) sum = __dadd_rn(sum, __ldcg(q.part + ((long long)ch * 12 + k) * q.cap + slot));
                            sink.run[k] = sum;
                        }
                    }
                }
                int id = 0;
                bool keep = false;
                if (live) {
                    id = __ldcg(q.act + slot);
                    keep = nm_consume(P, id, sink.run);
                }
                warp_append(keep, id, next_list, next_count);
            }
        } else {
            // ---------------- warp per point: 4 points x one chunk
            const long long nwork = ngrp * NCH;
            for (;;) {
                if (tid == 0) *next_item = (long long)atomicAdd(P.work3 + r0, 1u);
                __syncthreads();
                const long long w = *next_item;
                if (w >= nwork) break;
                const long long grp = w / NCH;
                const int c0 = (int)(w % NCH);
                interact_item_warp<MODE>(q, tr, tile, full, it, stage, n, grp, c0, c0 + 1);
                __threadfence();
                __syncthreads();
                if (tid == 0) {
                    const unsigned old = atomicAdd(P.done + grp, 1u);
                    const int last = old == (unsigned)(NCH - 1);
                    if (last) P.done[grp] = 0u;
                    *is_last = last;
                }
                __syncthreads();
                if (!*is_last) continue;
                __threadfence();
                const long long slot = grp * kFusedWarps + wib;
                const bool live = slot < n;
                double sum = 0.0;
                if (live && lane < 12) {
                    sum = __ldcg(q.part + (long long)lane * q.cap + slot);
                    for (int ch = 1; ch < NCH; ++ch) sum = __dadd_rn(sum, __ldcg(q.part + ((long long)ch * 12 + lane) * q.cap + slot));
                }
                double S[12];
#pragma unroll
                for (int k = 0; k < 12; ++k) S[k] = __shfl_sync(0xffffffffu, sum, k);
                int id = 0;
                bool keep = false;
                if (live && lane == 0) {
                    id = __ldcg(q.act + slot);
                    keep = nm_consume(P, id, S);
                }
                warp_append(keep, id, next_list, next_count);
            }
        }
        grid.sync();
    }
}

template <int MODE, int UNR>
static cudaError_t launch_fused(const FusedParams& p, int sm_count, cudaStream_t st) {
    auto kern = solve_nm_fused_kernel<MODE, UNR>;
    // per launch: the attribute belongs to the current device's copy of the kernel
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kFusedSmem);
    if (e != cudaSuccess) return e;
    int blocks_per_sm = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&blocks_per_sm, kern, kFusedThreads, kFusedSmem);
    if (e != cudaSuccess) return e;
    if (blocks_per_sm < 1) return cudaErrorLaunchOutOfResources;
    if (blocks_per_sm > kFusedMinB) blocks_per_sm = kFusedMinB;
    FusedParams q = p;
    // The grid must be co-resident.  sm_count is the device's; a context that may use only part of the SMs (MPS with
    // an active-thread percentage, a green context, a profiler holding SMs back) refuses that grid with
    // cudaErrorCooperativeLaunchTooLarge: shrink it by an eighth of the device at a time until it is accepted.  Work
    // items come from an atomic counter and sums are added in canonical chunk order, so any grid gives the same bits.
    const int full = sm_count * blocks_per_sm;
    const int dec = full / 8 > 0 ? full / 8 : 1;
    for (int grid = full; grid >= 1; grid -= dec) {
        q.warp_items_max = 11 * grid;   // warp shape while its items fit ~11 rounds of the grid (one item costs ~1/11 of a thread-shape item)
        void* args[] = {(void*)&q};
        e = cudaLaunchCooperativeKernel((const void*)kern, dim3(grid), dim3(kFusedThreads), args, kFusedSmem, st);
        if (e != cudaErrorCooperativeLaunchTooLarge) return e;
        (void)cudaGetLastError();       // not sticky: try a smaller grid
    }
    return cudaErrorCooperativeLaunchTooLarge;
}

cudaError_t launch_solve_nm_fused(const FusedParams& p, int sm_count, int* launches, cudaStream_t st) {
    if (p.count <= 0) return cudaSuccess;
    if (launches) *launches += 1;
    return p.k.analytic ? launch_fused<MODE_ANALYTIC, 4>(p, sm_count, st) : launch_fused<MODE_STENCIL4, 2>(p, sm_count, st);
}

}  // namespace dbie
