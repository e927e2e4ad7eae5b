// dbie_internal.h — structures shared by the translation units of libdbie_b200.so.
// Not part of the public ABI (that is include/dbie.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/dbie.h"
#include "dbie_nm.cuh"

namespace dbie {

constexpr int kTilePx = 512;     // pixels staged in shared memory at a time (16 KB fp64 records)
constexpr int kMaxChunks = 16;   // canonical partial sums per evaluation point
constexpr int kStencil = 4;      // r_i, r_i + delta x, + delta y, + delta z (Eq. 13, reading A-5)

// Device view of the boundary as staged by dbie_create.
// rec[k] = {x_k, Bx0[k], By0[k], Bz0[k]} (32 B, one LDS.128 pair per pixel), k = iy*nx + ix;
// yk[iy] = y0 + (iy + 1/2) h.  x_k, y_k are formed as x0 + (ix + 0.5)*h with separately rounded
// multiply and add, the order the paper's definition of a pixel centre (reading A-1) is
// written in DESIGN.md.
struct BoundaryView {
    int nx, ny;
    long long N;
    double h, x0, y0;
    const double4* rec;
    const double* yk;
    const float4* rec32;   // fp32 copy {x_k, Bx0, By0, Bz0} or nullptr
    const float* yk32;
    // tiling: a tile is `tile_rows` full rows (nx <= kTilePx) or one row segment of
    // `seg_w` columns (nx > kTilePx); a chunk is a run of consecutive UNITS, a unit being one row
    // (or one row segment): nunits = ny * segs_per_row.  Chunk boundaries may fall inside a tile
    // (small boundaries: 64 x 64 has 8 tiles of 8 rows and 16 chunks of 4 rows).
    int tile_rows, segs_per_row, seg_w;
    int ntiles, nunits, nchunks;
};

struct TileDesc {
    int row0, nrows, col0, ncols;
    long long px0;   // index of the first record (tiles are contiguous in rec[])
    int npx;
};

__host__ __device__ inline TileDesc tile_desc(const BoundaryView& b, int t) {
    TileDesc d;
    if (b.segs_per_row == 1) {
        d.row0 = t * b.tile_rows;
        d.nrows = (b.ny - d.row0 < b.tile_rows) ? (b.ny - d.row0) : b.tile_rows;
        d.col0 = 0;
        d.ncols = b.nx;
    } else {
        d.row0 = t / b.segs_per_row;
        d.nrows = 1;
        d.col0 = (t % b.segs_per_row) * b.seg_w;
        d.ncols = (b.nx - d.col0 < b.seg_w) ? (b.nx - d.col0) : b.seg_w;
    }
    d.px0 = (long long)d.row0 * b.nx + d.col0;
    d.npx = d.nrows * d.ncols;
    return d;
}

// first unit (row, or row segment when nx > kTilePx) of canonical chunk c; chunk nchunks starts at nunits
__host__ __device__ inline int chunk_first_unit(const BoundaryView& b, int c) {
    return (int)(((long long)c * b.nunits) / b.nchunks);
}
// the tile that holds unit u
__host__ __device__ inline int unit_tile(const BoundaryView& b, int u) {
    return (b.segs_per_row == 1) ? u / b.tile_rows : u;
}

// One launch of the interaction kernel.
//  MODE_EVAL:    slot i = evaluation point i with its own lambda triple; Q = 3 sums.
//  MODE_STENCIL4 / MODE_ANALYTIC: slot j = one objective evaluation of field point pid = act ? act[j] : j
//                with ONE lambda triple: the 4 stencil positions of Eq. 13, Q = 12 sums [s*3 + p], or the
//                four sums of the analytic gradient (O-5), Q = 12 sums [kind*3 + p].
// Partial sums go to part[(c*Q + q)*cap + slot], one per chunk c, and are added in chunk order
// by the consumer, so a result does not depend on how the launch was split.
struct InteractParams {
    BoundaryView bd;
    const double *x, *y, *z;     // by point id
    const double* lam;           // lam[p*ldlam + id]
    long long ldlam;
    const int* act;              // solver modes: slot -> point id, or nullptr (identity)
    const unsigned* count_ptr;   // device-resident slot count, or nullptr
    long long count;             // host-known slot count (used when count_ptr == nullptr)
    long long slot0;             // MODE_EVAL: id of slot 0 (batching)
    double delta_abs;            // finite-difference step of Eq. 13 (length units)
    double* part;
    long long cap;
    int target_items;            // split the pixel range until there are this many work items
    unsigned* zero_ptr;          // set to 0 by the launch (the next pass's list counter), or nullptr
    unsigned* work_ctr;          // persistent grid: atomic work-item counter (zero on entry), or nullptr
    unsigned* zero_work;         // set to 0 by the launch (the next pass's work counter), or nullptr
    // MODE_GRID (O-4): trial t of component c at point id is lo[c*ldlo + id] + W t/(T-1)
    const double* lo;
    long long ldlo;
    double W;
    double dlam;                 // W/(T-1): spacing of the trial values
    int T;
};

// One launch of the fp32 eval kernel (dbie_eval_f32): slot i = evaluation point slot0 + i.
struct InteractParamsF32 {
    BoundaryView bd;
    const float *x, *y, *z;
    const float* lam;            // lam[p*ldlam + id]
    long long ldlam;
    long long count, slot0;
    double* part;                // fp64 chunk sums, part[(c*3 + q)*cap + slot]
    long long cap;
    int target_items;
};

struct SolveArrays {            // per-point optimiser state, structure-of-arrays by point id
    double* V;                  // [12][M]  simplex vertices V[(j*3+p)*M + i]
    double* F;                  // [4][M]   Phi at the vertices
    double* aux;                // [20][M]  (Bx,By,Bz,f,g) at the vertices, aux[(j*5+a)*M + i]
    double* pend;               // [9][M]   reflection point kept while its follow-up is evaluated
    double* cand;               // [3][M]   lambda triple of the outstanding evaluation
    int* phase;                 // [M]
    int* iters;                 // [M]
    int* act[2];                // active lists (ping-pong)
    unsigned* nact;             // [2] device counters
};

// The fused Nelder-Mead solve (dbie_solve_fused.cu): ONE cooperative launch runs every pass of the search.
// List and work counters rotate over three slots: pass p consumes [p % 3], fills [(p+1) % 3] and clears
// [(p+2) % 3], so no counter is cleared while another CTA may still read or bump it.
struct FusedParams {
    InteractParams ip;          // bd, x, y, z, lam = s.cand, ldlam = count, delta_abs, part, cap, target_items
    SolveArrays s;              // s.act[2]: ping-pong lists; s.nact is unused here (nact3)
    NMConsts k;
    long long count, ldo;       // points of the batch; stride of the caller's output arrays
    double *B, *lam, *resid;
    int *iters, *status;
    unsigned long long* nevals;
    unsigned* nact3;            // [3] list lengths
    unsigned* work3;            // [3] work-item counters
    unsigned* done;             // [cap/4 + 2] arrivals per point block (thread mode) / point group (warp mode)
    int maxpass;
    int warp_items_max;         // warp-per-point path when ceil(n/4) * nchunks <= this
    unsigned long long* trace;  // profile mode: [2*(trace_cap)] (active points, %globaltimer ns) at the start of every
    int trace_cap;              //   pass and at the end of the search; nullptr otherwise
};

struct GridArrays {             // per-point GRID state (O-4), structure-of-arrays by point id
    double* lo;                 // [3][cap]  lower end of the current window per component
    double* inc;                // [12][cap] B at the 4 stencil positions for the incumbent, [s*3+p]
    double* il;                 // [3][cap]  incumbent lambda
    long long cap;
    int* act[2];                // active lists (ping-pong)
    unsigned* nact;             // [2] device counters
};

// Line tracing (dbie_trace.cu): per-line state, structure-of-arrays over L lines
struct TraceState {
    double* r;                  // [3][L] current point r_n
    double* k;                  // [3 stages][3][L] k1..k3 (k4 is consumed at once)
    double *px, *py, *pz;       // [L] the stage point handed to the field evaluation (z = -1: skip)
    int *alive, *good, *why;    // [L] line still traced; still integrating this step; stop reason if not
};
struct TraceBox {
    double x0, x1, y0, y1, z0, z1;   // region: x0 <= x <= x1, y0 <= y <= y1, z0 < z <= z1
};

struct GridConsts {
    int T, n_level;
    double W, Wn;               // this level's window width and the next one, 2 W/(T-1)
    double Lmax;                // lam_max / h
};

constexpr int kGridMaxTrials = 32;

// launchers (defined in the .cu files; all asynchronous on `st`)
cudaError_t launch_stage_boundary(int nx, int ny, double h, double x0, double y0, const double* bx,
                                  const double* by, const double* bz, double4* rec, double* yk,
                                  float4* rec32, float* yk32, cudaStream_t st);
cudaError_t launch_stage_q9(int nx, int ny, double h, double x0, double y0, const double* bx, const double* by,
                            const double* bz, int nsx, int nsy, double4* rec, double* yk, float4* rec32,
                            float* yk32, cudaStream_t st);
cudaError_t launch_interact_eval(const InteractParams& p, int sm_count, bool reduced_sincos, int* nparts,
                                 cudaStream_t st);
cudaError_t launch_interact_stencil(const InteractParams& p, int sm_count, cudaStream_t st);
cudaError_t launch_interact_grid(const InteractParams& p, int sm_count, cudaStream_t st);
cudaError_t launch_interact_analytic(const InteractParams& p, int sm_count, cudaStream_t st);
cudaError_t launch_interact_grid_analytic(const InteractParams& p, int sm_count, cudaStream_t st);
cudaError_t launch_eval_finalize(const BoundaryView& bd, int nparts, long long slot0, long long count,
                                 long long M, const double* z, const double* lam, const double* part,
                                 long long cap, double* B, cudaStream_t st);
cudaError_t launch_interact_f32(const InteractParamsF32& p, int sm_count, int sfu_mask, int* nparts, cudaStream_t st);
cudaError_t launch_eval_finalize_f32(const BoundaryView& bd, int nparts, long long slot0, long long count, long long M,
                                     const float* z, const float* lam, const double* part, long long cap,
                                     float* B, cudaStream_t st);
cudaError_t launch_probe(double millis, int sm_count, double* dfma_per_s, double* ffma_per_s);
cudaError_t launch_operand_probe(double millis, int sm_count, double rates[4]);

cudaError_t launch_solve_init(const SolveArrays& s, const NMConsts& k, long long M, long long ldo,
                              const double* x, const double* y, const double* z, double* B, double* lam,
                              double* resid, int* iters, int* status, cudaStream_t st);
cudaError_t launch_solve_nm_fused(const FusedParams& p, int sm_count, int* launches, cudaStream_t st);
cudaError_t launch_residual_finalize(const BoundaryView& bd, const NMConsts& k, long long M,
                                     long long ldo, const double* z, const double* part, long long cap,
                                     double* out, double* phi, cudaStream_t st);

cudaError_t launch_grid_init(const GridArrays& s, long long M, long long ldo, const double* x, const double* y,
                             const double* z, double* B, double* lam, double* resid, int* iters, int* status,
                             cudaStream_t st);
cudaError_t launch_grid_step(const GridArrays& s, const NMConsts& k, const GridConsts& gc, const BoundaryView& bd,
                             int lev, long long M, long long ldo, const double* z, const double* part,
                             long long cap, double* B, double* lam, double* resid, int* iters, int* status,
                             unsigned long long* nevals, cudaStream_t st);

cudaError_t launch_trace_init(const TraceState& t, const TraceBox& box, long long L, int S, const double* sx,
                              const double* sy, const double* sz, double* path, int* npts, int* status,
                              cudaStream_t st);
cudaError_t launch_trace_stage(const TraceState& t, const TraceBox& box, long long L, int S, int step, int stage,
                               int direction, double ds, const double* v, long long ldv, double* path, int* npts,
                               int* status, cudaStream_t st);
cudaError_t launch_trace_fill_lambda(double* lam, long long L, const double l[3], cudaStream_t st);

}  // namespace dbie
