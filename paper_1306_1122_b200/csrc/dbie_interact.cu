// dbie_interact.cu — the M x N point-pixel interaction kernel.
//
//   B_p(i) = (z_i h^2/2pi) sum_k [theta sin theta + cos theta]/r^3 * B_p0[k],  theta = |lambda_p| r
//   (Eq. 6, Eq. 16).
//
// This file holds the boundary staging kernel, the launchers of the fp64 interaction kernel
// (dbie_interact_fp64.cuh), the fp32 eval kernel, the eval epilogues and the pipe-rate probe.
// The bound is the FP64 pipe; there are no tensor-core or HBM-bound steps.
#include <cuda_runtime.h>
#include <stdint.h>

#include "dbie_internal.h"
#include "dbie_interact_fp64.cuh"
#include "dbie_math.cuh"
#include "dbie_math_f32.cuh"
#include "dbie_tma.cuh"

namespace dbie {

// ------------------------------------------------------------------ boundary staging ------
// A1: rec[k] = {x_k, Bx0, By0, Bz0}; x_k = x0 + (ix + 1/2) h, multiply and add rounded separately.
__global__ void stage_boundary_kernel(int nx, int ny, double h, double x0, double y0,
                                      const double* __restrict__ bx, const double* __restrict__ by,
                                      const double* __restrict__ bz, double4* __restrict__ rec,
                                      double* __restrict__ yk, float4* __restrict__ rec32,
                                      float* __restrict__ yk32) {
    const long long N = (long long)nx * ny;
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < N;
         k += (long long)gridDim.x * blockDim.x) {
        const int ix = (int)(k % nx);
        const double xk = __dadd_rn(x0, __dmul_rn((double)ix + 0.5, h));
        rec[k] = make_double4(xk, bx[k], by[k], bz[k]);
        if (rec32) rec32[k] = make_float4((float)xk, (float)bx[k], (float)by[k], (float)bz[k]);
        if (k < ny) {
            const double y = __dadd_rn(y0, __dmul_rn((double)k + 0.5, h));
            yk[k] = y;
            if (yk32) yk32[k] = (float)y;
        }
    }
}

cudaError_t launch_stage_boundary(int nx, int ny, double h, double x0, double y0, const double* bx,
                                  const double* by, const double* bz, double4* rec, double* yk,
                                  float4* rec32, float* yk32, cudaStream_t st) {
    const long long N = (long long)nx * ny;
    int grid = (int)((N + 255) / 256);
    if (grid > 4096) grid = 4096;
    stage_boundary_kernel<<<grid, 256, 0, st>>>(nx, ny, h, x0, y0, bx, by, bz, rec, yk, rec32, yk32);
    return cudaGetLastError();
}

// A1, 9-node element variant (Eq. 15; O-6): the nodes are
// the pixel centres, an element spans 3 x 3 of them (2h x 2h), biquadratic Lagrange shape functions,
// 3 x 3 Gauss-Legendre points.  Eq. 15 is then Eq. 16's sum over a tensor grid of Gauss-point sources
// with values w_g sum_j N_j(g) B_j: this kernel writes that grid in the same record layout, so the
// interaction kernels run on it unchanged (rec[].x and yk[] are explicit coordinates already).
struct Q9Axis {
    double pos, w, N[3];
    int base;
};
// Gauss abscissa `k` of an axis with n nodes whose first node sits at c0 + h/2.  When n is even the
// last element re-uses the last three nodes and is integrated over its outer half only.
__device__ inline Q9Axis q9_axis(int n, double c0, double h, int k) {
    const int e = k / 3, q = k - 3 * e;
    const double g = (q == 0) ? -0.7745966692414834 : (q == 1 ? 0.0 : 0.7745966692414834);   // sqrt(3/5)
    const double w = (q == 1) ? 8.0 / 9.0 : 5.0 / 9.0;
    const bool half = 2 * e + 2 > n - 1;
    Q9Axis a;
    a.base = half ? n - 3 : 2 * e;
    const double xi = half ? 0.5 + 0.5 * g : g;
    a.pos = c0 + ((double)(a.base + 1) + 0.5) * h + xi * h;
    a.w = half ? 0.5 * w : w;
    a.N[0] = 0.5 * xi * (xi - 1.0);
    a.N[1] = 1.0 - xi * xi;
    a.N[2] = 0.5 * xi * (xi + 1.0);
    return a;
}

__global__ void stage_q9_kernel(int nx, int ny, double h, double x0, double y0, const double* __restrict__ bx,
                                const double* __restrict__ by, const double* __restrict__ bz, int nsx, int nsy,
                                double4* __restrict__ rec, double* __restrict__ yk, float4* __restrict__ rec32,
                                float* __restrict__ yk32) {
    const long long NS = (long long)nsx * nsy;
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < NS;
         k += (long long)gridDim.x * blockDim.x) {
        const int gy = (int)(k / nsx), gx = (int)(k - (long long)gy * nsx);
        const Q9Axis ax = q9_axis(nx, x0, h, gx), ay = q9_axis(ny, y0, h, gy);
        double v[3] = {0.0, 0.0, 0.0};
        for (int b = 0; b < 3; ++b)
            for (int a = 0; a < 3; ++a) {
                const long long j = (long long)(ay.base + b) * nx + ax.base + a;
                const double Nab = ay.N[b] * ax.N[a];
                v[0] += Nab * bx[j];
                v[1] += Nab * by[j];
                v[2] += Nab * bz[j];
            }
        const double w = ay.w * ax.w;
        rec[k] = make_double4(ax.pos, w * v[0], w * v[1], w * v[2]);
        if (rec32) rec32[k] = make_float4((float)ax.pos, (float)(w * v[0]), (float)(w * v[1]), (float)(w * v[2]));
        if (gx == 0) {
            yk[gy] = ay.pos;
            if (yk32) yk32[gy] = (float)ay.pos;
        }
    }
}

cudaError_t launch_stage_q9(int nx, int ny, double h, double x0, double y0, const double* bx, const double* by,
                            const double* bz, int nsx, int nsy, double4* rec, double* yk, float4* rec32,
                            float* yk32, cudaStream_t st) {
    const long long NS = (long long)nsx * nsy;
    int grid = (int)((NS + 255) / 256);
    if (grid > 4096) grid = 4096;
    stage_q9_kernel<<<grid, 256, 0, st>>>(nx, ny, h, x0, y0, bx, by, bz, nsx, nsy, rec, yk, rec32, yk32);
    return cudaGetLastError();
}

// ------------------------------------------------------------------ fp64 launchers --------
// The kernel is dbie_interact_fp64.cuh.  Shapes measured on B200 (round-1 shape sweep, re-checked in round 2):
// 256 threads x 2 CTAs/SM (<= 128 registers), two pixels in flight per thread; GRID mode carries
// 4 (else 2, else 1) trial lambda triples per thread on one geometry.
constexpr int kThreads64 = 256, kMinB64 = 2;

template <int MODE, int NT, int UNR, int THREADS = kThreads64, int MINB = kMinB64>
static cudaError_t launch64(const InteractParams& p, int sm_count, int waves, cudaStream_t st) {
    InteractParams q = p;
    q.target_items = waves * sm_count * MINB;
    long long grid;
    if (q.count_ptr) {
        grid = (long long)sm_count * MINB;   // persistent: the slot count lives on the device
    } else {
        if (q.count <= 0) return cudaSuccess;
        const int G = (MODE == MODE_GRID || MODE == MODE_GRID_ANALYTIC) ? q.T / NT : 1;
        const long long nitems = q.count * items_per_slot(MODE, G);
        const long long nblk = (nitems + THREADS - 1) / THREADS;
        long long nsplit = 1;
        if (nblk < q.target_items) {
            nsplit = (q.target_items + nblk - 1) / nblk;
            if (nsplit > q.bd.nchunks) nsplit = q.bd.nchunks;
        }
        grid = nblk * nsplit;   // one work item per CTA: the hardware balances them
        if (grid > 0x7fffffffLL) return cudaErrorInvalidValue;
    }
    auto kern = interact64_kernel<MODE, NT, THREADS, MINB, UNR>;
    // per launch: the attribute belongs to the current device's copy of the kernel
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kInteractSmem);
    if (e != cudaSuccess) return e;
    kern<<<(unsigned)grid, THREADS, kInteractSmem, st>>>(q);
    return cudaGetLastError();
}

// *nparts: how many chunk slots the launch fills per output (1 when every CTA covers all chunks and adds
// them itself, else nchunks); the epilogue adds exactly that many, in chunk order.
cudaError_t launch_interact_eval(const InteractParams& p, int sm_count, bool reduced_sincos, int* nparts,
                                 cudaStream_t st) {
    const long long nblk = (p.count + kThreads64 - 1) / kThreads64;
    *nparts = (nblk >= 8LL * sm_count * kMinB64 || p.bd.nchunks == 1) ? 1 : p.bd.nchunks;
    // four pixels in flight (developer sweep at 512 x 512, M = 1,048,576: u1 1098 ms, u2 1081, u3 1088, u4 1071)
    if (reduced_sincos) return launch64<MODE_EVAL_R, 1, 4>(p, sm_count, 8, st);
    return launch64<MODE_EVAL, 1, 4>(p, sm_count, 8, st);
}

cudaError_t launch_interact_stencil(const InteractParams& p, int sm_count, cudaStream_t st) {
    // all 4 stencil positions of a point in one thread (one sincos per component, kernel_n_near for the offsets), two pixels in
    // flight: 128 threads x 2 CTAs/SM; +35 % over one position per thread (MODE_STENCIL, round-1 shape sweep)
    return launch64<MODE_STENCIL4, 1, 2, 128, 2>(p, sm_count, 16, st);
}

cudaError_t launch_interact_analytic(const InteractParams& p, int sm_count, cudaStream_t st) {
    return launch64<MODE_ANALYTIC, 1, 4, 128, 2>(p, sm_count, 16, st);
}

cudaError_t launch_interact_grid_analytic(const InteractParams& p, int sm_count, cudaStream_t st) {
    // two trial triples per thread share the geometry (79 instead of 86 instructions per interaction);
    // 24 accumulators + 2 x 6 lambda, lambda^2: 128 threads x 2 CTAs/SM (10 % faster than x 3 at 168 registers)
    if (p.T < 2) return cudaErrorInvalidValue;
    if (p.T % 2 == 0) return launch64<MODE_GRID_ANALYTIC, 2, 1, 128, 2>(p, sm_count, 16, st);
    return launch64<MODE_GRID_ANALYTIC, 1, 2>(p, sm_count, 16, st);
}

cudaError_t launch_interact_grid(const InteractParams& p, int sm_count, cudaStream_t st) {
    if (p.T < 2) return cudaErrorInvalidValue;
    // NT > 1 shares (sin, cos)(j d_theta) between the trials, which needs window starts lo >= 0 (dbie_solve accepts T >= 4 only)
    // 8 trial triples per thread need 234 registers: 128 threads x 2 CTAs/SM (round-1 shape sweep)
    if (p.T % 8 == 0) return launch64<MODE_GRID, 8, 1, 128, 2>(p, sm_count, 16, st);
    if (p.T % 4 == 0) return launch64<MODE_GRID, 4, 1, 128, 3>(p, sm_count, 16, st);
    if (p.T % 2 == 0 && p.T > 2) return launch64<MODE_GRID, 2, 2>(p, sm_count, 16, st);
    return launch64<MODE_GRID, 1, 2>(p, sm_count, 16, st);
}

// ------------------------------------------------------------------ fp32 eval kernel ------
// dbie_eval_f32 (BASELINE.json config 4, fp32 leg): geometry, theta, sincos and products in fp32;
// a row segment (<= 512 pixels) is summed in fp32, row sums are carried in fp64.
// SFU_MASK bit p set: component p takes sin/cos of the reduced argument from MUFU.SIN/COS, else from the
// angle table in shared memory (dbie_math_f32.cuh), to balance the SFU against the issue port (SURVEY 8(d)
// "fp32 variant").  Shared memory (dynamic): [fp32 angle table, 16 copies, 32 KB][2 tiles, 16 KB][mbarriers].
template <int R, int THREADS, int MINB, int SFU_MASK>
__global__ void __launch_bounds__(THREADS, MINB) interact_f32_kernel(const __grid_constant__ InteractParamsF32 p) {
    constexpr int SPB = THREADS * R;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float4(*tile)[kTilePx] = reinterpret_cast<float4(*)[kTilePx]>(smem_raw + kTrigTableBytesF);
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + kTrigTableBytesF + sizeof(float4) * 2 * kTilePx);

    const int tid = threadIdx.x;
    if (tid == 0) {
        mbar_init(&full[0], 1);
        mbar_init(&full[1], 1);
        mbar_fence_init();
    }
    TrigEntryF* tab = reinterpret_cast<TrigEntryF*>(smem_raw);
    if (SFU_MASK != 7) {   // some component reads the table
        for (int i = tid; i < DBIE_TRIG_ENTRIES * kTrigCopiesF; i += THREADS) tab[i] = kTrigTabGF[i / kTrigCopiesF];
    }
    const TrigRefF tr{tab, (unsigned)(tid & (kTrigCopiesF - 1)) * (unsigned)sizeof(TrigEntryF)};
    __syncthreads();

    const long long count = p.count;
    const long long nblk = (count + SPB - 1) / SPB;
    const BoundaryView& bd = p.bd;
    const int NCH = bd.nchunks;
    int nsplit = 1;
    if (nblk < p.target_items) {
        nsplit = (int)((p.target_items + nblk - 1) / nblk);
        if (nsplit > NCH) nsplit = NCH;
    }
    const long long nwork = nblk * nsplit;

    unsigned it = 0;
    for (long long w = blockIdx.x; w < nwork; w += gridDim.x) {
        const long long blk = w / nsplit;
        const int sp = (int)(w % nsplit);
        const int c0 = (int)(((long long)sp * NCH) / nsplit);
        const int c1 = (int)(((long long)(sp + 1) * NCH) / nsplit);

        float xi[R], yi[R], z2[R], lam[R][3];
        long long slot[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            slot[r] = blk * SPB + tid + (long long)r * THREADS;
            const long long id = p.slot0 + (slot[r] < count ? slot[r] : count - 1);
            xi[r] = p.x[id];
            yi[r] = p.y[id];
            const float z = p.z[id];
            z2[r] = z * z;
#pragma unroll
            for (int c = 0; c < 3; ++c) lam[r][c] = fabsf(p.lam[c * p.ldlam + id]);
        }
        double acc[R][3], run[R][3];   // run: running sum of the chunk sums of an unsplit launch
#pragma unroll
        for (int r = 0; r < R; ++r) acc[r][0] = acc[r][1] = acc[r][2] = 0.0;

        const int u0 = chunk_first_unit(bd, c0), u1 = chunk_first_unit(bd, c1);   // as in the fp64 interact_item
        const int t0 = unit_tile(bd, u0), t1 = unit_tile(bd, u1 - 1) + 1;
        int c = c0;
        int u_chunk_end = chunk_first_unit(bd, c + 1);
        if (tid == 0) {
            const TileDesc d = tile_desc(bd, t0);
            mbar_expect_tx(&full[it & 1], (unsigned)d.npx * 16u);
            bulk_g2s(&tile[it & 1][0], bd.rec32 + d.px0, (unsigned)d.npx * 16u, &full[it & 1]);
        }
        for (int t = t0; t < t1; ++t, ++it) {
            if (tid == 0 && t + 1 < t1) {
                const TileDesc dn = tile_desc(bd, t + 1);
                const unsigned sn = (it + 1) & 1;
                mbar_expect_tx(&full[sn], (unsigned)dn.npx * 16u);
                bulk_g2s(&tile[sn][0], bd.rec32 + dn.px0, (unsigned)dn.npx * 16u, &full[sn]);
            }
            const TileDesc d = tile_desc(bd, t);
            mbar_wait(&full[it & 1], (it >> 1) & 1);
            const float4* __restrict__ rp = &tile[it & 1][0];
            for (int row = 0; row < d.nrows; ++row, rp += d.ncols) {
                const int unit = (bd.segs_per_row == 1) ? d.row0 + row : t;
                if (unit < u0 || unit >= u1) continue;   // a row of a neighbouring chunk in a shared tile
                const float yk = __ldg(bd.yk32 + d.row0 + row);
                float cc[R], a32[R][3];
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const float dy = yk - yi[r];
                    cc[r] = fmaf(dy, dy, z2[r]);
                    a32[r][0] = a32[r][1] = a32[r][2] = 0.0f;
                }
#pragma unroll 2
                for (int j = 0; j < d.ncols; ++j) {
                    const float4 px = rp[j];  // {x_k, Bx0, By0, Bz0}: one broadcast LDS.128
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        const float dx = px.x - xi[r];
                        const float r2 = fmaf(dx, dx, cc[r]);
                        const float y = rsqrt_f32(r2);
                        const float rr = r2 * y;
                        const float wgt = (y * y) * y;
                        a32[r][0] = fmaf(kernel_n_f32<(SFU_MASK & 1) != 0>(lam[r][0] * rr, tr), wgt * px.y, a32[r][0]);
                        a32[r][1] = fmaf(kernel_n_f32<(SFU_MASK & 2) != 0>(lam[r][1] * rr, tr), wgt * px.z, a32[r][1]);
                        a32[r][2] = fmaf(kernel_n_f32<(SFU_MASK & 4) != 0>(lam[r][2] * rr, tr), wgt * px.w, a32[r][2]);
                    }
                }
#pragma unroll
                for (int r = 0; r < R; ++r)
#pragma unroll
                    for (int q = 0; q < 3; ++q) acc[r][q] += (double)a32[r][q];
                if (unit + 1 != u_chunk_end) continue;
                if (nsplit == 1) {   // unsplit launch: add the chunk sums here, in chunk order (as the epilogue would)
#pragma unroll
                    for (int r = 0; r < R; ++r)
#pragma unroll
                        for (int q = 0; q < 3; ++q) run[r][q] = (c == 0) ? acc[r][q] : __dadd_rn(run[r][q], acc[r][q]);
                    if (c == NCH - 1) {
#pragma unroll
                        for (int r = 0; r < R; ++r)
                            if (slot[r] < count) {
#pragma unroll
                                for (int q = 0; q < 3; ++q) p.part[(long long)q * p.cap + slot[r]] = run[r][q];
                            }
                    }
                } else {
#pragma unroll
                    for (int r = 0; r < R; ++r)
                        if (slot[r] < count) {
#pragma unroll
                            for (int q = 0; q < 3; ++q) p.part[((long long)c * 3 + q) * p.cap + slot[r]] = acc[r][q];
                        }
                }
#pragma unroll
                for (int r = 0; r < R; ++r) acc[r][0] = acc[r][1] = acc[r][2] = 0.0;
                ++c;
                u_chunk_end = chunk_first_unit(bd, c + 1);
            }
            __syncthreads();
        }
    }
}

constexpr int kF32R = 4, kF32Threads = 128, kF32MinB = 4;

template <int MASK>
static cudaError_t launch_f32_variant(const InteractParamsF32& q, unsigned grid, cudaStream_t st) {
    auto kern = interact_f32_kernel<kF32R, kF32Threads, kF32MinB, MASK>;
    constexpr size_t smem = kTrigTableBytesF + sizeof(float4) * 2 * kTilePx + 64;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    kern<<<grid, kF32Threads, smem, st>>>(q);
    return cudaGetLastError();
}

cudaError_t launch_interact_f32(const InteractParamsF32& p, int sm_count, int sfu_mask, int* nparts, cudaStream_t st) {
    *nparts = p.bd.nchunks;
    if (p.count <= 0) return cudaSuccess;
    InteractParamsF32 q = p;
    const long long spb = (long long)kF32Threads * kF32R;
    const long long nblk = (q.count + spb - 1) / spb;
    q.target_items = 8 * sm_count * kF32MinB;
    long long nsplit = 1;
    if (nblk < q.target_items) {
        nsplit = (q.target_items + nblk - 1) / nblk;
        if (nsplit > q.bd.nchunks) nsplit = q.bd.nchunks;
    }
    *nparts = (nsplit == 1) ? 1 : q.bd.nchunks;
    const long long nwork = nblk * nsplit;
    if (nwork > 0x7fffffffLL) return cudaErrorInvalidValue;
    switch (sfu_mask & 7) {
        case 0: return launch_f32_variant<0>(q, (unsigned)nwork, st);
        case 1: return launch_f32_variant<1>(q, (unsigned)nwork, st);
        case 3: return launch_f32_variant<3>(q, (unsigned)nwork, st);
        case 7: return launch_f32_variant<7>(q, (unsigned)nwork, st);
        default: return cudaErrorInvalidValue;
    }
}

// B_p = (z h^2 / 2 pi) * (chunk sums in chunk order), fp64 arithmetic, rounded to float once.
__global__ void eval_finalize_f32_kernel(int nchunks, double h2_over_2pi, long long slot0, long long count,
                                         long long M, const float* __restrict__ z,
                                         const float* __restrict__ lam, const double* __restrict__ part,
                                         long long cap, float* __restrict__ B) {
    const long long s = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (s >= count) return;
    const long long id = slot0 + s;
    const float zi = z[id];
    bool ok = (zi > 0.0f) && isfinite(zi);
    float out[3];
#pragma unroll
    for (int q = 0; q < 3; ++q) {
        double sum = part[(long long)q * cap + s];
        for (int c = 1; c < nchunks; ++c) sum += part[((long long)c * 3 + q) * cap + s];
        out[q] = (float)(((double)zi * h2_over_2pi) * sum);
        ok = ok && isfinite(lam[q * M + id]);
    }
#pragma unroll
    for (int q = 0; q < 3; ++q) B[q * M + id] = ok ? out[q] : __int_as_float(0x7fc00000);
}

cudaError_t launch_eval_finalize_f32(const BoundaryView& bd, int nparts, long long slot0, long long count, long long M,
                                     const float* z, const float* lam, const double* part, long long cap,
                                     float* B, cudaStream_t st) {
    if (count <= 0) return cudaSuccess;
    const double h2_over_2pi = bd.h * bd.h / (2.0 * 3.14159265358979323846);
    const unsigned grid = (unsigned)((count + 255) / 256);
    eval_finalize_f32_kernel<<<grid, 256, 0, st>>>(nparts, h2_over_2pi, slot0, count, M, z, lam, part, cap, B);
    return cudaGetLastError();
}

// ------------------------------------------------------------------ eval epilogue ---------
// A4: B_p = (z h^2 / 2 pi) * (sum of the chunk partial sums, in chunk order).
__global__ void eval_finalize_kernel(int nchunks, double h2_over_2pi, long long slot0, long long count,
                                     long long M, const double* __restrict__ z,
                                     const double* __restrict__ lam, const double* __restrict__ part,
                                     long long cap, double* __restrict__ B) {
    const long long s = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (s >= count) return;
    const long long id = slot0 + s;
    const double zi = z[id];
    bool ok = (zi > 0.0) && isfinite(zi);
    double out[3];
#pragma unroll
    for (int q = 0; q < 3; ++q) {
        double sum = part[(long long)q * cap + s];
        for (int c = 1; c < nchunks; ++c) sum += part[((long long)c * 3 + q) * cap + s];
        out[q] = (zi * h2_over_2pi) * sum;
        ok = ok && isfinite(lam[q * M + id]);
    }
#pragma unroll
    for (int q = 0; q < 3; ++q) B[q * M + id] = ok ? out[q] : __longlong_as_double(0x7ff8000000000000LL);
}

cudaError_t launch_eval_finalize(const BoundaryView& bd, int nparts, long long slot0, long long count, long long M,
                                 const double* z, const double* lam, const double* part, long long cap,
                                 double* B, cudaStream_t st) {
    if (count <= 0) return cudaSuccess;
    const double h2_over_2pi = bd.h * bd.h / (2.0 * 3.14159265358979323846);
    const unsigned grid = (unsigned)((count + 255) / 256);
    eval_finalize_kernel<<<grid, 256, 0, st>>>(nparts, h2_over_2pi, slot0, count, M, z, lam, part, cap, B);
    return cudaGetLastError();
}

// ------------------------------------------------------------------ pipe-rate probe -------
// Register-only FMA chains: the measured denominator of the ALU roofline.
template <typename T>
__global__ void __launch_bounds__(256) fma_probe_kernel(int iters, T seed, T* sink) {
    T a[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) a[i] = seed + (T)(threadIdx.x + i);
    const T m = (T)0.999999, c = (T)1e-7;
    for (int k = 0; k < iters; ++k) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
#pragma unroll
            for (int i = 0; i < 8; ++i) a[i] = fma(a[i], m, c);
        }
    }
    T s = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += a[i];
    if (s == (T)-1.2345) sink[0] = s;  // never true; keeps the chains alive
}

// FP64 operand patterns: KIND 0 = DFMA with two register operands and an immediate,
// 1 = DFMA whose three operands are three different, changing registers, 2 = DMUL, 3 = DFMA with one changing and
// two loop-invariant register operands (served by the operand-reuse cache).
template <int KIND>
__global__ void __launch_bounds__(256) fp64_operand_probe_kernel(int iters, double seed, double* sink) {
    double a[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) a[i] = seed + 1e-9 * (double)(threadIdx.x + i);
    const double m = seed * 0.999999, c = seed * 1e-7;
    for (int k = 0; k < iters; ++k) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                if (KIND == 0) a[i] = fma(a[i], m, 0.5);
                if (KIND == 1) a[i] = fma(a[i], a[(i + 1) & 7], a[(i + 2) & 7]);
                if (KIND == 2) a[i] = a[i] * m;
                if (KIND == 3) a[i] = fma(a[i], m, c);
            }
        }
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += a[i];
    if (s == -1.2345) sink[0] = s;  // never true; keeps the chains alive
}

template <int KIND>
static cudaError_t operand_probe_one(double millis, int sm_count, double* rate) {
    double* sink = nullptr;
    cudaError_t e = cudaMalloc(&sink, sizeof(double));
    if (e != cudaSuccess) return e;
    cudaEvent_t ev0, ev1;
    cudaEventCreate(&ev0);
    cudaEventCreate(&ev1);
    const int grid = sm_count * 8, threads = 256;
    int iters = 2000;
    float ms = 0.f;
    for (int attempt = 0; attempt < 8; ++attempt) {
        fp64_operand_probe_kernel<KIND><<<grid, threads>>>(iters / 4 + 1, 1.0, sink);  // warm-up
        cudaEventRecord(ev0);
        fp64_operand_probe_kernel<KIND><<<grid, threads>>>(iters, 1.0, sink);
        cudaEventRecord(ev1);
        e = cudaEventSynchronize(ev1);
        if (e != cudaSuccess) break;
        cudaEventElapsedTime(&ms, ev0, ev1);
        if (ms >= millis * 0.5 || iters > (1 << 28)) break;
        const double scale = (ms > 0.01f) ? (millis / ms) * 1.1 : 16.0;
        iters = (int)(iters * (scale > 16.0 ? 16.0 : scale)) + 1;
    }
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e == cudaSuccess) *rate = (double)grid * threads * 64.0 * (double)iters / (ms * 1e-3);
    cudaEventDestroy(ev0);
    cudaEventDestroy(ev1);
    cudaFree(sink);
    return e;
}

cudaError_t launch_operand_probe(double millis, int sm_count, double rates[4]) {
    cudaError_t e = operand_probe_one<0>(millis, sm_count, &rates[0]);
    if (e == cudaSuccess) e = operand_probe_one<1>(millis, sm_count, &rates[1]);
    if (e == cudaSuccess) e = operand_probe_one<2>(millis, sm_count, &rates[2]);
    if (e == cudaSuccess) e = operand_probe_one<3>(millis, sm_count, &rates[3]);
    return e;
}

template <typename T>
static cudaError_t probe_one(double millis, int sm_count, double* rate) {
    T* sink = nullptr;
    cudaError_t e = cudaMalloc(&sink, sizeof(T));
    if (e != cudaSuccess) return e;
    cudaEvent_t ev0, ev1;
    cudaEventCreate(&ev0);
    cudaEventCreate(&ev1);
    const int grid = sm_count * 8, threads = 256;
    int iters = 2000;
    float ms = 0.f;
    for (int attempt = 0; attempt < 8; ++attempt) {
        fma_probe_kernel<T><<<grid, threads>>>(iters / 4 + 1, (T)1, sink);  // warm-up
        cudaEventRecord(ev0);
        fma_probe_kernel<T><<<grid, threads>>>(iters, (T)1, sink);
        cudaEventRecord(ev1);
        e = cudaEventSynchronize(ev1);
        if (e != cudaSuccess) break;
        cudaEventElapsedTime(&ms, ev0, ev1);
        if (ms >= millis * 0.5 || iters > (1 << 28)) break;
        const double scale = (ms > 0.01f) ? (millis / ms) * 1.1 : 16.0;
        iters = (int)(iters * (scale > 16.0 ? 16.0 : scale)) + 1;
    }
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e == cudaSuccess) *rate = (double)grid * threads * 64.0 * (double)iters / (ms * 1e-3);
    cudaEventDestroy(ev0);
    cudaEventDestroy(ev1);
    cudaFree(sink);
    return e;
}

cudaError_t launch_probe(double millis, int sm_count, double* dfma_per_s, double* ffma_per_s) {
    cudaError_t e = cudaSuccess;
    if (dfma_per_s) e = probe_one<double>(millis, sm_count, dfma_per_s);
    if (e == cudaSuccess && ffma_per_s) e = probe_one<float>(millis, sm_count, ffma_per_s);
    return e;
}

}  // namespace dbie
