// dbie_grid.cu — GRID mode of the per-point lambda search (O-4).
//
// BASELINE.json config 5 asks for ">= 8 trial lambda per component per iteration"; that is NOT in
// the paper (which only names the Downhill Simplex method).  The reading: because
// B_p depends on lambda_p only, T trial values per component cost 3T kernel sums per
// stencil position but give (T+1)^3 candidate triples (the T trials plus the incumbent per
// component).  Per level: the interaction kernel (MODE_GRID, dbie_interact_fp64.cuh) evaluates
// the 4 x 3 x T sums of every active point; grid_step_kernel (one warp per point) forms B at the
// stencil, the forward differences of Eq. 13 once per (trial, component), Phi = f + w_g g
// (Eq. 8, 9, 14) of every candidate triple, takes the argmin (ties: lowest (t_x, t_y, t_z)), makes
// it the incumbent, applies the Eq. 12 exit and shrinks the window around it.
// Every decision is a comparison of separately rounded IEEE operations (mul_/add_/... of
// dbie_nm.cuh; this file is compiled with -fmad=false), in the oracle's order.
#include <cuda_runtime.h>
#include <math.h>

#include "dbie_internal.h"
#include "dbie_nm.cuh"
#include "dbie_solver_common.cuh"

namespace dbie {

constexpr int kGridWarps = 4;   // points per CTA of the step kernel

__global__ void grid_init_kernel(GridArrays s, long long M, long long ldo, const double* __restrict__ x,
                                 const double* __restrict__ y, const double* __restrict__ z, double* B,
                                 double* lam, double* resid, int* iters, int* status) {
    const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    bool keep = false;
    if (i < M) {
        const double xi = x[i], yi = y[i], zi = z[i];
        const bool invalid = !(zi > 0.0) || !isfinite(xi) || !isfinite(yi) || !isfinite(zi);
        if (invalid) {
            write_invalid(ldo, i, B, lam, resid, iters, status);
        } else {
            for (int c = 0; c < 3; ++c) {
                s.lo[c * s.cap + i] = 0.0;   // level 0 window: [0, lam_max/h]
                s.il[c * s.cap + i] = 0.0;
            }
            keep = true;
        }
    }
    warp_append(keep, (int)i, s.act[0], &s.nact[0]);
}

// trial t of a component whose window starts at lo (O-4): lo + W t/(T-1)
__device__ __forceinline__ double grid_trial(double lo, double W, int t, int T) {
    return add_(lo, div_(mul_(W, (double)t), (double)(T - 1)));
}

// level `lev` consumes list lev&1 and builds list (lev+1)&1; one warp per active point
__global__ void __launch_bounds__(kGridWarps * 32)
grid_step_kernel(GridArrays s, NMConsts k, GridConsts gc, int nchunks, int lev, long long ldo,
                 const double* __restrict__ z, const double* __restrict__ part, long long cap, double* B,
                 double* lam, double* resid, int* iters, int* status, unsigned long long* nevals) {
    extern __shared__ double sh[];
    const int T = gc.T, C1 = T + 1;
    const int cur = lev & 1;
    const unsigned n = s.nact[cur];
    if (blockIdx.x * kGridWarps >= n) return;   // whole block idle (uniform)
    if (blockIdx.x == 0 && threadIdx.x == 0 && nevals) atomicAdd(nevals, (unsigned long long)n * T);
    const int wib = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const unsigned j = blockIdx.x * kGridWarps + wib;   // slot of this warp
    if (j >= n) return;                                  // warp-uniform
    double* S = sh + (size_t)wib * C1 * 21;   // S[t*12 + s*3 + p]: B_p at stencil position s, trial t
    double* G = S + C1 * 12;                  // G[t*9 + p*3 + jj]: dB_p/dx_jj for trial t of component p
    const int id = s.act[cur][j];
    const double zi = z[id];
    const double c0 = mul_(zi, k.h2_over_2pi);
    const double c3 = mul_(add_(zi, k.delta_abs), k.h2_over_2pi);
    const long long Q = 12LL * T;

    const int C = (lev > 0) ? C1 : T;   // level 0 has no incumbent
    if (!k.analytic) {
        // A4: chunk sums in chunk order -> B at the stencil for every trial
        for (int q = lane; q < 12 * T; q += 32) {
            const int sp = q / T, t = q - sp * T;
            double sum = part[(long long)q * cap + j];
            for (int ch = 1; ch < nchunks; ++ch) sum = add_(sum, part[((long long)ch * Q + q) * cap + j]);
            S[t * 12 + sp] = mul_(sp >= 9 ? c3 : c0, sum);
        }
        if (lane < 12) S[T * 12 + lane] = (lev > 0) ? s.inc[lane * s.cap + id] : 0.0;   // the incumbent
        __syncwarp();
        // Eq. 13: forward differences, once per (candidate value, component)
        for (int e = lane; e < C * 9; e += 32) {
            const int t = e / 9, r9 = e - t * 9, p = r9 / 3, jj = r9 - p * 3;
            G[e] = div_(sub_(S[t * 12 + (jj + 1) * 3 + p], S[t * 12 + p]), k.delta_abs);
        }
    } else {
        // O-5: raw sums S[t*12 + kind*3 + p], kind = (K b, D dx b, D dy b, D b) -> B and the gradient
        for (int q = lane; q < 12 * T; q += 32) {
            const int sp = q / T, t = q - sp * T;
            double sum = part[(long long)q * cap + j];
            for (int ch = 1; ch < nchunks; ++ch) sum = add_(sum, part[((long long)ch * Q + q) * cap + j]);
            S[t * 12 + sp] = sum;
        }
        __syncwarp();
        const double zz = mul_(zi, zi);
        for (int e = lane; e < T * 9; e += 32) {
            const int t = e / 9, r9 = e - t * 9, p = r9 / 3, jj = r9 - p * 3;
            const double* St = S + t * 12;
            G[e] = (jj == 0)   ? -mul_(c0, St[3 + p])
                   : (jj == 1) ? -mul_(c0, St[6 + p])
                               : mul_(k.h2_over_2pi, add_(St[p], mul_(zz, St[9 + p])));
        }
        __syncwarp();
        for (int e = lane; e < T * 3; e += 32) {
            const int t = e / 3, p = e - t * 3;
            S[t * 12 + p] = mul_(c0, S[t * 12 + p]);   // B_p (after d/dz has used the raw sum)
        }
        if (lev > 0 && lane < 12) {   // the incumbent: inc[0..2] = B, inc[3 + p*3 + jj] = dB_p/dx_jj
            const double v = s.inc[lane * s.cap + id];
            if (lane < 3) S[T * 12 + lane] = v;
            else G[T * 9 + lane - 3] = v;
        }
    }
    __syncwarp();

    // Phi of every candidate triple; strict '<' in index order keeps the lexicographically first
    double best = INFINITY;
    int bidx = 0x7fffffff;
    const int ncand = C * C * C;
    for (int idx = lane; idx < ncand; idx += 32) {
        const int tx = idx / (C * C), ty = (idx / C) % C, tz = idx % C;
        const int tt[3] = {tx, ty, tz};
        double Gm[3][3], B0[3];
        for (int p = 0; p < 3; ++p) {
            B0[p] = S[tt[p] * 12 + p];
            for (int jj = 0; jj < 3; ++jj) Gm[p][jj] = G[tt[p] * 9 + p * 3 + jj];
        }
        const double ph = as_inf_(residual_from_gradient(Gm, B0, k).phi);
        if (ph < best) {
            best = ph;
            bidx = idx;
        }
    }
    for (int off = 16; off > 0; off >>= 1) {
        const double ob = __shfl_xor_sync(0xffffffffu, best, off);
        const int oi = __shfl_xor_sync(0xffffffffu, bidx, off);
        if (ob < best || (ob == best && oi < bidx)) {
            best = ob;
            bidx = oi;
        }
    }
    if (!(best < INFINITY)) {   // no finite candidate: |B| = 0 or non-finite sums
        if (lane == 0) write_invalid(ldo, id, B, lam, resid, iters, status);
        return;
    }
    const int bt[3] = {bidx / (C * C), (bidx / C) % C, bidx % C};
    double Gm[3][3], B0[3], il[3];
    for (int p = 0; p < 3; ++p) {
        B0[p] = S[bt[p] * 12 + p];
        for (int jj = 0; jj < 3; ++jj) Gm[p][jj] = G[bt[p] * 9 + p * 3 + jj];
        il[p] = (bt[p] < T) ? grid_trial(s.lo[p * s.cap + id], gc.W, bt[p], T) : s.il[p * s.cap + id];
    }
    const Residual r = residual_from_gradient(Gm, B0, k);
    int st = -1;
    if (k.use_eq12 && r.f <= k.eps_f && r.g <= k.eps_g) st = 0;       // Eq. 12
    else if (lev + 1 >= gc.n_level) st = 1;                           // all levels done
    if (st >= 0) {
        if (lane == 0) {
            for (int p = 0; p < 3; ++p) {
                B[p * ldo + id] = r.B[p];
                lam[p * ldo + id] = fabs(il[p]);
            }
            resid[id] = r.f;
            resid[ldo + id] = r.g;
            iters[id] = lev + 1;
            status[id] = st;
        }
        return;
    }
    // the argmin becomes the incumbent; next window centred on it, clipped to [0, lam_max/h]
    if (lane < 12) {
        if (!k.analytic) s.inc[lane * s.cap + id] = S[bt[lane % 3] * 12 + lane];
        else if (lane < 3) s.inc[lane * s.cap + id] = S[bt[lane] * 12 + lane];
        else s.inc[lane * s.cap + id] = G[bt[(lane - 3) / 3] * 9 + lane - 3];
    }
    if (lane == 0) {
        for (int p = 0; p < 3; ++p) {
            double l = sub_(il[p], mul_(0.5, gc.Wn));
            if (l < 0.0) l = 0.0;
            if (add_(l, gc.Wn) > gc.Lmax) l = sub_(gc.Lmax, gc.Wn);
            s.lo[p * s.cap + id] = l;
            s.il[p * s.cap + id] = il[p];
        }
        const unsigned pos = atomicAdd(&s.nact[cur ^ 1], 1u);
        s.act[cur ^ 1][pos] = id;
    }
}

cudaError_t launch_grid_init(const GridArrays& s, long long M, long long ldo, const double* x, const double* y,
                             const double* z, double* B, double* lam, double* resid, int* iters, int* status,
                             cudaStream_t st) {
    if (M <= 0) return cudaSuccess;
    const unsigned grid = (unsigned)((M + 127) / 128);
    grid_init_kernel<<<grid, 128, 0, st>>>(s, M, ldo, x, y, z, B, lam, resid, iters, status);
    return cudaGetLastError();
}

cudaError_t launch_grid_step(const GridArrays& s, const NMConsts& k, const GridConsts& gc, const BoundaryView& bd,
                             int lev, long long M, long long ldo, const double* z, const double* part,
                             long long cap, double* B, double* lam, double* resid, int* iters, int* status,
                             unsigned long long* nevals, cudaStream_t st) {
    if (M <= 0) return cudaSuccess;
    const unsigned grid = (unsigned)((M + kGridWarps - 1) / kGridWarps);   // blocks past the device-side count exit
    const size_t smem = (size_t)kGridWarps * (gc.T + 1) * 21 * sizeof(double);
    grid_step_kernel<<<grid, kGridWarps * 32, smem, st>>>(s, k, gc, bd.nchunks, lev, ldo, z, part, cap, B, lam,
                                                          resid, iters, status, nevals);
    return cudaGetLastError();
}

}  // namespace dbie
