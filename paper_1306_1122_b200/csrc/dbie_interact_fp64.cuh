// dbie_interact_fp64.cuh — the fp64 M x N point-pixel interaction kernel.
//
//   S_p(i) = sum_k [theta sin theta + cos theta]/r^3 * B_p0[k],  theta = |lambda_p| r
//   (Eq. 6, Eq. 16; the prefactor z h^2/2pi is applied by the
//   consumer of the chunk sums).
//
// Mapping (the inverse of the paper's, which strides the PIXELS of one point
// over 80x128 threads): evaluation positions are the parallel dimension.  A thread owns one field
// point (eval, analytic gradient), all 4 stencil positions of a field point (Eq. 13: MODE_STENCIL4),
// or one stencil position with NT equally spaced trial lambda triples (GRID).  The boundary is
// streamed through shared memory in 16 KB tiles by the TMA bulk-copy engine (cp.async.bulk +
// mbarrier, double buffered) and every thread of the CTA reads the same pixel record as a broadcast
// LDS.128 pair; UNR pixels are in flight per thread.  sin/cos come from a 256-entry angle table that every CTA
// keeps in shared memory (8 interleaved copies, dbie_math.cuh) plus short polynomials.  The bound is the FP64
// pipe; the stencil launch went 14.17 -> 11.11 -> 9.04 -> 8.39 ms over round 1 (its captures and the shape sweep
// behind the THREADS x MINB x UNR choices are in git history, profiles/r01_*), round 2's table kernel is in
// profiles/r02_ncu_full_interact64_eval_cfg4.md.
//
// The body of one work item (a block of evaluation positions x a range of canonical chunks) is the
// device function interact_item; what happens to a finished chunk sum is the caller's `sink`:
// interact64_kernel writes it to the partial-sum scratch (PartSink), the fused Nelder-Mead kernel
// (dbie_solve_fused.cu) keeps it in registers or hands it to the CTA that finishes the point block last.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "dbie_internal.h"
#include "dbie_math.cuh"
#include "dbie_tma.cuh"

namespace dbie {

// MODE_ANALYTIC (O-5): one position per field point; besides the Eq. 6 sum
// it accumulates the three sums of the analytic gradient (kinds 1..3 below), 12 sums per slot like
// the stencil, from the same sincos: d/dr[n(lambda r)/r^3] = lambda^2 cos(lambda r)/r^2 - 3 n/r^4.
// MODE_GRID_ANALYTIC: the same four sums for NT trial triples of GRID mode (item = slot * G + g).
// MODE_STENCIL4: the Eq. 13 stencil with all 4 positions of a field point in ONE thread (item = slot).
// The positions are delta = 1e-3 h apart, so theta_s = lambda r_s differs from theta_0 by eps <= lambda delta:
// one full sincos per component at r_i and, for the other three positions, n(theta_0 + eps) from (sin, cos)(theta_0)
// (kernel_n_near); geometry (dx, dy, z terms) is shared where the offsets allow.  52.25 FP64 instructions per
// interaction instead of 61.  Threads whose lambda delta exceeds kNearEpsMax take the plain path (60.5).
// MODE_EVAL_R: MODE_EVAL with the reduced-degree sincos of reading A-12 (DBIE_EVAL_REDUCED_SINCOS): 55 instructions.
enum { MODE_EVAL = 0, MODE_GRID = 2, MODE_ANALYTIC = 3, MODE_GRID_ANALYTIC = 4, MODE_STENCIL4 = 5, MODE_EVAL_R = 6 };

// items (threads' units of work) per slot
__host__ __device__ inline long long items_per_slot(int mode, int G) {
    if (mode == MODE_EVAL || mode == MODE_EVAL_R || mode == MODE_ANALYTIC || mode == MODE_STENCIL4) return 1;
    if (mode == MODE_GRID_ANALYTIC) return G;
    return (long long)kStencil * G;   // MODE_GRID: one item per stencil position and group of NT trials
}

// One pixel of MODE_STENCIL4: the 4 stencil positions (x_i, x_i + delta | y, y + delta | z, z + delta share
// dx / dy^2 + z^2 terms where they can).  FAST: one sincos per component at r_i, kernel_n_near for the rest.
// The pixel's 12 terms are returned as factor pairs: the accumulation is acc[q][c] = fma(nv[q][c], wb[q][c], acc[q][c]),
// in pixel order, whoever performs it (the owning thread, or a chain lane of the warp-per-point path).
template <bool FAST>
__device__ __forceinline__ void stencil4_terms(const TrigRef& tr, const double4 px, double xi, double xi1, double cc,
                                               double cc2, double cc3, const double (&lam)[3], double (&nv)[4][3],
                                               double (&wb)[4][3]) {
    const double dx0 = px.x - xi, dx1 = px.x - xi1;
    const double r2s[4] = {fma(dx0, dx0, cc), fma(dx1, dx1, cc), fma(dx0, dx0, cc2), fma(dx0, dx0, cc3)};
    double rs[4], ws[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const double y = rsqrt_full(r2s[q]);
        rs[q] = r2s[q] * y;
        ws[q] = (y * y) * y;
    }
    const double b0[3] = {px.y, px.z, px.w};
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        if (FAST) {
            const double th0 = lam[c] * rs[0];
            double s0, c0;
            sincos_pos(th0, tr, s0, c0);
            nv[0][c] = fma(th0, s0, c0);
            wb[0][c] = ws[0] * b0[c];
#pragma unroll
            for (int q = 1; q < 4; ++q) {
                const double thq = lam[c] * rs[q];
                nv[q][c] = kernel_n_near(thq, s0, c0, thq - th0);
                wb[q][c] = ws[q] * b0[c];
            }
        } else {
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                nv[q][c] = kernel_n(lam[c] * rs[q], tr);
                wb[q][c] = ws[q] * b0[c];
            }
        }
    }
}

template <bool FAST>
__device__ __forceinline__ void stencil4_pixel(const TrigRef& tr, const double4 px, double xi, double xi1, double cc,
                                               double cc2, double cc3, const double (&lam)[3], double (&acc)[4][3]) {
    double nv[4][3], wb[4][3];
    stencil4_terms<FAST>(tr, px, xi, xi1, cc, cc2, cc3, lam, nv, wb);
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int q = 0; q < 4; ++q) acc[q][c] = fma(nv[q][c], wb[q][c], acc[q][c]);
}

// One pixel of MODE_ANALYTIC (one lambda triple) as factor pairs, kind = 0: sum K b, 1: sum D dx b, 2: sum D dy b,
// 3: sum D b; the accumulation is acc[kind][c] = fma(fa[kind][c], fb[kind][c], acc[kind][c]) (kind 3 has fb = 1, which
// rounds exactly like acc + fa).  The same expressions as the thread-per-point loop of interact_item below.
__device__ __forceinline__ void analytic_terms(const TrigRef& tr, const double4 px, double xi, double dy, double cc,
                                               const double (&lam)[3], const double (&lam2)[3], double (&fa)[4][3],
                                               double (&fb)[4][3]) {
    const double dx = px.x - xi;
    const double r2 = fma(dx, dx, cc);
    const double y = rsqrt_full(r2);
    const double rr = r2 * y;
    const double wgt = (y * y) * y;
    const double wb[3] = {wgt * px.y, wgt * px.z, wgt * px.w};
    const double m3y2 = (y * y) * -3.0;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        double n, cs;
        kernel_n_cos(lam[c] * rr, tr, n, cs);
        const double e = fma(lam2[c], cs, n * m3y2);
        const double gb = e * wb[c];
        fa[0][c] = n;  fb[0][c] = wb[c];
        fa[1][c] = gb; fb[1][c] = dx;
        fa[2][c] = gb; fb[2][c] = dy;
        fa[3][c] = gb; fb[3][c] = 1.0;
    }
}

struct ItemCtx {      // what a sink needs to know about the calling thread's work item
    bool live;        // the thread owns a real item (not padding of the last block)
    long long slot;   // its slot
    int s, g;         // MODE_GRID: stencil position and trial group; MODE_GRID_ANALYTIC: trial group
};

// The sink of interact64_kernel: chunk sums go to the scratch, part[(c*Q + q)*cap + slot] (A4).
template <int MODE, int NT>
struct PartSink {
    const InteractParams& p;
    int nsplit, nch;
    double run[3];   // MODE_EVAL, unsplit launch: running sum of the chunk sums
    template <int NA>
    __device__ __forceinline__ void operator()(const ItemCtx& ic, int c, const double (&acc)[NA][3]) {
        if (!ic.live) return;
        const long long slot = ic.slot;
        if (MODE == MODE_EVAL || MODE == MODE_EVAL_R) {
            if (nsplit == 1) {
                // this CTA sees every chunk: add them here, in chunk order with the epilogue's own
                // operation (bit-identical), and write one sum instead of nchunks partial sums
#pragma unroll
                for (int q = 0; q < 3; ++q) run[q] = (c == 0) ? acc[0][q] : __dadd_rn(run[q], acc[0][q]);
                if (c == nch - 1) {
#pragma unroll
                    for (int q = 0; q < 3; ++q) p.part[(long long)q * p.cap + slot] = run[q];
                }
            } else {
#pragma unroll
                for (int q = 0; q < 3; ++q) p.part[((long long)c * 3 + q) * p.cap + slot] = acc[0][q];
            }
        } else if (MODE == MODE_ANALYTIC || MODE == MODE_STENCIL4) {   // rows = kinds / stencil positions
#pragma unroll
            for (int kd = 0; kd < 4; ++kd)
#pragma unroll
                for (int q = 0; q < 3; ++q) p.part[((long long)c * 12 + kd * 3 + q) * p.cap + slot] = acc[kd][q];
        } else if (MODE == MODE_GRID_ANALYTIC) {
            const long long Q = 12LL * p.T;
#pragma unroll
            for (int tt = 0; tt < NT; ++tt)
#pragma unroll
                for (int kd = 0; kd < 4; ++kd)
#pragma unroll
                    for (int q = 0; q < 3; ++q)
                        p.part[(c * Q + (long long)(kd * 3 + q) * p.T + ic.g * NT + tt) * p.cap + slot] =
                            acc[4 * tt + kd][q];
        } else {
            const long long Q = 12LL * p.T;
#pragma unroll
            for (int tt = 0; tt < NT; ++tt)
#pragma unroll
                for (int q = 0; q < 3; ++q)
                    p.part[(c * Q + (long long)(ic.s * 3 + q) * p.T + ic.g * NT + tt) * p.cap + slot] = acc[tt][q];
        }
    }
};

// One work item: the evaluation positions of block `blk` (THREADS items) against the canonical chunks
// [c0, c1).  `it` counts the tiles this CTA has consumed (stage = it & 1, mbarrier parity = (it >> 1) & 1).
// At the end of every chunk the chunk sums go to sink(ctx, c, acc) and the accumulators restart from zero.
// Every tile ends with a __syncthreads, so the caller may reuse its shared scalars after the call.
template <int MODE, int NT, int THREADS, int UNR, class Sink>
__device__ __forceinline__ void interact_item(const InteractParams& p, const TrigRef& tr, double4 (*tile)[kTilePx],
                                              uint64_t* full, unsigned& it, long long nitems, int G, long long blk,
                                              int c0, int c1, Sink& sink) {
    constexpr bool kGridLam = (MODE == MODE_GRID || MODE == MODE_GRID_ANALYTIC);   // lambda from the GRID window
    constexpr bool kAnalytic = (MODE == MODE_ANALYTIC || MODE == MODE_GRID_ANALYTIC);
    static_assert(kGridLam || NT == 1, "only GRID modes carry several lambda triples per thread");
    const int tid = threadIdx.x;
    const BoundaryView& bd = p.bd;

    // ---- this thread's evaluation position and lambda triples
    const long long item = blk * THREADS + tid;
    ItemCtx ic;
    ic.live = item < nitems;
    const long long jt = ic.live ? item : nitems - 1;
    int s = 0, g = 0;
    long long slot;
    if (MODE == MODE_EVAL || MODE == MODE_EVAL_R || MODE == MODE_ANALYTIC || MODE == MODE_STENCIL4) {
        slot = jt;
    } else if (MODE == MODE_GRID_ANALYTIC) {
        g = (int)(jt % G);
        slot = jt / G;
    } else {
        g = (int)(jt % G);
        const long long js = jt / G;
        s = (int)(js & 3);
        slot = js >> 2;
    }
    ic.slot = slot;
    ic.s = s;
    ic.g = g;
    // the active list and the trial lambda may have been written earlier in the SAME launch by another SM
    // (fused solver): read them through L2
    constexpr bool kEval = (MODE == MODE_EVAL || MODE == MODE_EVAL_R);
    const long long id = kEval ? p.slot0 + slot : (p.act ? (long long)__ldcg(p.act + slot) : slot);
    double xi = p.x[id], yi = p.y[id], zi = p.z[id];
    if (MODE == MODE_GRID) {   // Eq. 13: r_i, r_i + delta x, + delta y, + delta z
        if (s == 1) xi = __dadd_rn(xi, p.delta_abs);
        if (s == 2) yi = __dadd_rn(yi, p.delta_abs);
        if (s == 3) zi = __dadd_rn(zi, p.delta_abs);
    }
    const double z2 = zi * zi;
    // MODE_STENCIL4: the offset coordinates of positions 1 (x), 2 (y), 3 (z)
    const double xi1 = __dadd_rn(xi, p.delta_abs), yi2 = __dadd_rn(yi, p.delta_abs);
    const double zi3 = __dadd_rn(zi, p.delta_abs), z23 = zi3 * zi3;
    double lam[NT][3];
    if (kGridLam) {
        // trial t of component c: lo_c + W t/(T-1), each operation rounded separately (O-4)
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const double lo = p.lo[c * p.ldlo + id];
#pragma unroll
            for (int tt = 0; tt < NT; ++tt) {
                const int t = g * NT + tt;
                lam[tt][c] = fabs(__dadd_rn(lo, __ddiv_rn(__dmul_rn(p.W, (double)t), (double)(p.T - 1))));
            }
        }
    } else {
#pragma unroll
        for (int c = 0; c < 3; ++c) lam[0][c] = fabs(__ldcg(p.lam + c * p.ldlam + id));
    }

    // accumulators: one row per lambda triple; MODE_ANALYTIC: rows = sum K b, sum D dx b, sum D dy b, sum D b
    // (row 4 tt + kind in the analytic modes)
    constexpr int NA = (kAnalytic || MODE == MODE_STENCIL4) ? 4 * NT : NT;
    double acc[NA][3];
#pragma unroll
    for (int tt = 0; tt < NA; ++tt) acc[tt][0] = acc[tt][1] = acc[tt][2] = 0.0;
    const bool lam_all_zero = (lam[0][0] == 0.0) && (lam[0][1] == 0.0) && (lam[0][2] == 0.0);   // MODE_EVAL
    const bool small_eps = fmax(fmax(lam[0][0], lam[0][1]), lam[0][2]) * p.delta_abs <= kNearEpsMax;
    double lam2[NT][3];   // analytic modes: lambda^2
#pragma unroll
    for (int tt = 0; tt < NT; ++tt)
#pragma unroll
        for (int c = 0; c < 3; ++c) lam2[tt][c] = lam[tt][c] * lam[tt][c];

    // the item's canonical chunks [c0, c1) = units [u0, u1); the tiles that hold them (the first and the last tile may
    // also hold rows of neighbouring chunks, which are skipped)
    const int u0 = chunk_first_unit(bd, c0), u1 = chunk_first_unit(bd, c1);
    const int t0 = unit_tile(bd, u0), t1 = unit_tile(bd, u1 - 1) + 1;
    int c = c0;
    int u_chunk_end = chunk_first_unit(bd, c + 1);
    if (tid == 0) {
        const TileDesc d = tile_desc(bd, t0);
        mbar_expect_tx(&full[it & 1], (unsigned)d.npx * 32u);
        bulk_g2s(&tile[it & 1][0], bd.rec + d.px0, (unsigned)d.npx * 32u, &full[it & 1]);
    }
    for (int t = t0; t < t1; ++t, ++it) {
        if (tid == 0 && t + 1 < t1) {  // prefetch the next tile into the other stage
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
            const double cc2 = fma(dy2, dy2, z2), cc3 = fma(dy, dy, z23);   // MODE_STENCIL4
            bool row_done = false;
            if constexpr (MODE == MODE_STENCIL4) {
                // the small-angle / plain decision is per thread: two loops instead of a branch per pixel
                if (small_eps) {
#pragma unroll UNR
                    for (int j = 0; j < d.ncols; ++j) stencil4_pixel<true>(tr, rp[j], xi, xi1, cc, cc2, cc3, lam[0], acc);
                } else {
#pragma unroll UNR
                    for (int j = 0; j < d.ncols; ++j) stencil4_pixel<false>(tr, rp[j], xi, xi1, cc, cc2, cc3, lam[0], acc);
                }
                row_done = true;
            }
            if constexpr (kEval) {
                // lambda = 0 in all three components (the potential field, BASELINE config 1): n(0) = 1
                // exactly, so the term is w B_p0 and the sum is bit-identical to the general loop's
                // fma(1, w B, acc) at 15 instead of 61 FP64 instructions.  Per-thread decision.
                if (lam_all_zero) {
#pragma unroll 4
                    for (int j = 0; j < d.ncols; ++j) {
                        const double4 px = rp[j];
                        const double dx = px.x - xi;
                        const double r2 = fma(dx, dx, cc);
                        const double y = rsqrt_full(r2);
                        const double wgt = (y * y) * y;
                        acc[0][0] = __dadd_rn(acc[0][0], __dmul_rn(wgt, px.y));   // no contraction: same
                        acc[0][1] = __dadd_rn(acc[0][1], __dmul_rn(wgt, px.z));   // roundings as fma(1, w B, acc)
                        acc[0][2] = __dadd_rn(acc[0][2], __dmul_rn(wgt, px.w));
                    }
                    row_done = true;
                }
            }
            if (!row_done) {
#pragma unroll UNR
            for (int j = 0; j < d.ncols; ++j) {
                const double4 px = rp[j];  // {x_k, Bx0, By0, Bz0}: two broadcast LDS.128
                const double dx = px.x - xi;
                const double r2 = fma(dx, dx, cc);
                const double y = rsqrt_full(r2);   // 1/r
                const double rr = r2 * y;          // r
                const double wgt = (y * y) * y;    // 1/r^3
                const double wx = wgt * px.y, wy = wgt * px.z, wz = wgt * px.w;
                if (kAnalytic) {
                    // K b = n w b;  D b = (lambda^2 cos(theta) - 3 n / r^2) w b  (w = 1/r^3)
                    const double m3y2 = (y * y) * -3.0;
                    const double wb[3] = {wx, wy, wz};
#pragma unroll
                    for (int tt = 0; tt < NT; ++tt)
#pragma unroll
                        for (int c = 0; c < 3; ++c) {
                            double n, cs;
                            kernel_n_cos(lam[tt][c] * rr, tr, n, cs);
                            const double e = fma(lam2[tt][c], cs, n * m3y2);
                            const double gb = e * wb[c];
                            acc[4 * tt + 0][c] = fma(n, wb[c], acc[4 * tt + 0][c]);
                            acc[4 * tt + 1][c] = fma(gb, dx, acc[4 * tt + 1][c]);
                            acc[4 * tt + 2][c] = fma(gb, dy, acc[4 * tt + 2][c]);
                            acc[4 * tt + 3][c] += gb;
                        }
                    continue;
                }
                if (MODE == MODE_GRID && NT > 1) {
                    // The NT trial values of a component are equally spaced (lambda_t = lo + W t/(T-1)), so theta
                    // advances by the same d_theta = W/(T-1) r for all three components.  With (s_j, c_j) =
                    // (sin, cos)(j d_theta), j = 1..NT/2, formed ONCE per pixel (one full sincos, then angle doubling /
                    // addition), and one full sincos per component at the middle trial,
                    //   n(theta_m + j d) = s_m (theta c_j - s_j) + c_m (theta s_j + c_j),   theta = fl(lambda_t r):
                    // 5 FP64 instructions per further trial and component instead of a 16-instruction kernel_n, every
                    // trial independent of the others (no chained rotation).  theta_m + j d_theta differs from
                    // fl(lambda_t r) by a few ulp(theta), the size of the rounding theta carries anyway.
                    // Needs lo >= 0 (no |.| fold inside the group): true for T >= 3 (dbie_solve rejects T < 4).
                    constexpr int TB = NT / 2;   // the full sincos is taken at the middle trial
                    double sj[TB + 1], cj[TB + 1];
                    sincos_pos(p.dlam * rr, tr, sj[1], cj[1]);
#pragma unroll
                    for (int j = 2; j <= TB; ++j) {
                        if (j % 2 == 0) {   // doubling: sin 2a = 2 sin a cos a, cos 2a = 1 - 2 sin^2 a
                            const double d2 = sj[j / 2] + sj[j / 2];
                            sj[j] = d2 * cj[j / 2];
                            cj[j] = fma(-d2, sj[j / 2], 1.0);
                        } else {            // addition of one step
                            sj[j] = fma(sj[j - 1], cj[1], cj[j - 1] * sj[1]);
                            cj[j] = fma(cj[j - 1], cj[1], -(sj[j - 1] * sj[1]));
                        }
                    }
                    const double wb[3] = {wx, wy, wz};
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        const double thb = lam[TB][c] * rr;
                        double sb, cb;
                        sincos_pos(thb, tr, sb, cb);
                        acc[TB][c] = fma(fma(thb, sb, cb), wb[c], acc[TB][c]);
                        // the weight w B_p0 is folded into (sin, cos)(theta_m) once per component, so a further
                        // trial costs theta, P, Q and two accumulating FMAs: 5 instructions
                        const double sbw = sb * wb[c], cbw = cb * wb[c];
#pragma unroll
                        for (int tt = 0; tt < NT; ++tt) {
                            if (tt == TB) continue;
                            const int j = tt > TB ? tt - TB : TB - tt;
                            const double th = lam[tt][c] * rr;
                            // sin(+-j d) = +-s_j: the sign is an operand modifier
                            const double pp = tt > TB ? fma(th, cj[j], -sj[j]) : fma(th, cj[j], sj[j]);
                            const double qq = tt > TB ? fma(th, sj[j], cj[j]) : fma(th, -sj[j], cj[j]);
                            acc[tt][c] = fma(sbw, pp, fma(cbw, qq, acc[tt][c]));
                        }
                    }
                    continue;
                }
#pragma unroll
                for (int tt = 0; tt < NT; ++tt) {
                    acc[tt][0] = fma(kernel_n<MODE == MODE_EVAL_R>(lam[tt][0] * rr, tr), wx, acc[tt][0]);
                    acc[tt][1] = fma(kernel_n<MODE == MODE_EVAL_R>(lam[tt][1] * rr, tr), wy, acc[tt][1]);
                    acc[tt][2] = fma(kernel_n<MODE == MODE_EVAL_R>(lam[tt][2] * rr, tr), wz, acc[tt][2]);
                }
            }
            }
            if (unit + 1 == u_chunk_end) {  // A4: one partial sum per chunk, added in chunk order later
                sink(ic, c, acc);
#pragma unroll
                for (int tt = 0; tt < NA; ++tt) acc[tt][0] = acc[tt][1] = acc[tt][2] = 0.0;
                ++c;
                u_chunk_end = chunk_first_unit(bd, c + 1);
            }
        }
        __syncthreads();  // everyone is done with stage it&1 before it is refilled
    }
}

// shared memory of interact64_kernel
constexpr size_t kInteractSmem = kTrigTableBytes + sizeof(double4) * 2 * kTilePx + 64;

// Every CTA copies the 4 KB angle table from global memory (L2-resident) into 8 interleaved copies at the start of
// its dynamic shared memory; the caller's __syncthreads publishes it.  Returns the calling lane's copy.
__device__ __forceinline__ TrigRef trig_fill(unsigned char* smem, int tid, int nthreads) {
    TrigEntry* tab = reinterpret_cast<TrigEntry*>(smem);
    for (int i = tid; i < kTrigEntries * kTrigCopies; i += nthreads) tab[i] = kTrigTabG[i / kTrigCopies];
    return TrigRef{tab, (unsigned)(tid & (kTrigCopies - 1)) * (unsigned)sizeof(TrigEntry)};
}

// split of the chunk range of a launch with `nblk` position blocks (shared by the kernels and their launchers)
__host__ __device__ inline int chunk_split(long long nblk, int target_items, int nchunks) {
    int nsplit = 1;
    if (nblk < target_items) {
        nsplit = (int)((target_items + nblk - 1) / nblk);
        if (nsplit > nchunks) nsplit = nchunks;
    }
    return nsplit;
}

template <int MODE, int NT, int THREADS, int MINB, int UNR>
__global__ void __launch_bounds__(THREADS, MINB) interact64_kernel(const __grid_constant__ InteractParams p) {
    constexpr bool kGridLam = (MODE == MODE_GRID || MODE == MODE_GRID_ANALYTIC);
    // dynamic shared memory: [trig table, 8 copies, 32 KB][2 boundary tiles, 32 KB][mbarriers, work-item slot]
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double4(*tile)[kTilePx] = reinterpret_cast<double4(*)[kTilePx]>(smem_raw + kTrigTableBytes);
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + kTrigTableBytes + sizeof(double4) * 2 * kTilePx);
    long long& next_item = *reinterpret_cast<long long*>(full + 2);

    const int tid = threadIdx.x;
    if (tid == 0) {
        mbar_init(&full[0], 1);
        mbar_init(&full[1], 1);
        mbar_fence_init();
    }
    const TrigRef tr = trig_fill(smem_raw, tid, THREADS);
    __syncthreads();

    if (blockIdx.x == 0 && tid == 0) {
        if (p.zero_ptr) *p.zero_ptr = 0u;    // next pass's list counter
        if (p.zero_work) *p.zero_work = 0u;  // next pass's work counter
    }
    const long long count = p.count_ptr ? (long long)(*p.count_ptr) : p.count;   // slots
    const int G = kGridLam ? p.T / NT : 1;
    const long long nitems = count * items_per_slot(MODE, G);
    const long long nblk = (nitems + THREADS - 1) / THREADS;
    if (nblk == 0) return;
    const int NCH = p.bd.nchunks;
    const int nsplit = chunk_split(nblk, p.target_items, NCH);
    const long long nwork = nblk * nsplit;

    unsigned it = 0;  // tiles consumed by this CTA so far
    // Work items: one per CTA when the host knows the count (the hardware scheduler balances them);
    // a persistent grid (count on the device) takes them from an atomic counter in index order,
    // which balances the same way (static striding measured 1-15 % slower in round 1's shape sweep).
    for (long long w = blockIdx.x;; w += gridDim.x) {
        if (p.work_ctr) {
            if (tid == 0) next_item = (long long)atomicAdd(p.work_ctr, 1u);
            __syncthreads();
            w = next_item;   // every item ends with a __syncthreads, so the slot is free to rewrite
        }
        if (w >= nwork) break;
        const long long blk = w / nsplit;
        const int sp = (int)(w % nsplit);
        const int c0 = (int)(((long long)sp * NCH) / nsplit);
        const int c1 = (int)(((long long)(sp + 1) * NCH) / nsplit);
        PartSink<MODE, NT> sink{p, nsplit, NCH, {0.0, 0.0, 0.0}};
        interact_item<MODE, NT, THREADS, UNR>(p, tr, tile, full, it, nitems, G, blk, c0, c1, sink);
    }
}

}  // namespace dbie
