/* dbie.h — C ABI of libdbie_b200.so: the data-parallel hot path of the Direct Boundary
 * Integral Equation (DBIE) method for nonlinear force-free coronal fields
 * (Wang, Yan & Tan, arXiv 1306.1122; citations are PAPER.md:<line>).
 *
 * What the library computes
 * -------------------------
 *  Eq. 6 discretised as the nodal sum Eq. 16, for every
 *  evaluation point i and Cartesian component p in {x,y,z}:
 *
 *      B_p(i) = (z_i h^2 / 2 pi) * sum_{k<N} [theta sin(theta) + cos(theta)] / r_ik^3 * B_p0[k],
 *      r_ik   = sqrt((x_k-x_i)^2 + (y_k-y_i)^2 + z_i^2),  theta = |lambda_p(i)| r_ik,
 *      (x_k, y_k) = (x0 + (ix+1/2) h, y0 + (iy+1/2) h),   k = iy*nx + ix,
 *
 *  and, in dbie_solve, the per-point search of the pseudo-force-free factors
 *  (lambda_x, lambda_y, lambda_z) by the Downhill Simplex method
 *  that minimises f_i (Eq. 8) and g_i (Eq. 9), with the frozen-lambda
 *  first-order finite differences of Eq. 13 and J = curl B (Eq. 14,
 *  PAPER.md:108-110).  The readings taken where the paper is silent (pixel centres, the scalar
 *  objective, thresholds, the initial simplex, the GRID mode) are listed in DESIGN.md section 3.
 *
 * Conventions
 * -----------
 *  - Every array pointer is a CUDA DEVICE pointer unless the function name ends in _host,
 *    in which case every array pointer is a HOST pointer (pageable or pinned).
 *  - Arrays are structure-of-arrays, fp64 unless stated: a "3*M" array holds component p of
 *    point i at [p*M + i].
 *  - Lengths (x, y, z, h, 1/lambda) share one unit; B is in the units of the boundary data.
 *  - Ownership: the context copies the boundary in dbie_create (the caller may free its arrays
 *    when the call returns).  Inputs/outputs of eval/solve are caller-allocated and
 *    caller-owned.  Scratch memory is owned by the context and grown lazily, so ONE context
 *    must not be used from two streams or two host threads at the same time.
 *  - Device-pointer entry points are asynchronous on the given stream (they only enqueue work;
 *    growing the scratch may synchronise the device once).  _host entry points return after
 *    the results are in the host arrays.
 *  - Errors: no exceptions, no aborts, no printing.  Every entry point returns a dbie_status;
 *    argument errors are detected before any launch.  Per-point problems (z_i <= 0 or a
 *    non-finite coordinate/lambda) do not fail the call: that point's outputs are NaN (and
 *    status 3 in dbie_solve).
 *  - There is no CPU fallback: without a CUDA device every compute entry point returns
 *    DBIE_ECUDA.
 *  - Devices: a context belongs to the CUDA device that was current in dbie_create.  Every later
 *    entry point makes that device current for the duration of the call and restores the caller's
 *    device before returning; the arrays and the stream passed in must belong to the context's device.
 *    The Nelder-Mead dbie_solve (and a lambda-solving dbie_trace) runs as ONE cooperative launch: the device must
 *    support cooperative launches (else DBIE_ESTATE; the GRID method does not need them), and the grid must be
 *    co-resident.  Where the context may use only part of the SMs (MPS active-thread percentage, green contexts) the
 *    launch is retried with smaller grids; results do not depend on the grid.
 *  - Range of lambda: theta = |lambda| r must stay below 2^20 (about 1e6 rad) for every point-pixel
 *    pair; the one-step argument reduction of the kernel is exact up to theta * 4e-17 there (relative
 *    to theta: the same size as the rounding of theta itself).  Beyond that the result is unspecified
 *    (finite, wrong).  The paper's lambda are ~0.1 / pixel on windows of <= 1500 pixels: theta < 200.
 *  - Const-ness: eval / residual / solve take a NON-const context although they do not change the
 *    boundary: they grow and use the context's scratch memory and record counters (SURVEY 8(b)
 *    wrote `const dbie_ctx*`; the deviation is deliberate and is why one context serves one stream
 *    at a time).
 *  - dbie_last_cuda_error(NULL) reads a process-global buffer (the last failure that had no
 *    context, i.e. inside dbie_create): it is not synchronised between threads.
 */
#ifndef DBIE_H
#define DBIE_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dbie_ctx dbie_ctx; /* opaque; owns its device copy of the boundary */

typedef enum {
    DBIE_OK = 0,
    DBIE_EINVAL = 1, /* null pointer, nx/ny < 1, h <= 0, M < 0, bad option            */
    DBIE_ENOMEM = 2, /* device or host allocation failed                              */
    DBIE_ECUDA = 3,  /* a CUDA call failed; see dbie_last_cuda_error                  */
    DBIE_ESTATE = 4  /* the context lacks what the call needs (e.g. no fp32 copy)     */
} dbie_status;

/* dbie_create flags */
#define DBIE_WITH_FP32 1u /* also keep an fp32 copy of the boundary for dbie_eval_f32 */
#define DBIE_QUAD_9NODE 2u /* Eq. 15: integrate the boundary with 9-node biquadratic
                              elements (nodes = pixel centres, 3 x 3 Gauss points per 2h x 2h element;
                              DESIGN.md O-6) instead of one source per pixel (Eq. 16 as read in A-1).
                              Needs nx, ny >= 3.  The sums then run over 3 ceil((nx-1)/2) x
                              3 ceil((ny-1)/2) weighted sources; everything else is unchanged.     */

#define DBIE_EVAL_REDUCED_SINCOS 4u /* dbie_eval / dbie_eval_host (and the fixed-lambda field lines of dbie_trace,
                              which call dbie_eval) only (reading A-12): sin and cos of the
                              reduced argument from polynomials with one coefficient fewer each (55 instead of
                              61 FP64 instructions per interaction).  Approximation error 3e-13 absolute on
                              sin/cos; measured on BASELINE config 4: max |dB|/|B| = 2e-12 against the oracle
                              (bound 1e-9).  dbie_residual, dbie_solve and the lambda-solving dbie_trace never
                              use it: their finite differences need the full-accuracy kernel. */

/* Boundary staging (Eq. 3, Eq. 16).
 * nx, ny: boundary grid, N = nx*ny, pixel k = iy*nx + ix (x fastest).
 * h: pixel size.  (x0, y0): coordinate of the CORNER of pixel (0,0); its centre is
 * (x0 + h/2, y0 + h/2, 0) (reading A-1).  bx, by, bz: N doubles each, device, read once.
 * Outside the nx*ny window the field is zero (reading A-4).
 * The call synchronises the device before returning. */
dbie_status dbie_create(dbie_ctx** out, int nx, int ny, double h, double x0, double y0,
                        const double* bx, const double* by, const double* bz, unsigned flags);
/* Same with HOST boundary arrays. */
dbie_status dbie_create_host(dbie_ctx** out, int nx, int ny, double h, double x0, double y0,
                             const double* bx, const double* by, const double* bz,
                             unsigned flags);
void dbie_destroy(dbie_ctx* ctx);

/* Eq. 6 / Eq. 16 at given lambda.
 * x, y, z: M each, z > 0.  lam: 3*M, lam[p*M+i] = lambda_p(i); only |lambda| matters
 * (the kernel is even in lambda, reading A-3).  B: out, 3*M.  M = 0 is a no-op. */
dbie_status dbie_eval(dbie_ctx* ctx, long long M, const double* x, const double* y,
                      const double* z, const double* lam, double* B, void* cuda_stream);
dbie_status dbie_eval_host(dbie_ctx* ctx, long long M, const double* x, const double* y,
                           const double* z, const double* lam, double* B);

/* fp32-arithmetic variant of dbie_eval (BASELINE.json config 4 "fp64 and fp32"; needs a context
 * created with DBIE_WITH_FP32, else DBIE_ESTATE).  x, y, z: M floats each; lam: 3*M floats;
 * B: out, 3*M floats; all DEVICE pointers.  Geometry, theta, sincos and products are fp32; the
 * sum of a row segment (<= 512 pixels) is fp32 and row sums are carried in fp64.  Target accuracy
 * (north_star): relative vector error <= 2e-4 against the fp64 definition. */
dbie_status dbie_eval_f32(dbie_ctx* ctx, long long M, const float* x, const float* y,
                          const float* z, const float* lam, float* B, void* cuda_stream);
/* Same with HOST arrays (BASELINE.json config 4 "fp64 and fp32": the end-to-end leg of the fp32 variant): the
 * copies in and out are inside the call, which returns when B is in the host array. */
dbie_status dbie_eval_f32_host(dbie_ctx* ctx, long long M, const float* x, const float* y,
                               const float* z, const float* lam, float* B);

/* dbie_eval for callers that must not allocate device memory.
 *
 * Who needs it: dbie_eval keeps its per-chunk partial sums (Eq. 16's sum is split into up to 16 row
 * chunks, added in chunk order) in a buffer the context obtains with cudaMalloc on first use and
 * regrows when M grows.  Some hosts cannot tolerate that: a program that hands the whole of HBM to its
 * own pool at start-up, so that a later cudaMalloc fails; a real-time or in-situ loop (field
 * extrapolation next to an MHD step) in which cudaMalloc / cudaFree, which may synchronise the whole
 * device, must never run; code that holds a lock other threads' allocations wait on.  For them this
 * entry point computes exactly what dbie_eval computes (same kernels, same summation order: the two
 * results are bit-identical) with the partial sums in a fixed array that is part of the library image.
 *
 * The limit: M <= DBIE_NOALLOC_MAX_POINTS (16,384 points per call; loop over larger sets).  The array is
 * 16 chunks x 3 components x 16,384 points x 8 B = 6 MiB of device memory on every GPU that loads the
 * library, held until the process exits whether or not this function is ever called.  A larger M returns
 * DBIE_EINVAL before anything is launched, and dbie_last_cuda_error(ctx) then names the limit.
 *
 * What the call does not do: no cudaMalloc, cudaFree, event or stream creation, and nothing is grown or
 * cached in the context (profile mode is ignored, dbie_last_kernel_time keeps the previous call's events).
 * x, y, z, lam, B are caller-allocated DEVICE arrays as in dbie_eval.  The context must exist already:
 * dbie_create does allocate (the staged boundary), so create contexts during start-up.
 *
 * First call per device: the first call on a given GPU looks up the device address of the array
 * (cudaGetSymbolAddress, done once per device and remembered) and, like any first launch, lets the CUDA
 * runtime load the kernels.  Make that first call during set-up, before any stream capture is begun.
 *
 * Sharing: there is ONE array per GPU, shared by every context, stream and host thread of the process.
 * Two dbie_eval_noalloc calls whose kernels may overlap on the GPU (different streams, or different host
 * threads) race on it and give wrong results; run them on one stream or order them with events.  The
 * array keeps the previous call's partial sums; nothing in it has to start at zero, because every element
 * the epilogue reads is written by the same call's interaction kernel first, so the call clears nothing.
 * Asynchronous on the stream, like dbie_eval.  M = 0 is a no-op. */
#define DBIE_NOALLOC_MAX_POINTS 16384
dbie_status dbie_eval_noalloc(dbie_ctx* ctx, long long M, const double* x, const double* y,
                              const double* z, const double* lam, double* B, void* cuda_stream);
/* DBIE_NOALLOC_MAX_POINTS of the loaded library (for bindings that cannot read the macro). */
long long dbie_noalloc_max_points(void);

/* Options of dbie_solve.  Fill with dbie_solve_default_opts, then change fields. */
typedef struct {
    int method;       /* 0 = NM: Downhill Simplex; 1 = GRID (O-4)     */
    double delta;     /* finite-difference step as a FRACTION of h; 1e-3        */
    double cell;      /* d in g_i = |div B| (d/6) / |B|, fraction of h; 1.0 (reading A-6)     */
    double w_g;       /* Phi = f + w_g g; 1.0 (reading A-7)                                   */
    double eps_f;     /* Eq. 12 thresholds; 1e-3, 1e-4 (reading A-8)         */
    double eps_g;
    double lam0;      /* NM initial simplex: V0 = (lam0,lam0,lam0)/h, V_j = V0 + step/h e_j;  */
    double step;      /*   0.05, 0.05 (reading A-9)                                           */
    double xtol;      /* NM stop: max |V_j - V_0| <= xtol/h and max |Phi_j - Phi_0| <= ftol;  */
    double ftol;      /*   1e-4, 1e-6                                                         */
    int maxiter;      /* NM iteration cap; 200 (0 <= maxiter <= 2^24, else DBIE_EINVAL)                 */
    int n_trial;      /* GRID: T trial lambda per component per level, 4 <= T <= 32 (else
                         DBIE_EINVAL: below 4 the refined window 2W/(T-1) does not shrink); 8.
                         Multiples of 8 (then 4, then 2) run fastest.                            */
    int n_level;      /* GRID: number of refinement levels (>= 1); 10                           */
    double lam_max;   /* GRID: search window [0, lam_max/h] (> 0); 0.4                          */
    int use_eq12;     /* 1: stop a point as soon as f <= eps_f and g <= eps_g (Eq. 12)        */
    int analytic;     /* 0 (default): J and div B from the finite differences of Eq. 13 (the
                         paper's method).  1: from the analytic gradient of Eq. 6, a second sum
                         over the same pixels with d/dr[n(lambda r)/r^3] = lambda^2 cos(lambda r)/r^2
                         - 3 n(lambda r)/r^4 ("possible if the function f_i can be
                         calculated analytically"; O-5): one evaluation position instead
                         of four per objective evaluation; delta is ignored.                                  */
} dbie_solve_opts;

void dbie_solve_default_opts(dbie_solve_opts* opts);

/* Per-point lambda optimisation.  The whole search
 * runs on the device; no per-iteration data returns to the host.
 * B: out 3*M, field at lambda*.  lam: out 3*M, lambda* >= 0 (reading A-3).
 * resid: out 2*M, resid[i] = f_i (Eq. 8), resid[M+i] = g_i (Eq. 9) at lambda*.
 * iters: out M (NM iterations / GRID levels done).  status: out M: 0 = Eq. 12 thresholds
 * met, 1 = simplex tolerance (GRID: all levels done), 2 = maxiter, 3 = invalid point.
 * M must be < 2^31.  Large M is processed in batches (the context's scratch is bounded); a
 * point's result does not depend on the batch or on M. */
dbie_status dbie_solve(dbie_ctx* ctx, long long M, const double* x, const double* y,
                       const double* z, const dbie_solve_opts* opts, double* B, double* lam,
                       double* resid, int* iters, int* status, void* cuda_stream);
dbie_status dbie_solve_host(dbie_ctx* ctx, long long M, const double* x, const double* y,
                            const double* z, const dbie_solve_opts* opts, double* B,
                            double* lam, double* resid, int* iters, int* status);

/* Eq. 8, 9, 13, 14 at given lambda triples (one objective evaluation per point; the same
 * code path the solver uses).  out: 9*M, rows B_x,B_y,B_z, f, g, J_x,J_y,J_z, div B.
 * delta, cell, w_g, analytic are taken from opts (NULL = defaults).  phi: out M (may be NULL). */
dbie_status dbie_residual(dbie_ctx* ctx, long long M, const double* x, const double* y,
                          const double* z, const double* lam, const dbie_solve_opts* opts,
                          double* out, double* phi, void* cuda_stream);

/* Field-line and current-line tracing.  The paper draws lines of the reconstructed B
 * and "current lines" of J = curl B (Eq. 14) in its Figs. 5-11
 * without giving the integrator; reading T-1 of DESIGN.md: dr/ds = direction * v/|v| in arc length s,
 * classical RK4 at a fixed step, v = B or J evaluated by this library AT the four stage points of
 * every step (nothing is interpolated): B and lambda from the per-point search of dbie_solve (or Eq. 6
 * at a fixed lambda triple), J from the stencil of Eq. 13 at that lambda. */
typedef struct {
    double ds;         /* arc-length step as a FRACTION of h; 0.5                                       */
    int max_steps;     /* S: steps per line (each line stores up to S + 1 points); 100                  */
    int direction;     /* +1: along v; -1: against v                                                    */
    int current;       /* 0: field lines (v = B); 1: current lines (v = J, Eq. 14)                      */
    int fixed_lambda;  /* 0: lambda from the per-point search (solve options); 1: the triple `lam`      */
    double lam[3];     /* fixed lambda triple, units 1/length (0, 0, 0 = the potential field)           */
    double z_min;      /* a line lives in z_min h < z <= z_max h and inside the magnetogram window;     */
    double z_max;      /*   0, 1e300                                                                    */
} dbie_trace_opts;

void dbie_trace_default_opts(dbie_trace_opts* opts);

/* x0, y0, z0: L seed points (device).  sopts: options of the lambda search and of Eq. 13 (NULL = defaults).
 * path: out, 3*(S+1)*L doubles, point k of line i at path[(c*(S+1) + k)*L + i], c = 0, 1, 2; NaN beyond a
 * line's last point.  npts: out L, points stored (0 if the seed is outside the region).  status: out L:
 * 0 = max_steps reached, 1 = left the region (a stage point or the new point), 2 = v zero or not finite at
 * a stage point.  Asynchronous on the stream; 4 S field evaluations of L points are enqueued, lines that
 * have stopped cost nothing in the lambda search (with a fixed lambda, and for current lines, a stopped line still
 * pays its sums: they are evaluated for all L lines at every stage). */
dbie_status dbie_trace(dbie_ctx* ctx, long long L, const double* x0, const double* y0, const double* z0,
                       const dbie_solve_opts* sopts, const dbie_trace_opts* topts, double* path, int* npts,
                       int* status, void* cuda_stream);

/* ------------------------------------------------------------------------------------------------
 * Diagnostics and measurement.  Not needed to use the library; bench.py and the tests call them.
 * ---------------------------------------------------------------------------------------------- */

/* Counters of the last eval/solve/residual call on this context (host values, valid after
 * the stream has been synchronised): point-pixel interactions evaluated (one interaction =
 * one (evaluation point, pixel) pair, all three components), kernel launches enqueued, and
 * objective evaluations.  Any pointer may be NULL.  After dbie_trace the interactions and evaluations cover the
 * eval / residual calls of the trace only: the lambda searches of a lambda-solving trace are NOT included (each inner
 * solve restarts the device counter), so treat them as undefined there. */
dbie_status dbie_last_counters(dbie_ctx* ctx, double* interactions, long long* launches,
                               long long* objective_evals);

/* Profile mode: when enabled, every later eval/residual/solve call on this context records a
 * CUDA-event pair around each launch of the interaction kernel (on the caller's stream).
 * dbie_last_kernel_time waits for the last call's events and returns the summed device time of
 * its interaction-kernel launches and their number. */
dbie_status dbie_profile(dbie_ctx* ctx, int enable);
dbie_status dbie_last_kernel_time(dbie_ctx* ctx, double* interact_ms, long long* interact_launches);

/* Profile mode, Nelder-Mead solve: the pass timeline of the LAST fused launch of the last dbie_solve call (its last
 * batch).  active[i] = points still searching at the start of pass i, ms[i] = duration of pass i on the device
 * (%globaltimer of CTA 0 at consecutive pass starts).  cap: capacity of the two host arrays; *npass = passes of the
 * launch (may exceed cap; 0 if nothing was recorded, and 0 whenever the context's LAST call was anything but a
 * profiled Nelder-Mead dbie_solve: an eval, residual, GRID solve or trace in between invalidates the timeline).  At
 * most the first 65,536 passes of a launch are recorded.  Synchronises the device. */
dbie_status dbie_last_pass_trace(dbie_ctx* ctx, int cap, long long* active, double* ms, int* npass);

/* Measured peak of the FP64 pipe: runs a register-only DFMA loop on every SM for about
 * `millis` ms and returns DFMA instructions (per lane) per second.  Synchronises. */
dbie_status dbie_probe_dfma_rate(double millis, double* dfma_per_s, double* ffma_per_s);

/* FP64 issue cost by operand pattern (the design rule of the interaction kernels):
 * rates[0] = DFMA with two register operands and an immediate, rates[1] = DFMA reading three different,
 * changing registers, rates[2] = DMUL, rates[3] = DFMA with one changing and two loop-invariant registers
 * (operand-reuse cache); lane-instructions per second, about `millis` ms each.  Synchronises. */
dbie_status dbie_probe_fp64_operands(double millis, double* rates /* host, 4 */);

/* Tuning knob of dbie_eval_f32: bit p of mask set = component p takes sin/cos of the reduced
 * argument from the SFU (MUFU.SIN/COS after a reduction by 2 pi); bit clear = from the fp32 angle table in
 * shared memory (the fp64 kernel's scheme in fp32, no MUFU).  Allowed masks: 0, 1, 3, 7 (default: all three
 * from the SFU, the fastest measured: 5.6e11 interactions/s against 5.4e11 / 5.0e11 / 4.6e11 for 3 / 1 / 0).
 * Results differ at the 1e-6 level between masks; all meet the 2e-4 target (measured 4e-5). */
dbie_status dbie_set_f32_sfu_mask(dbie_ctx* ctx, int mask);

/* Test knob: process eval / residual / solve in internal batches of at most `points` points
 * (0 restores the defaults: 2^21 for eval, 2^22 for residual and the Nelder-Mead solve, a 2 GiB
 * scratch bound for GRID).  Results do not depend on it, bit for bit; the tests use it to run the
 * multi-batch paths at small sizes. */
dbie_status dbie_debug_set_batch_limit(dbie_ctx* ctx, long long points);

const char* dbie_strerror(dbie_status s);
/* CUDA error string of the last DBIE_ECUDA on this context (or of the last failure with
 * no context when ctx is NULL).  Never NULL. */
const char* dbie_last_cuda_error(const dbie_ctx* ctx);
/* Library version string, e.g. "dbie-b200 0.2 (sm_100a)". */
const char* dbie_version(void);

#ifdef __cplusplus
}
#endif
#endif /* DBIE_H */
