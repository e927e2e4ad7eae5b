// dbie_api.cu — the C ABI of include/dbie.h: argument checks, context and scratch management,
// and the launch sequences of eval / residual / solve.  No arithmetic of the method lives here.
#include <cuda_runtime.h>
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <mutex>

#include <nvtx3/nvToolsExt.h>   // header-only; ranges show up in Nsight tools, a no-op otherwise

#include "dbie_internal.h"

using namespace dbie;

namespace {
struct NvtxRange {   // ranges around create / eval / residual / solve
    explicit NvtxRange(const char* name) { nvtxRangePushA(name); }
    ~NvtxRange() { nvtxRangePop(); }
};
}  // namespace

struct dbie_ctx {
    int device, sm_count;
    int win_nx, win_ny;                       // the magnetogram's pixel grid (bd.nx, bd.ny count SOURCES: 9-node staging changes them)
    BoundaryView bd;
    double4* rec;
    double* yk;
    float4* rec32;
    float* yk32;
    double* part;       size_t part_bytes;    // chunk partial sums
    char* state;        size_t state_bytes;   // optimiser state
    char* io;           size_t io_bytes;      // device staging of the _host entry points
    char* trace;        size_t trace_bytes;   // dbie_trace: line state and the field at the line heads
    unsigned* counters;                       // device: list lengths [0..2], nevals (u64) at +16 B, work-item counters at +32 B
    cudaStream_t own_stream;
    double last_interactions;
    long long last_launches, last_evals;
    int evals_on_device;                      // last call was a solve: read nevals back on demand
    int positions_per_eval;                   // evaluation positions per objective evaluation of that solve (4, or 1 analytic)
    int f32_sfu_mask;                         // dbie_eval_f32: components whose sincos use the SFU
    bool eval_reduced;                        // DBIE_EVAL_REDUCED_SINCOS: dbie_eval uses the reduced-degree sincos
    long long batch_limit;                    // dbie_debug_set_batch_limit: points per internal batch (0: defaults)
    int profile;                              // record CUDA events around every interaction launch
    unsigned long long* pass_trace;           // profile mode: pass timeline of the last fused Nelder-Mead launch
    int pass_trace_cap;
    bool pass_trace_valid;                    // the buffer holds the timeline of the LAST call (a profiled NM solve); any other call clears it
    int coop_launch;                          // cudaDevAttrCooperativeLaunch of the device (the Nelder-Mead solve needs it)
    cudaEvent_t* ev;    int ev_cap, ev_n;     // event pairs of the last call (profile mode)
    char err[256];
};

static char g_err[256] = "no error";
static const size_t kCounterBytes = 128;   // device counters: list lengths [0..2], objective evaluations (u64) at +16 B, work items at +32 B
static const int kMaxIter = 1 << 24;       // dbie_solve_opts.maxiter above this is refused (the pass bound 5 maxiter + 5 stays far inside int)
static const int kPassTraceMax = 1 << 16;  // profile mode records at most this many passes of a fused launch (1 MiB)
static const int kDefaultF32SfuMask = 7;   // sin/cos of the reduced argument from the SFU for all three components:
                                           // measured fastest (4.90e11 vs 4.26e11 interactions/s with polynomials), same accuracy

static dbie_status fail_cuda(dbie_ctx* c, cudaError_t e, const char* where) {
    char* dst = c ? c->err : g_err;
    snprintf(dst, 256, "%s: %s", where, cudaGetErrorString(e));
    if (c) memcpy(g_err, c->err, 256);
    (void)cudaGetLastError();
    return e == cudaErrorMemoryAllocation ? DBIE_ENOMEM : DBIE_ECUDA;
}
#define CU(call)                                                   \
    do {                                                           \
        cudaError_t e_ = (call);                                   \
        if (e_ != cudaSuccess) return fail_cuda(ctx, e_, #call);   \
    } while (0)

// A context belongs to the device that was current in dbie_create.  Every entry point makes that device
// current for the duration of the call and restores the caller's device on return, so a context can be
// used after the caller switched devices (pointers must still belong to the context's device).
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    cudaError_t err = cudaSuccess;
    explicit DeviceGuard(const dbie_ctx* c);
    ~DeviceGuard() {
        if (switched) (void)cudaSetDevice(prev);
    }
};

static dbie_status ensure(dbie_ctx* ctx, void** ptr, size_t* have, size_t need) {
    if (need <= *have) return DBIE_OK;
    if (*ptr) {
        CU(cudaFree(*ptr));   // synchronises the device: nothing in flight uses the old buffer after this
        *ptr = nullptr;
        *have = 0;
    }
    CU(cudaMalloc(ptr, need));
    *have = need;
    return DBIE_OK;
}

DeviceGuard::DeviceGuard(const dbie_ctx* c) {
    err = cudaGetDevice(&prev);
    if (err == cudaSuccess && c && prev != c->device) {
        err = cudaSetDevice(c->device);
        switched = err == cudaSuccess;
    }
}
#define GUARD_DEVICE()                                                          \
    DeviceGuard guard_(ctx);                                                    \
    if (guard_.err != cudaSuccess) return fail_cuda(ctx, guard_.err, "cudaSetDevice(context's device)")

// profile mode: an event pair around each interaction-kernel launch of the current call
static void prof_reset(dbie_ctx* ctx) { ctx->ev_n = 0; }
static void prof_mark(dbie_ctx* ctx, cudaStream_t st) {
    if (!ctx->profile) return;
    if (ctx->ev_n == ctx->ev_cap) {
        const int ncap = ctx->ev_cap ? 2 * ctx->ev_cap : 256;
        cudaEvent_t* n = (cudaEvent_t*)realloc(ctx->ev, sizeof(cudaEvent_t) * ncap);
        if (!n) return;
        for (int i = ctx->ev_cap; i < ncap; ++i) cudaEventCreate(&n[i]);
        ctx->ev = n;
        ctx->ev_cap = ncap;
    }
    cudaEventRecord(ctx->ev[ctx->ev_n++], st);
}

extern "C" dbie_status dbie_profile(dbie_ctx* ctx, int enable) {
    if (!ctx) return DBIE_EINVAL;
    ctx->profile = enable != 0;
    return DBIE_OK;
}

extern "C" dbie_status dbie_last_kernel_time(dbie_ctx* ctx, double* interact_ms, long long* interact_launches) {
    if (!ctx) return DBIE_EINVAL;
    GUARD_DEVICE();
    double total = 0.0;
    const int pairs = ctx->ev_n / 2;
    if (pairs > 0) CU(cudaEventSynchronize(ctx->ev[2 * pairs - 1]));
    for (int i = 0; i < pairs; ++i) {
        float ms = 0.f;
        CU(cudaEventElapsedTime(&ms, ctx->ev[2 * i], ctx->ev[2 * i + 1]));
        total += ms;
    }
    if (interact_ms) *interact_ms = total;
    if (interact_launches) *interact_launches = pairs;
    return DBIE_OK;
}

extern "C" dbie_status dbie_last_pass_trace(dbie_ctx* ctx, int cap, long long* active, double* ms, int* npass) {
    if (!ctx || cap < 0 || !npass || (cap > 0 && (!active || !ms))) return DBIE_EINVAL;
    GUARD_DEVICE();
    *npass = 0;
    if (!ctx->pass_trace || !ctx->pass_trace_valid) return DBIE_OK;   // the last call was not a profiled Nelder-Mead solve
    CU(cudaDeviceSynchronize());
    const int n = ctx->pass_trace_cap;
    unsigned long long* h = (unsigned long long*)malloc(sizeof(unsigned long long) * 2 * n);
    if (!h) return DBIE_ENOMEM;
    const cudaError_t e = cudaMemcpy(h, ctx->pass_trace, sizeof(unsigned long long) * 2 * n, cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) { free(h); return fail_cuda(ctx, e, "dbie_last_pass_trace"); }
    // passes are the entries before the first stamp with no active point (the stamp of the search's end)
    int np = 0;
    while (np < n && h[2 * np] != 0ull) ++np;
    const bool have_end = np < n && h[2 * np + 1] != 0ull;
    const int full = have_end ? np : (np > 0 ? np - 1 : 0);   // passes with both a start and an end stamp
    for (int i = 0; i < full && i < cap; ++i) {
        active[i] = (long long)h[2 * i];
        ms[i] = (double)(h[2 * i + 3] - h[2 * i + 1]) * 1e-6;
    }
    *npass = full;
    free(h);
    return DBIE_OK;
}

extern "C" const char* dbie_strerror(dbie_status s) {
    switch (s) {
        case DBIE_OK: return "ok";
        case DBIE_EINVAL: return "invalid argument";
        case DBIE_ENOMEM: return "out of memory";
        case DBIE_ECUDA: return "CUDA error (see dbie_last_cuda_error)";
        case DBIE_ESTATE: return "context lacks what the call needs";
    }
    return "unknown status";
}
extern "C" const char* dbie_last_cuda_error(const dbie_ctx* ctx) { return ctx ? ctx->err : g_err; }
extern "C" const char* dbie_version(void) { return "dbie-b200 0.2 (sm_100a)"; }

extern "C" void dbie_solve_default_opts(dbie_solve_opts* o) {
    if (!o) return;
    memset(o, 0, sizeof *o);
    o->method = 0;
    o->delta = 1e-3;
    o->cell = 1.0;
    o->w_g = 1.0;
    o->eps_f = 1e-3;
    o->eps_g = 1e-4;
    o->lam0 = 0.05;
    o->step = 0.05;
    o->xtol = 1e-4;
    o->ftol = 1e-6;
    o->maxiter = 200;
    o->n_trial = 8;
    o->n_level = 10;
    o->lam_max = 0.4;
    o->use_eq12 = 1;
    o->analytic = 0;
}

static void setup_tiling(BoundaryView& b) {
    if (b.nx <= kTilePx) {
        b.tile_rows = kTilePx / b.nx;
        if (b.tile_rows < 1) b.tile_rows = 1;
        b.segs_per_row = 1;
        b.seg_w = b.nx;
        b.ntiles = (b.ny + b.tile_rows - 1) / b.tile_rows;
    } else {
        b.tile_rows = 1;
        b.segs_per_row = (b.nx + kTilePx - 1) / kTilePx;
        b.seg_w = (b.nx + b.segs_per_row - 1) / b.segs_per_row;
        b.seg_w += b.seg_w & 1;
        b.ntiles = b.ny * b.segs_per_row;
    }
    b.nunits = b.ny * b.segs_per_row;
    b.nchunks = b.nunits < kMaxChunks ? b.nunits : kMaxChunks;
}

extern "C" void dbie_destroy(dbie_ctx* ctx) {
    if (!ctx) return;
    DeviceGuard guard_(ctx->device >= 0 ? ctx : nullptr);
    cudaFree(ctx->rec);
    cudaFree(ctx->yk);
    cudaFree(ctx->rec32);
    cudaFree(ctx->yk32);
    cudaFree(ctx->part);
    cudaFree(ctx->state);
    cudaFree(ctx->io);
    cudaFree(ctx->trace);
    cudaFree(ctx->pass_trace);
    cudaFree(ctx->counters);
    if (ctx->own_stream) cudaStreamDestroy(ctx->own_stream);
    for (int i = 0; i < ctx->ev_cap; ++i) cudaEventDestroy(ctx->ev[i]);
    free(ctx->ev);
    (void)cudaGetLastError();
    free(ctx);
}

extern "C" dbie_status dbie_create(dbie_ctx** out, int nx, int ny, double h, double x0, double y0,
                                   const double* bx, const double* by, const double* bz, unsigned flags) {
    if (!out) return DBIE_EINVAL;
    *out = nullptr;
    if (nx < 1 || ny < 1 || !(h > 0.0) || !isfinite(h) || !isfinite(x0) || !isfinite(y0) || !bx || !by || !bz)
        return DBIE_EINVAL;
    if ((long long)nx * ny > (1LL << 30)) return DBIE_EINVAL;
    if ((flags & DBIE_QUAD_9NODE) && (nx < 3 || ny < 3)) return DBIE_EINVAL;
    NvtxRange nvtx_("dbie_create");
    dbie_ctx* ctx = (dbie_ctx*)calloc(1, sizeof(dbie_ctx));
    if (!ctx) return DBIE_ENOMEM;
    strcpy(ctx->err, "no error");
    ctx->f32_sfu_mask = kDefaultF32SfuMask;
    dbie_status st = DBIE_OK;
    do {
        cudaError_t e;
        if ((e = cudaGetDevice(&ctx->device)) != cudaSuccess) { st = fail_cuda(ctx, e, "cudaGetDevice"); break; }
        if ((e = cudaDeviceGetAttribute(&ctx->sm_count, cudaDevAttrMultiProcessorCount, ctx->device)) != cudaSuccess) {
            st = fail_cuda(ctx, e, "cudaDeviceGetAttribute"); break;
        }
        if ((e = cudaDeviceGetAttribute(&ctx->coop_launch, cudaDevAttrCooperativeLaunch, ctx->device)) != cudaSuccess) {
            st = fail_cuda(ctx, e, "cudaDeviceGetAttribute(cooperative launch)"); break;
        }
        BoundaryView& b = ctx->bd;
        const bool q9 = (flags & DBIE_QUAD_9NODE) != 0;
        ctx->eval_reduced = (flags & DBIE_EVAL_REDUCED_SINCOS) != 0;
        // 9-node elements: the sources are 3 Gauss abscissae per element and direction (O-6)
        const int sx = q9 ? 3 * (nx / 2) : nx, sy = q9 ? 3 * (ny / 2) : ny;
        ctx->win_nx = nx; ctx->win_ny = ny;
        b.nx = sx; b.ny = sy; b.N = (long long)sx * sy;
        b.h = h; b.x0 = x0; b.y0 = y0;
        setup_tiling(b);
        if ((e = cudaMalloc(&ctx->rec, sizeof(double4) * b.N)) != cudaSuccess) { st = fail_cuda(ctx, e, "cudaMalloc(rec)"); break; }
        if ((e = cudaMalloc(&ctx->yk, sizeof(double) * b.ny)) != cudaSuccess) { st = fail_cuda(ctx, e, "cudaMalloc(yk)"); break; }
        if (flags & DBIE_WITH_FP32) {
            if ((e = cudaMalloc(&ctx->rec32, sizeof(float4) * b.N)) != cudaSuccess) { st = fail_cuda(ctx, e, "cudaMalloc(rec32)"); break; }
            if ((e = cudaMalloc(&ctx->yk32, sizeof(float) * b.ny)) != cudaSuccess) { st = fail_cuda(ctx, e, "cudaMalloc(yk32)"); break; }
        }
        if ((e = cudaMalloc(&ctx->counters, kCounterBytes)) != cudaSuccess) { st = fail_cuda(ctx, e, "cudaMalloc(counters)"); break; }
        if ((e = cudaMemset(ctx->counters, 0, kCounterBytes)) != cudaSuccess) { st = fail_cuda(ctx, e, "cudaMemset"); break; }
        if ((e = cudaStreamCreateWithFlags(&ctx->own_stream, cudaStreamNonBlocking)) != cudaSuccess) { st = fail_cuda(ctx, e, "cudaStreamCreate"); break; }
        e = q9 ? launch_stage_q9(nx, ny, h, x0, y0, bx, by, bz, sx, sy, ctx->rec, ctx->yk, ctx->rec32, ctx->yk32, 0)
               : launch_stage_boundary(nx, ny, h, x0, y0, bx, by, bz, ctx->rec, ctx->yk, ctx->rec32, ctx->yk32, 0);
        if (e != cudaSuccess) {
            st = fail_cuda(ctx, e, "stage_boundary"); break;
        }
        if ((e = cudaDeviceSynchronize()) != cudaSuccess) { st = fail_cuda(ctx, e, "stage_boundary(sync)"); break; }
        b.rec = ctx->rec; b.yk = ctx->yk; b.rec32 = ctx->rec32; b.yk32 = ctx->yk32;
    } while (0);
    if (st != DBIE_OK) {
        memcpy(g_err, ctx->err, 256);
        dbie_destroy(ctx);
        return st;
    }
    *out = ctx;
    return DBIE_OK;
}

extern "C" dbie_status dbie_create_host(dbie_ctx** out, int nx, int ny, double h, double x0, double y0,
                                        const double* bx, const double* by, const double* bz, unsigned flags) {
    if (!out) return DBIE_EINVAL;
    *out = nullptr;
    if (nx < 1 || ny < 1 || !bx || !by || !bz) return DBIE_EINVAL;
    dbie_ctx* ctx = nullptr;   // for CU()
    const size_t n = (size_t)nx * ny;
    double* d = nullptr;
    CU(cudaMalloc(&d, 3 * n * sizeof(double)));
    cudaError_t e = cudaMemcpy(d, bx, n * sizeof(double), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(d + n, by, n * sizeof(double), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(d + 2 * n, bz, n * sizeof(double), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) { cudaFree(d); return fail_cuda(nullptr, e, "cudaMemcpy(boundary)"); }
    const dbie_status st = dbie_create(out, nx, ny, h, x0, y0, d, d + n, d + 2 * n, flags);
    cudaFree(d);
    return st;
}

// ------------------------------------------------------------------------------ eval ------
static const long long kEvalBatch = 1LL << 21;
static const long long kStencilBatch = 1LL << 22;
static long long eval_batch(const dbie_ctx* c) { return c->batch_limit > 0 ? c->batch_limit : kEvalBatch; }
static long long stencil_batch(const dbie_ctx* c) { return c->batch_limit > 0 ? c->batch_limit : kStencilBatch; }

extern "C" dbie_status dbie_debug_set_batch_limit(dbie_ctx* ctx, long long points) {
    if (!ctx || points < 0) return DBIE_EINVAL;
    ctx->batch_limit = points;
    return DBIE_OK;
}

extern "C" dbie_status dbie_eval(dbie_ctx* ctx, long long M, const double* x, const double* y, const double* z,
                                 const double* lam, double* B, void* cuda_stream) {
    if (!ctx || M < 0) return DBIE_EINVAL;
    if (M == 0) return DBIE_OK;
    if (!x || !y || !z || !lam || !B) return DBIE_EINVAL;
    GUARD_DEVICE();
    NvtxRange nvtx_("dbie_eval");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const long long cap = M < eval_batch(ctx) ? M : eval_batch(ctx);
    const dbie_status s = ensure(ctx, (void**)&ctx->part, &ctx->part_bytes,
                                 (size_t)ctx->bd.nchunks * 3 * cap * sizeof(double));
    if (s != DBIE_OK) return s;
    long long launches = 0;
    prof_reset(ctx);
    for (long long off = 0; off < M; off += cap) {
        const long long cnt = (M - off < cap) ? (M - off) : cap;
        InteractParams p;
        memset(&p, 0, sizeof p);
        p.bd = ctx->bd;
        p.x = x; p.y = y; p.z = z; p.lam = lam; p.ldlam = M;
        p.count = cnt; p.slot0 = off;
        p.part = ctx->part; p.cap = cap;
        prof_mark(ctx, st);
        int nparts = ctx->bd.nchunks;
        CU(launch_interact_eval(p, ctx->sm_count, ctx->eval_reduced, &nparts, st));
        prof_mark(ctx, st);
        CU(launch_eval_finalize(ctx->bd, nparts, off, cnt, M, z, lam, ctx->part, cap, B, st));
        launches += 2;
    }
    ctx->last_interactions = (double)M * (double)ctx->bd.N;
    ctx->last_launches = launches;
    ctx->last_evals = 0;
    ctx->evals_on_device = 0;
    ctx->pass_trace_valid = false;
    return DBIE_OK;
}

static dbie_status io_reserve(dbie_ctx* ctx, size_t bytes) { return ensure(ctx, (void**)&ctx->io, &ctx->io_bytes, bytes); }

extern "C" dbie_status dbie_eval_host(dbie_ctx* ctx, long long M, const double* x, const double* y,
                                      const double* z, const double* lam, double* B) {
    if (!ctx || M < 0) return DBIE_EINVAL;
    if (M == 0) return DBIE_OK;
    if (!x || !y || !z || !lam || !B) return DBIE_EINVAL;
    GUARD_DEVICE();
    const size_t m = (size_t)M * sizeof(double);
    CU(cudaDeviceSynchronize());   // earlier work on this context may be in flight on another stream
    dbie_status s = io_reserve(ctx, 9 * m);
    if (s != DBIE_OK) return s;
    double* d = (double*)ctx->io;   // x, y, z, lam[3], B[3]
    cudaStream_t st = ctx->own_stream;
    CU(cudaMemcpyAsync(d, x, m, cudaMemcpyHostToDevice, st));
    CU(cudaMemcpyAsync(d + M, y, m, cudaMemcpyHostToDevice, st));
    CU(cudaMemcpyAsync(d + 2 * M, z, m, cudaMemcpyHostToDevice, st));
    CU(cudaMemcpyAsync(d + 3 * M, lam, 3 * m, cudaMemcpyHostToDevice, st));
    s = dbie_eval(ctx, M, d, d + M, d + 2 * M, d + 3 * M, d + 6 * M, st);
    if (s != DBIE_OK) return s;
    CU(cudaMemcpyAsync(B, d + 6 * M, 3 * m, cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    return DBIE_OK;
}

// ------------------------------------------------------------------ eval, no allocation ---
// dbie_eval for callers that cannot allocate device memory (a process whose own pool owns all of HBM, a
// real-time loop that must never hit the device-wide synchronisation of cudaMalloc / cudaFree): the chunk
// partial sums live in this fixed array instead of the context's lazily grown buffer.  It is part of the
// library image, so every GPU that loads the library holds these 6 MiB until the process exits.
static const long long kNoAllocMaxPoints = DBIE_NOALLOC_MAX_POINTS;
static __device__ __align__(256) double g_noalloc_part[(size_t)kMaxChunks * 3 * DBIE_NOALLOC_MAX_POINTS];

// In host code `g_noalloc_part` is only a handle for the runtime, not a device address: the address a kernel
// may use comes from cudaGetSymbolAddress, asked once per device with that device current and kept here.
static const int kNoAllocMaxDevices = 64;
static double* g_noalloc_addr[kNoAllocMaxDevices];   // zero-initialised: "not looked up yet"
static std::mutex g_noalloc_mutex;

static dbie_status noalloc_scratch(dbie_ctx* ctx, double** out) {   // ctx's device is current
    const int dev = ctx->device;
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    if (dev >= 0 && dev < kNoAllocMaxDevices && g_noalloc_addr[dev]) {
        *out = g_noalloc_addr[dev];
        return DBIE_OK;
    }
    double* ptr = nullptr;
    CU(cudaGetSymbolAddress((void**)&ptr, g_noalloc_part));
    if (!ptr) {
        snprintf(ctx->err, 256, "dbie_eval_noalloc: cudaGetSymbolAddress returned a null address");
        return DBIE_ECUDA;
    }
    if (dev >= 0 && dev < kNoAllocMaxDevices) g_noalloc_addr[dev] = ptr;   // beyond the table: asked again every call
    *out = ptr;
    return DBIE_OK;
}

extern "C" long long dbie_noalloc_max_points(void) { return kNoAllocMaxPoints; }

extern "C" dbie_status dbie_eval_noalloc(dbie_ctx* ctx, long long M, const double* x, const double* y,
                                         const double* z, const double* lam, double* B, void* cuda_stream) {
    if (!ctx || M < 0) return DBIE_EINVAL;
    if (M == 0) return DBIE_OK;
    if (!x || !y || !z || !lam || !B) return DBIE_EINVAL;
    if (M > kNoAllocMaxPoints) {
        snprintf(ctx->err, 256, "dbie_eval_noalloc: M = %lld exceeds DBIE_NOALLOC_MAX_POINTS = %lld (the fixed "
                 "scratch array holds no more; split the points over several calls)", M, kNoAllocMaxPoints);
        return DBIE_EINVAL;
    }
    GUARD_DEVICE();
    NvtxRange nvtx_("dbie_eval_noalloc");
    double* part = nullptr;
    const dbie_status s = noalloc_scratch(ctx, &part);   // the first call on this device looks the address up
    if (s != DBIE_OK) return s;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // One batch (M <= the limit), laid out as dbie_eval lays out a batch of M points: part[(c*3 + q)*M + slot].
    // Every element the epilogue reads is written by the interaction launch before it, so the previous
    // call's contents are never read and nothing is cleared.
    InteractParams p;
    memset(&p, 0, sizeof p);
    p.bd = ctx->bd;
    p.x = x; p.y = y; p.z = z; p.lam = lam; p.ldlam = M;
    p.count = M; p.slot0 = 0;
    p.part = part; p.cap = M;
    int nparts = ctx->bd.nchunks;
    CU(launch_interact_eval(p, ctx->sm_count, ctx->eval_reduced, &nparts, st));
    CU(launch_eval_finalize(ctx->bd, nparts, 0, M, M, z, lam, part, M, B, st));
    ctx->last_interactions = (double)M * (double)ctx->bd.N;
    ctx->last_launches = 2;
    ctx->last_evals = 0;
    ctx->evals_on_device = 0;
    ctx->pass_trace_valid = false;
    return DBIE_OK;
}

extern "C" dbie_status dbie_eval_f32(dbie_ctx* ctx, long long M, const float* x, const float* y, const float* z,
                                     const float* lam, float* B, void* cuda_stream) {
    if (!ctx || M < 0) return DBIE_EINVAL;
    if (!ctx->rec32) {
        snprintf(ctx->err, 256, "dbie_eval_f32: the context was created without DBIE_WITH_FP32");
        return DBIE_ESTATE;
    }
    if (M == 0) return DBIE_OK;
    if (!x || !y || !z || !lam || !B) return DBIE_EINVAL;
    GUARD_DEVICE();
    NvtxRange nvtx_("dbie_eval_f32");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const long long cap = M < eval_batch(ctx) ? M : eval_batch(ctx);
    const dbie_status s = ensure(ctx, (void**)&ctx->part, &ctx->part_bytes,
                                 (size_t)ctx->bd.nchunks * 3 * cap * sizeof(double));
    if (s != DBIE_OK) return s;
    long long launches = 0;
    prof_reset(ctx);
    for (long long off = 0; off < M; off += cap) {
        const long long cnt = (M - off < cap) ? (M - off) : cap;
        InteractParamsF32 p;
        memset(&p, 0, sizeof p);
        p.bd = ctx->bd;
        p.x = x; p.y = y; p.z = z; p.lam = lam; p.ldlam = M;
        p.count = cnt; p.slot0 = off;
        p.part = ctx->part; p.cap = cap;
        prof_mark(ctx, st);
        int nparts = ctx->bd.nchunks;
        CU(launch_interact_f32(p, ctx->sm_count, ctx->f32_sfu_mask, &nparts, st));
        prof_mark(ctx, st);
        CU(launch_eval_finalize_f32(ctx->bd, nparts, off, cnt, M, z, lam, ctx->part, cap, B, st));
        launches += 2;
    }
    ctx->last_interactions = (double)M * (double)ctx->bd.N;
    ctx->last_launches = launches;
    ctx->last_evals = 0;
    ctx->evals_on_device = 0;
    ctx->pass_trace_valid = false;
    return DBIE_OK;
}

extern "C" dbie_status dbie_eval_f32_host(dbie_ctx* ctx, long long M, const float* x, const float* y, const float* z,
                                          const float* lam, float* B) {
    if (!ctx || M < 0) return DBIE_EINVAL;
    if (!ctx->rec32) {
        snprintf(ctx->err, 256, "dbie_eval_f32_host: the context was created without DBIE_WITH_FP32");
        return DBIE_ESTATE;
    }
    if (M == 0) return DBIE_OK;
    if (!x || !y || !z || !lam || !B) return DBIE_EINVAL;
    GUARD_DEVICE();
    const size_t m = (size_t)M * sizeof(float);
    CU(cudaDeviceSynchronize());   // earlier work on this context may be in flight on another stream
    dbie_status s = io_reserve(ctx, 9 * m);
    if (s != DBIE_OK) return s;
    float* d = (float*)ctx->io;   // x, y, z, lam[3], B[3]
    cudaStream_t st = ctx->own_stream;
    CU(cudaMemcpyAsync(d, x, m, cudaMemcpyHostToDevice, st));
    CU(cudaMemcpyAsync(d + M, y, m, cudaMemcpyHostToDevice, st));
    CU(cudaMemcpyAsync(d + 2 * M, z, m, cudaMemcpyHostToDevice, st));
    CU(cudaMemcpyAsync(d + 3 * M, lam, 3 * m, cudaMemcpyHostToDevice, st));
    s = dbie_eval_f32(ctx, M, d, d + M, d + 2 * M, d + 3 * M, d + 6 * M, st);
    if (s != DBIE_OK) return s;
    CU(cudaMemcpyAsync(B, d + 6 * M, 3 * m, cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    return DBIE_OK;
}

extern "C" dbie_status dbie_set_f32_sfu_mask(dbie_ctx* ctx, int mask) {
    if (!ctx || (mask != 0 && mask != 1 && mask != 3 && mask != 7)) return DBIE_EINVAL;
    ctx->f32_sfu_mask = mask;
    return DBIE_OK;
}

// ------------------------------------------------------------------------------ solve -----
static dbie_status make_consts(const dbie_ctx* ctx, const dbie_solve_opts* o, NMConsts* k) {
    dbie_solve_opts d;
    if (!o) { dbie_solve_default_opts(&d); o = &d; }
    const double h = ctx->bd.h;
    if (!(o->delta > 0.0) || !(o->cell > 0.0) || !isfinite(o->w_g) || o->maxiter < 0 || o->maxiter > kMaxIter || !(o->xtol >= 0.0) ||
        !(o->ftol >= 0.0) || !isfinite(o->lam0) || !isfinite(o->step) || o->step == 0.0)
        return DBIE_EINVAL;
    k->delta_abs = o->delta * h;
    k->d_abs = o->cell * h;
    k->w_g = o->w_g;
    k->eps_f = o->eps_f;
    k->eps_g = o->eps_g;
    k->xtol_abs = o->xtol / h;
    k->ftol = o->ftol;
    k->lam0_abs = o->lam0 / h;
    k->step_abs = o->step / h;
    k->h2_over_2pi = h * h / (2.0 * 3.14159265358979323846);
    k->maxiter = o->maxiter;
    k->use_eq12 = o->use_eq12;
    k->analytic = o->analytic != 0;
    return DBIE_OK;
}

extern "C" dbie_status dbie_residual(dbie_ctx* ctx, long long M, const double* x, const double* y,
                                     const double* z, const double* lam, const dbie_solve_opts* opts,
                                     double* out, double* phi, void* cuda_stream) {
    if (!ctx || M < 0) return DBIE_EINVAL;
    if (M == 0) return DBIE_OK;
    if (!x || !y || !z || !lam || !out) return DBIE_EINVAL;
    GUARD_DEVICE();
    NvtxRange nvtx_("dbie_residual");
    NMConsts k;
    dbie_status s = make_consts(ctx, opts, &k);
    if (s != DBIE_OK) return s;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const long long cap = M < stencil_batch(ctx) ? M : stencil_batch(ctx);
    s = ensure(ctx, (void**)&ctx->part, &ctx->part_bytes, (size_t)ctx->bd.nchunks * 12 * cap * sizeof(double));
    if (s != DBIE_OK) return s;
    long long launches = 0;
    prof_reset(ctx);
    for (long long off = 0; off < M; off += cap) {
        const long long cnt = (M - off < cap) ? (M - off) : cap;
        InteractParams p;
        memset(&p, 0, sizeof p);
        p.bd = ctx->bd;
        p.x = x + off; p.y = y + off; p.z = z + off;
        p.lam = lam + off; p.ldlam = M;
        p.count = cnt;
        p.delta_abs = k.delta_abs;
        p.part = ctx->part; p.cap = cap;
        prof_mark(ctx, st);
        CU(k.analytic ? launch_interact_analytic(p, ctx->sm_count, st) : launch_interact_stencil(p, ctx->sm_count, st));
        prof_mark(ctx, st);
        CU(launch_residual_finalize(ctx->bd, k, cnt, M, z + off, ctx->part, cap, out + off, phi ? phi + off : nullptr, st));
        launches += 2;
    }
    ctx->last_interactions = (double)M * (k.analytic ? 1 : kStencil) * (double)ctx->bd.N;
    ctx->last_launches = launches;
    ctx->last_evals = M;
    ctx->evals_on_device = 0;
    ctx->pass_trace_valid = false;
    return DBIE_OK;
}

static size_t align256(size_t v) { return (v + 255) & ~(size_t)255; }

// GRID mode (O-4; BASELINE.json config 5 reading, not in the paper): per level one
// MODE_GRID interaction launch (4 x 3 x T sums per active point) and one grid_step launch.
static dbie_status solve_grid(dbie_ctx* ctx, long long M, const double* x, const double* y, const double* z,
                              const dbie_solve_opts* opts, const NMConsts& k, double* B, double* lam, double* resid,
                              int* iters, int* status, void* cuda_stream) {
    ctx->pass_trace_valid = false;
    const int T = opts->n_trial, L = opts->n_level;
    // T < 4: the refined window 2W/(T-1) would not shrink (T = 3) or would grow (T = 2)
    if (T < 4 || T > kGridMaxTrials || L < 1 || !(opts->lam_max > 0.0) || !isfinite(opts->lam_max)) return DBIE_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const BoundaryView& bd = ctx->bd;
    // batch so that the chunk sums (nchunks x 12 T doubles per point) stay below 2 GiB
    const size_t per_point = (size_t)bd.nchunks * 12 * T * sizeof(double);
    long long batch = (long long)(((size_t)2 << 30) / per_point);
    if (batch < 1024) batch = 1024;
    if (ctx->batch_limit > 0) batch = ctx->batch_limit;
    const long long cap = M < batch ? M : batch;
    dbie_status s = ensure(ctx, (void**)&ctx->part, &ctx->part_bytes, per_point * cap);
    if (s != DBIE_OK) return s;
    const size_t isz = align256((size_t)cap * sizeof(int));
    const size_t dstride = (size_t)cap * sizeof(double);
    s = ensure(ctx, (void**)&ctx->state, &ctx->state_bytes, 3 * align256(12 * dstride) + 2 * isz);
    if (s != DBIE_OK) return s;
    GridArrays a;
    char* base = ctx->state;
    a.lo = (double*)base;                base += align256(3 * dstride);
    a.inc = (double*)base;               base += align256(12 * dstride);
    a.il = (double*)base;                base += align256(3 * dstride);
    a.act[0] = (int*)base;               base += isz;
    a.act[1] = (int*)base;               base += isz;
    a.cap = cap;
    a.nact = ctx->counters;
    unsigned long long* nevals = (unsigned long long*)((char*)ctx->counters + 16);
    CU(cudaMemsetAsync(ctx->counters, 0, kCounterBytes, st));
    GridConsts gc;
    gc.T = T;
    gc.n_level = L;
    gc.Lmax = opts->lam_max / bd.h;
    long long launches = 0;
    prof_reset(ctx);
    for (long long off = 0; off < M; off += cap) {
        const long long cnt = (M - off < cap) ? (M - off) : cap;
        CU(cudaMemsetAsync(ctx->counters, 0, 8, st));        // list counters
        CU(cudaMemsetAsync(ctx->counters + 8, 0, 8, st));    // work-item counters
        CU(launch_grid_init(a, cnt, M, x + off, y + off, z + off, B + off, lam + off, resid + off, iters + off,
                            status + off, st));
        ++launches;
        double W = gc.Lmax;
        for (int lev = 0; lev < L; ++lev) {
            gc.W = W;
            gc.Wn = 2.0 * W / (double)(T - 1);
            InteractParams p;
            memset(&p, 0, sizeof p);
            p.bd = bd;
            p.x = x + off; p.y = y + off; p.z = z + off;
            p.act = a.act[lev & 1];
            p.count_ptr = &a.nact[lev & 1];
            p.zero_ptr = &a.nact[(lev + 1) & 1];
            p.work_ctr = ctx->counters + 8 + (lev & 1);
            p.zero_work = ctx->counters + 8 + ((lev + 1) & 1);
            p.delta_abs = k.delta_abs;
            p.part = ctx->part; p.cap = cap;
            p.lo = a.lo; p.ldlo = cap; p.W = W; p.T = T; p.dlam = W / (double)(T - 1);
            prof_mark(ctx, st);
            CU(k.analytic ? launch_interact_grid_analytic(p, ctx->sm_count, st) : launch_interact_grid(p, ctx->sm_count, st));
            prof_mark(ctx, st);
            CU(launch_grid_step(a, k, gc, bd, lev, cnt, M, z + off, ctx->part, cap, B + off, lam + off, resid + off,
                                iters + off, status + off, nevals, st));
            launches += 2;
            W = gc.Wn;
        }
    }
    ctx->last_launches = launches;
    ctx->evals_on_device = 1;
    ctx->positions_per_eval = k.analytic ? 1 : kStencil;
    return DBIE_OK;
}

extern "C" dbie_status dbie_solve(dbie_ctx* ctx, long long M, const double* x, const double* y, const double* z,
                                  const dbie_solve_opts* opts, double* B, double* lam, double* resid, int* iters,
                                  int* status, void* cuda_stream) {
    if (!ctx || M < 0) return DBIE_EINVAL;
    if (M == 0) return DBIE_OK;
    if (!x || !y || !z || !B || !lam || !resid || !iters || !status) return DBIE_EINVAL;
    if (M > 0x7fffffffLL) return DBIE_EINVAL;
    GUARD_DEVICE();
    NvtxRange nvtx_("dbie_solve");
    NMConsts k;
    dbie_status s = make_consts(ctx, opts, &k);
    if (s != DBIE_OK) return s;
    if (opts && opts->method == 1) return solve_grid(ctx, M, x, y, z, opts, k, B, lam, resid, iters, status, cuda_stream);
    if (opts && opts->method != 0) return DBIE_EINVAL;
    ctx->pass_trace_valid = false;
    if (!ctx->coop_launch) {
        snprintf(ctx->err, 256, "dbie_solve: the Nelder-Mead search is one cooperative launch and this device does not "
                 "support cooperative launches (cudaDevAttrCooperativeLaunch = 0); method = 1 (GRID) does not need them");
        return DBIE_ESTATE;
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const long long cap = M < stencil_batch(ctx) ? M : stencil_batch(ctx);
    s = ensure(ctx, (void**)&ctx->part, &ctx->part_bytes, (size_t)ctx->bd.nchunks * 12 * cap * sizeof(double));
    if (s != DBIE_OK) return s;
    // state layout: 48 doubles + 4 ints per point (structure-of-arrays, rows of `count` points of the current
    // batch, count <= cap) + the arrival counters of the fused kernel
    const size_t isz = align256((size_t)cap * sizeof(int));
    const size_t dsz = align256(((size_t)cap / 4 + 2) * sizeof(unsigned));
    s = ensure(ctx, (void**)&ctx->state, &ctx->state_bytes, 48 * (size_t)cap * sizeof(double) + 5 * 256 + 4 * isz + dsz);
    if (s != DBIE_OK) return s;
    SolveArrays a;
    char* base = ctx->state;
    const size_t dstride = (size_t)cap * sizeof(double);
    a.V = (double*)base;                 base += align256(12 * dstride);
    a.F = (double*)base;                 base += align256(4 * dstride);
    a.aux = (double*)base;               base += align256(20 * dstride);
    a.pend = (double*)base;              base += align256(9 * dstride);
    a.cand = (double*)base;              base += align256(3 * dstride);
    a.phase = (int*)base;                base += isz;
    a.iters = (int*)base;                base += isz;
    a.act[0] = (int*)base;               base += isz;
    a.act[1] = (int*)base;               base += isz;
    unsigned* done = (unsigned*)base;
    a.nact = ctx->counters;
    unsigned long long* nevals = (unsigned long long*)((char*)ctx->counters + 16);
    CU(cudaMemsetAsync(ctx->counters, 0, kCounterBytes, st));
    CU(cudaMemsetAsync(done, 0, dsz, st));
    long long launches = 0;
    prof_reset(ctx);
    for (long long off = 0; off < M; off += cap) {
        const long long cnt = (M - off < cap) ? (M - off) : cap;
        CU(cudaMemsetAsync(ctx->counters, 0, 16, st));        // list counters (three rotating slots)
        CU(cudaMemsetAsync(ctx->counters + 8, 0, 16, st));    // work-item counters
        CU(launch_solve_init(a, k, cnt, M, x + off, y + off, z + off, B + off, lam + off, resid + off,
                             iters + off, status + off, st));
        ++launches;
        // One cooperative launch runs every pass of the search (dbie_solve_fused.cu): no per-pass host work,
        // no read-back, no partial-sum round trip for large batches.
        FusedParams f;
        memset(&f, 0, sizeof f);
        f.ip.bd = ctx->bd;
        f.ip.x = x + off; f.ip.y = y + off; f.ip.z = z + off;
        f.ip.lam = a.cand; f.ip.ldlam = cnt;
        f.ip.delta_abs = k.delta_abs;
        f.ip.part = ctx->part; f.ip.cap = cap;
        f.s = a;
        f.k = k;
        f.count = cnt; f.ldo = M;
        f.B = B + off; f.lam = lam + off; f.resid = resid + off;
        f.iters = iters + off; f.status = status + off;
        f.nevals = nevals;
        f.nact3 = ctx->counters;
        f.work3 = ctx->counters + 8;
        f.done = done;
        f.maxpass = 4 + 5 * k.maxiter + 1;   // 4 initial evaluations + at most 5 per iteration; maxiter <= kMaxIter, so no overflow
        if (ctx->profile) {   // diagnostic: (active points, time stamp) of every pass of this launch, the first kPassTraceMax of them
            const int need = (f.maxpass < kPassTraceMax ? f.maxpass : kPassTraceMax) + 1;
            if (ctx->pass_trace_cap < need) {
                if (ctx->pass_trace) CU(cudaFree(ctx->pass_trace));
                ctx->pass_trace = nullptr; ctx->pass_trace_cap = 0;
                CU(cudaMalloc(&ctx->pass_trace, sizeof(unsigned long long) * 2 * need));
                ctx->pass_trace_cap = need;
            }
            CU(cudaMemsetAsync(ctx->pass_trace, 0, sizeof(unsigned long long) * 2 * need, st));
            f.trace = ctx->pass_trace; f.trace_cap = need;
            ctx->pass_trace_valid = true;
        }
        prof_mark(ctx, st);
        int nl = 0;
        CU(launch_solve_nm_fused(f, ctx->sm_count, &nl, st));
        prof_mark(ctx, st);
        launches += nl;
    }
    ctx->last_launches = launches;
    ctx->evals_on_device = 1;
    ctx->positions_per_eval = k.analytic ? 1 : kStencil;
    return DBIE_OK;
}

extern "C" dbie_status dbie_solve_host(dbie_ctx* ctx, long long M, const double* x, const double* y,
                                       const double* z, const dbie_solve_opts* opts, double* B, double* lam,
                                       double* resid, int* iters, int* status) {
    if (!ctx || M < 0) return DBIE_EINVAL;
    if (M == 0) return DBIE_OK;
    if (!x || !y || !z || !B || !lam || !resid || !iters || !status) return DBIE_EINVAL;
    GUARD_DEVICE();
    const size_t m = (size_t)M * sizeof(double);
    CU(cudaDeviceSynchronize());   // earlier work on this context may be in flight on another stream
    dbie_status s = io_reserve(ctx, 11 * m + 2 * align256((size_t)M * sizeof(int)) + 512);
    if (s != DBIE_OK) return s;
    double* d = (double*)ctx->io;   // x, y, z, B[3], lam[3], resid[2], iters, status
    int* di = (int*)(ctx->io + align256(11 * m));
    int* ds = (int*)((char*)di + align256((size_t)M * sizeof(int)));
    cudaStream_t st = ctx->own_stream;
    CU(cudaMemcpyAsync(d, x, m, cudaMemcpyHostToDevice, st));
    CU(cudaMemcpyAsync(d + M, y, m, cudaMemcpyHostToDevice, st));
    CU(cudaMemcpyAsync(d + 2 * M, z, m, cudaMemcpyHostToDevice, st));
    s = dbie_solve(ctx, M, d, d + M, d + 2 * M, opts, d + 3 * M, d + 6 * M, d + 9 * M, di, ds, st);
    if (s != DBIE_OK) return s;
    CU(cudaMemcpyAsync(B, d + 3 * M, 3 * m, cudaMemcpyDeviceToHost, st));
    CU(cudaMemcpyAsync(lam, d + 6 * M, 3 * m, cudaMemcpyDeviceToHost, st));
    CU(cudaMemcpyAsync(resid, d + 9 * M, 2 * m, cudaMemcpyDeviceToHost, st));
    CU(cudaMemcpyAsync(iters, di, (size_t)M * sizeof(int), cudaMemcpyDeviceToHost, st));
    CU(cudaMemcpyAsync(status, ds, (size_t)M * sizeof(int), cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    return DBIE_OK;
}

// ------------------------------------------------------------------------------ trace -----
extern "C" void dbie_trace_default_opts(dbie_trace_opts* o) {
    if (!o) return;
    memset(o, 0, sizeof *o);
    o->ds = 0.5;
    o->max_steps = 100;
    o->direction = 1;
    o->current = 0;
    o->fixed_lambda = 0;
    o->z_min = 0.0;
    o->z_max = 1e300;
}

extern "C" dbie_status dbie_trace(dbie_ctx* ctx, long long L, const double* x0, const double* y0, const double* z0,
                                  const dbie_solve_opts* sopts, const dbie_trace_opts* topts, double* path, int* npts,
                                  int* status, void* cuda_stream) {
    if (!ctx || L < 0) return DBIE_EINVAL;
    if (L == 0) return DBIE_OK;
    if (!x0 || !y0 || !z0 || !path || !npts || !status || L > 0x7fffffffLL) return DBIE_EINVAL;
    dbie_trace_opts td;
    if (!topts) { dbie_trace_default_opts(&td); topts = &td; }
    if (!(topts->ds > 0.0) || !isfinite(topts->ds) || topts->max_steps < 0 || (topts->direction != 1 && topts->direction != -1) ||
        !(topts->z_max > topts->z_min))
        return DBIE_EINVAL;
    if (topts->fixed_lambda && !(isfinite(topts->lam[0]) && isfinite(topts->lam[1]) && isfinite(topts->lam[2]))) return DBIE_EINVAL;
    GUARD_DEVICE();
    NvtxRange nvtx_("dbie_trace");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const BoundaryView& bd = ctx->bd;
    const double h = bd.h;
    // layout of the scratch: r[3], k[12], px, py, pz, B[3], lam[3], resid[2], out9[9] doubles; 5 ints per line
    const size_t dl = (size_t)L * sizeof(double), il = align256((size_t)L * sizeof(int));
    dbie_status s = ensure(ctx, (void**)&ctx->trace, &ctx->trace_bytes, align256(35 * dl) + 5 * il);
    if (s != DBIE_OK) return s;
    double* d = (double*)ctx->trace;
    TraceState t;
    t.r = d;               d += 3 * L;
    t.k = d;               d += 12 * L;
    t.px = d;              d += L;
    t.py = d;              d += L;
    t.pz = d;              d += L;
    double* fB = d;        d += 3 * L;
    double* flam = d;      d += 3 * L;
    double* fres = d;      d += 2 * L;
    double* fout = d;      d += 9 * L;
    char* ib = ctx->trace + align256(35 * dl);
    t.alive = (int*)ib;    ib += il;
    t.good = (int*)ib;     ib += il;
    t.why = (int*)ib;      ib += il;
    int* fit = (int*)ib;   ib += il;
    int* fst = (int*)ib;
    TraceBox box;
    // the region written as the oracle writes it: x0 + nx h etc. (nx, ny of the magnetogram, not of a 9-node source grid)
    box.x0 = bd.x0; box.x1 = bd.x0 + (double)ctx->win_nx * h;
    box.y0 = bd.y0; box.y1 = bd.y0 + (double)ctx->win_ny * h;
    box.z0 = topts->z_min * h; box.z1 = topts->z_max * h;
    const double ds = topts->ds * h;
    const int S = topts->max_steps;
    CU(launch_trace_init(t, box, L, S, x0, y0, z0, path, npts, status, st));
    if (topts->fixed_lambda) CU(launch_trace_fill_lambda(flam, L, topts->lam, st));
    double interactions = 0.0;
    long long launches = 1, evals = 0;
    for (int step = 0; step < S; ++step)
        for (int stage = 0; stage < 4; ++stage) {
            const double* v = fB;
            if (!topts->fixed_lambda) {
                s = dbie_solve(ctx, L, t.px, t.py, t.pz, sopts, fB, flam, fres, fit, fst, st);
                if (s != DBIE_OK) return s;
                launches += ctx->last_launches;
            } else if (!topts->current) {
                s = dbie_eval(ctx, L, t.px, t.py, t.pz, flam, fB, st);
                if (s != DBIE_OK) return s;
                launches += ctx->last_launches;
                interactions += ctx->last_interactions;
            }
            if (topts->current) {
                s = dbie_residual(ctx, L, t.px, t.py, t.pz, flam, sopts, fout, nullptr, st);
                if (s != DBIE_OK) return s;
                launches += ctx->last_launches;
                interactions += ctx->last_interactions;
                evals += L;
                v = fout + 5 * L;   // rows 5..7 of dbie_residual's output: J (Eq. 14)
            }
            CU(launch_trace_stage(t, box, L, S, step, stage, topts->direction, ds, v, L, path, npts, status, st));
            ++launches;
        }
    // counters: the interactions of the lambda searches live on the device (they are not summed over the calls)
    ctx->last_interactions = interactions;
    ctx->last_launches = launches;
    ctx->last_evals = evals;
    ctx->evals_on_device = 0;
    return DBIE_OK;
}

extern "C" dbie_status dbie_last_counters(dbie_ctx* ctx, double* interactions, long long* launches,
                                          long long* objective_evals) {
    if (!ctx) return DBIE_EINVAL;
    GUARD_DEVICE();
    if (ctx->evals_on_device) {
        unsigned long long n = 0;
        CU(cudaMemcpy(&n, (char*)ctx->counters + 16, sizeof n, cudaMemcpyDeviceToHost));
        ctx->last_evals = (long long)n;
        ctx->last_interactions = (double)n * ctx->positions_per_eval * (double)ctx->bd.N;
    }
    if (interactions) *interactions = ctx->last_interactions;
    if (launches) *launches = ctx->last_launches;
    if (objective_evals) *objective_evals = ctx->last_evals;
    return DBIE_OK;
}

extern "C" dbie_status dbie_probe_fp64_operands(double millis, double* rates) {
    dbie_ctx* ctx = nullptr;
    if (!(millis > 0.0) || !rates) return DBIE_EINVAL;
    int dev = 0, sms = 0;
    CU(cudaGetDevice(&dev));
    CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    CU(launch_operand_probe(millis, sms, rates));
    return DBIE_OK;
}

extern "C" dbie_status dbie_probe_dfma_rate(double millis, double* dfma_per_s, double* ffma_per_s) {
    dbie_ctx* ctx = nullptr;
    if (!(millis > 0.0)) return DBIE_EINVAL;
    int dev = 0, sms = 0;
    CU(cudaGetDevice(&dev));
    CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    CU(launch_probe(millis, sms, dfma_per_s, ffma_per_s));
    return DBIE_OK;
}
