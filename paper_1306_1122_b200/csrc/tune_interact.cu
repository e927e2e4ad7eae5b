// tune_interact.cu — shape sweep of the fp64 interaction kernel and an issue-slot probe of the FP64 pipe.
// A developer tool that sits beside the kernel it tunes: `python -m paper_1306_1122_b200.build --tune`
// builds paper_1306_1122_b200/dbie_tune; `dbie_tune [nx] [M]` prints one line per variant
// (threads x CTAs/SM, pixels in flight, trial triples per thread; one CTA per work item or a
// persistent grid) with its time, interactions/s and fraction of 148 x 64 x 1.965e9 FP64 lanes/s,
// then the DFMA rate with k integer-pipe instructions interleaved per DFMA.  The shapes the
// library launches (dbie_interact.cu) are the winners of this sweep; profiles/r01_variants.md
// holds its round-1 output.  Nothing in the library or the tests depends on this file.
#include <cstdio>
#include <cstdlib>
#include <vector>
#include <cmath>
#include "dbie_interact_fp64.cuh"
using namespace dbie;

static void setup_tiling(BoundaryView& b) {
    if (b.nx <= kTilePx) {
        b.tile_rows = kTilePx / b.nx; if (b.tile_rows < 1) b.tile_rows = 1;
        b.segs_per_row = 1; b.seg_w = b.nx;
        b.ntiles = (b.ny + b.tile_rows - 1) / b.tile_rows;
    } else {
        b.tile_rows = 1; b.segs_per_row = (b.nx + kTilePx - 1) / kTilePx;
        b.seg_w = (b.nx + b.segs_per_row - 1) / b.segs_per_row; b.seg_w += b.seg_w & 1;
        b.ntiles = b.ny * b.segs_per_row;
    }
    b.nchunks = b.ntiles < kMaxChunks ? b.ntiles : kMaxChunks;
}
static unsigned* g_work = nullptr;
static double urand() { return rand() / (double)RAND_MAX; }

template <int MODE, int NT, int TH, int MB, int U>
static void run_new(const char* name, InteractParams p, int sms, int waves_target, int persistent, double inter) {
    // persistent: 0 = one CTA per work item, 1 = persistent grid with static striding, 2 = persistent grid
    // taking items from an atomic counter (what the library does when the slot count lives on the device)
    const int G = (MODE == MODE_GRID) ? p.T / NT : 1;
    const long long nitems = p.count * items_per_slot(MODE, G);
    const long long nblk = (nitems + TH - 1) / TH;
    p.target_items = waves_target * sms * MB;
    long long nsplit = 1;
    if (nblk < p.target_items) { nsplit = (p.target_items + nblk - 1) / nblk; if (nsplit > p.bd.nchunks) nsplit = p.bd.nchunks; }
    long long grid = persistent ? (long long)sms * MB : nblk * nsplit;
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    float best = 1e30f;
    for (int rep = 0; rep < 3; ++rep) {
        cudaMemset(p.part, 0, 64);
        if (persistent == 2) { cudaMemset(g_work, 0, 8); p.work_ctr = g_work; }
        cudaEventRecord(e0);
        interact64_kernel<MODE, NT, TH, MB, U><<<(unsigned)grid, TH>>>(p);
        cudaEventRecord(e1); cudaEventSynchronize(e1);
        float ms; cudaEventElapsedTime(&ms, e0, e1); if (rep > 0 && ms < best) best = ms;
    }
    cudaError_t e = cudaGetLastError();
    std::vector<double> h(3); cudaMemcpy(h.data(), p.part, 24, cudaMemcpyDeviceToHost);
    printf("%-50s grid %6lld nsplit %2lld  %9.3f ms  %.4e int/s  frac76 %.3f  chk %.15e %s\n", name, grid, nsplit, best,
           inter / (best * 1e-3), inter / (best * 1e-3) * 76 / (148 * 64 * 1.965e9), h[0], e == cudaSuccess ? "" : cudaGetErrorString(e));
}

// ---- issue-slot probe: 8 independent DFMA chains per thread with k integer-pipe instructions per DFMA
__constant__ double kc[4] = {0.999999, 1e-7, 1.000001, -1e-7};
// MODE: 0 pure DFMA reg operands; 1 DFMA with const-bank operands; 2 DFMA + 1 LOP3 per DFMA; 3 DFMA + 1 LOP3 per 2 DFMA;
// 4 DFMA + FSEL per DFMA ; 5 DMUL only; 6 DADD only; 7 DFMA + IMAD per DFMA; 8: DFMA + 2 LOP3 per DFMA
template <int MODE>
__global__ void __launch_bounds__(256) pipe_probe(int iters, double seed, double* sink, int iseed) {
    double a[8];
    unsigned b[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) { a[i] = seed + threadIdx.x + i; b[i] = iseed + threadIdx.x * 7 + i; }
    const double m = seed * 0.999999, c = seed * 1e-7;
    for (int k = 0; k < iters; ++k) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                if (MODE == 1) a[i] = fma(a[i], kc[0], kc[1]);
                else if (MODE == 5) a[i] = a[i] * m;
                else if (MODE == 6) a[i] = a[i] + c;
                else a[i] = fma(a[i], m, c);
                if (MODE == 2 || MODE == 8) b[i] = (b[i] ^ (b[(i + 1) & 7] & 0x55555555u)) ;
                if (MODE == 8) b[i] = (b[i] | (b[(i + 3) & 7] & 0x33333333u)) ^ 0x1234567u;
                if (MODE == 3 && (i & 1)) b[i] = (b[i] ^ (b[(i + 1) & 7] & 0x55555555u));
                if (MODE == 4) b[i] = (b[(i+1)&7] > 77u) ? b[i] + 0u : b[(i + 2) & 7];
                if (MODE == 7) b[i] = b[i] * 3u + b[(i + 1) & 7];
            }
        }
    }
    double s = 0; unsigned t = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) { s += a[i]; t ^= b[i]; }
    if (s == -1.2345 || t == 0x7fffffff) sink[0] = s + t;
}
template <int MODE> static void run_probe(const char* name) {
    double* sink; cudaMalloc(&sink, 8);
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int grid = 148 * 8, iters = 20000;
    pipe_probe<MODE><<<grid, 256>>>(100, 1.0, sink, 1);
    cudaEventRecord(e0);
    pipe_probe<MODE><<<grid, 256>>>(iters, 1.0, sink, 1);
    cudaEventRecord(e1); cudaEventSynchronize(e1);
    float ms; cudaEventElapsedTime(&ms, e0, e1);
    double rate = (double)grid * 256 * 64.0 * iters / (ms * 1e-3);
    printf("%-40s %8.3f ms  %.4e fp64-instr/s  (%.3f of 148*64*1.965e9)\n", name, ms, rate, rate / (148 * 64 * 1.965e9));
}

int main(int argc, char** argv) {
    int nx = argc > 1 ? atoi(argv[1]) : 512, ny = nx;
    long long M = argc > 2 ? atoll(argv[2]) : 148 * 2048;
    int sms = 148;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, 0);
    const long long N = (long long)nx * ny;
    std::vector<double> bx(N), by(N), bz(N), x(M), y(M), z(M), lam(3 * M), lo(3 * M);
    srand(1);
    for (long long k = 0; k < N; ++k) { bx[k] = urand() - .5; by[k] = urand() - .5; bz[k] = urand() - .5; }
    for (long long i = 0; i < M; ++i) { x[i] = urand() * nx; y[i] = urand() * ny; z[i] = 1 + urand() * nx / 2;
        for (int c = 0; c < 3; ++c) { lam[c * M + i] = 0.4 * urand() - 0.2; lo[c * M + i] = 0.1 * urand(); } }
    double *dbx, *dby, *dbz, *dx, *dy, *dz, *dlam, *dlo, *dyk, *part; double4* rec;
    cudaMalloc(&dbx, N * 8); cudaMalloc(&dby, N * 8); cudaMalloc(&dbz, N * 8); cudaMalloc(&rec, N * 32); cudaMalloc(&dyk, ny * 8);
    cudaMalloc(&dx, M * 8); cudaMalloc(&dy, M * 8); cudaMalloc(&dz, M * 8); cudaMalloc(&dlam, 3 * M * 8); cudaMalloc(&dlo, 3 * M * 8);
    cudaMemcpy(dbx, bx.data(), N * 8, cudaMemcpyHostToDevice); cudaMemcpy(dby, by.data(), N * 8, cudaMemcpyHostToDevice);
    cudaMemcpy(dbz, bz.data(), N * 8, cudaMemcpyHostToDevice);
    cudaMemcpy(dx, x.data(), M * 8, cudaMemcpyHostToDevice); cudaMemcpy(dy, y.data(), M * 8, cudaMemcpyHostToDevice);
    cudaMemcpy(dz, z.data(), M * 8, cudaMemcpyHostToDevice); cudaMemcpy(dlam, lam.data(), 3 * M * 8, cudaMemcpyHostToDevice);
    cudaMemcpy(dlo, lo.data(), 3 * M * 8, cudaMemcpyHostToDevice);
    const int T = 8;
    cudaMalloc(&g_work, 8);
    cudaMalloc(&part, (size_t)kMaxChunks * 12 * T * M * 8);
    {   // stage rec[k] = {x_k, Bx0, By0, Bz0} and yk[] on the host (the library does this in stage_boundary_kernel)
        std::vector<double> hrec(4 * N), hyk(ny);
        for (long long k = 0; k < N; ++k) {
            hrec[4 * k] = 0.0 + ((double)(k % nx) + 0.5) * 1.0;
            hrec[4 * k + 1] = bx[k]; hrec[4 * k + 2] = by[k]; hrec[4 * k + 3] = bz[k];
        }
        for (int j = 0; j < ny; ++j) hyk[j] = 0.0 + ((double)j + 0.5) * 1.0;
        cudaMemcpy(rec, hrec.data(), N * 32, cudaMemcpyHostToDevice);
        cudaMemcpy(dyk, hyk.data(), ny * 8, cudaMemcpyHostToDevice);
    }
    InteractParams p; memset(&p, 0, sizeof p);
    p.bd.nx = nx; p.bd.ny = ny; p.bd.N = N; p.bd.h = 1; p.bd.x0 = 0; p.bd.y0 = 0; p.bd.rec = rec; p.bd.yk = dyk;
    setup_tiling(p.bd);
    p.x = dx; p.y = dy; p.z = dz; p.lam = dlam; p.ldlam = M; p.count = M; p.part = part; p.cap = M; p.delta_abs = 1e-3;
    p.lo = dlo; p.ldlo = M; p.W = 0.05; p.T = T; p.dlam = p.W / (T - 1);
    printf("nx %d M %lld ntiles %d nchunks %d\n", nx, M, p.bd.ntiles, p.bd.nchunks);
    const double ie = (double)M * N, is = 4.0 * M * N, ig = 4.0 * T * M * N;
    run_new<0, 1, 256, 2, 2>("eval   NT1 256x2 u2  [library]", p, sms, 8, 0, ie);
    run_new<0, 1, 256, 2, 1>("eval   NT1 256x2 u1", p, sms, 8, 0, ie);
    run_new<0, 1, 256, 2, 4>("eval   NT1 256x2 u4", p, sms, 8, 0, ie);
    run_new<0, 1, 256, 3, 1>("eval   NT1 256x3 u1", p, sms, 8, 0, ie);
    run_new<0, 1, 256, 4, 1>("eval   NT1 256x4 u1", p, sms, 8, 0, ie);
    run_new<0, 1, 128, 4, 2>("eval   NT1 128x4 u2", p, sms, 8, 0, ie);
    run_new<0, 1, 512, 1, 2>("eval   NT1 512x1 u2", p, sms, 8, 0, ie);
    run_new<0, 1, 128, 2, 2>("eval   NT1 128x2 u2", p, sms, 8, 0, ie);
    run_new<0, 1, 128, 2, 4>("eval   NT1 128x2 u4", p, sms, 8, 0, ie);
    run_new<0, 1, 128, 3, 4>("eval   NT1 128x3 u4", p, sms, 8, 0, ie);
    run_new<0, 1, 256, 1, 4>("eval   NT1 256x1 u4", p, sms, 8, 0, ie);
    run_new<0, 1, 128, 2, 8>("eval   NT1 128x2 u8", p, sms, 8, 0, ie);
    run_new<0, 1, 128, 2, 6>("eval   NT1 128x2 u6", p, sms, 8, 0, ie);
    run_new<0, 1, 64, 4, 8>("eval   NT1 64x4 u8", p, sms, 8, 0, ie);
    { InteractParams q = p; q.count = M / 4;
      run_new<1, 1, 256, 2, 2>("stencil NT1 256x2 u2 persistent dynamic [library]", q, sms, 16, 2, is / 4);
      run_new<1, 1, 256, 2, 2>("stencil NT1 256x2 u2 persistent static", q, sms, 16, 1, is / 4);
      run_new<1, 1, 256, 2, 2>("stencil NT1 256x2 u2 one CTA per item", q, sms, 16, 0, is / 4);
      run_new<1, 1, 256, 4, 1>("stencil NT1 256x4 u1 one CTA per item", q, sms, 16, 0, is / 4);
      // 4 stencil positions per thread, small-angle rotation between them (61.25 FP64 instr. per interaction)
      run_new<5, 1, 128, 2, 1>("stencil4 128x2 u1 persistent dynamic", q, sms, 16, 2, is / 4);
      run_new<5, 1, 128, 2, 1>("stencil4 128x2 u1", q, sms, 16, 0, is / 4);
      run_new<5, 1, 128, 3, 1>("stencil4 128x3 u1", q, sms, 16, 0, is / 4);
      run_new<5, 1, 256, 1, 1>("stencil4 256x1 u1", q, sms, 16, 0, is / 4);
      run_new<5, 1, 64, 4, 1>("stencil4 64x4 u1", q, sms, 16, 0, is / 4);
      run_new<5, 1, 128, 2, 2>("stencil4 128x2 u2", q, sms, 16, 0, is / 4);
      run_new<5, 1, 128, 2, 2>("stencil4 128x2 u2 persistent dynamic [library]", q, sms, 16, 2, is / 4);
      run_new<5, 1, 128, 2, 3>("stencil4 128x2 u3", q, sms, 16, 0, is / 4);
      run_new<5, 1, 128, 2, 4>("stencil4 128x2 u4", q, sms, 16, 0, is / 4);
      run_new<5, 1, 256, 1, 2>("stencil4 256x1 u2", q, sms, 16, 0, is / 4);
      run_new<5, 1, 64, 4, 2>("stencil4 64x4 u2", q, sms, 16, 0, is / 4);
      run_new<5, 1, 128, 3, 2>("stencil4 128x3 u2", q, sms, 16, 0, is / 4); }
    { InteractParams q = p;   // analytic gradient: 95 FP64 instructions per interaction (frac76 x 95/76 = pipe utilisation)
      run_new<3, 1, 256, 2, 1>("analytic NT1 256x2 u1 persistent dynamic [library]", q, sms, 16, 2, ie);
      run_new<3, 1, 256, 2, 1>("analytic NT1 256x2 u1", q, sms, 16, 0, ie);
      run_new<3, 1, 256, 2, 2>("analytic NT1 256x2 u2", q, sms, 16, 0, ie);
      run_new<3, 1, 128, 4, 2>("analytic NT1 128x4 u2", q, sms, 16, 0, ie);
      run_new<3, 1, 128, 2, 2>("analytic NT1 128x2 u2", q, sms, 16, 0, ie);
      run_new<3, 1, 128, 2, 4>("analytic NT1 128x2 u4", q, sms, 16, 0, ie);
      run_new<3, 1, 256, 1, 4>("analytic NT1 256x1 u4", q, sms, 16, 0, ie); }
    { InteractParams q = p; q.count = M / 8;   // GRID on the analytic gradient (88 instr. per interaction at NT2)
      const double iga = (double)T * (M / 8) * N;
      run_new<4, 2, 128, 3, 1>("grid-analytic NT2 128x3 u1 [library]", q, sms, 16, 0, iga);
      run_new<4, 2, 128, 2, 1>("grid-analytic NT2 128x2 u1", q, sms, 16, 0, iga);
      run_new<4, 2, 128, 2, 2>("grid-analytic NT2 128x2 u2", q, sms, 16, 0, iga);
      run_new<4, 1, 256, 2, 2>("grid-analytic NT1 256x2 u2", q, sms, 16, 0, iga); }
    { InteractParams q = p; q.count = M / 32;
      run_new<2, 4, 256, 2, 1>("grid   NT4 256x2 u1 persistent dynamic [library]", q, sms, 16, 2, ig / 32);
      run_new<2, 4, 256, 2, 1>("grid   NT4 256x2 u1 persistent static", q, sms, 16, 1, ig / 32);
      run_new<2, 4, 256, 2, 1>("grid   NT4 256x2 u1", q, sms, 16, 0, ig / 32);
      run_new<2, 2, 256, 2, 2>("grid   NT2 256x2 u2", q, sms, 16, 0, ig / 32);
      run_new<2, 1, 256, 2, 2>("grid   NT1 256x2 u2", q, sms, 16, 0, ig / 32);
      run_new<2, 4, 128, 3, 2>("grid   NT4 128x3 u2", q, sms, 16, 0, ig / 32);
      run_new<2, 8, 128, 2, 1>("grid   NT8 128x2 u1", q, sms, 16, 0, ig / 32);
      run_new<2, 8, 128, 3, 1>("grid   NT8 128x3 u1", q, sms, 16, 0, ig / 32);
      run_new<2, 8, 256, 1, 1>("grid   NT8 256x1 u1", q, sms, 16, 0, ig / 32);
      run_new<2, 8, 256, 2, 1>("grid   NT8 256x2 u1", q, sms, 16, 0, ig / 32); }
    printf("FP64 pipe, 8 DFMA chains per thread, k integer-pipe instructions per DFMA:\n");
    run_probe<0>("DFMA only");
    run_probe<5>("DMUL only");
    run_probe<6>("DADD only");
    run_probe<3>("DFMA + 0.5 LOP3");
    run_probe<2>("DFMA + 1 LOP3");
    run_probe<4>("DFMA + 1 SEL + 1 ISETP");
    run_probe<8>("DFMA + 3 LOP3");
    run_probe<7>("DFMA + 1 IMAD (FMA pipe)");
    return 0;
}
