/*
 * blip_harness.c — a plain-C caller of libblipgpu.so (include/blipgpu.h), no Python anywhere.
 *
 *   blip_harness latency [calls]   per-call latency of blipgpu_eval at M = 1 ... 1,536 on a table
 *                                  of the TiO2-sized shape (64x64x40 grid, 768 orbitals), as a
 *                                  CASINO-like particle-by-particle caller would see it
 *                                  (PAPER.md:268 kernel (1) "GPU/PbP"; BASELINE.json configs[3]).
 *                                  Every call evaluates different positions (a pool that touches
 *                                  far more table rows than the L2 holds), so the rows come from
 *                                  HBM, not from a cache warmed by the previous call.  One JSON
 *                                  line on stdout.
 *   blip_harness fullsize          the TiO2-sized launch configuration (49,152 x 768, staged kernel)
 *                                  three times through eval / eval_contract: for the checked build.
 *   blip_harness selftest [oracle] every kernel once on a small table (staged, tensor-core staged,
 *                                  direct, split, fp64, contraction; both modes): exit code 0 iff all
 *                                  calls return OK, the results are finite and the staged kernel
 *                                  returns the bits of the direct one; with the path of
 *                                  oracle/libblip_oracle.so as second argument (loaded with dlopen,
 *                                  never linked) also iff every kernel's val / grad / lap are within
 *                                  north_star's tolerances of the CPU fp64 oracle.  This is the program
 *                                  the compute-sanitizer runs of profiles/ are taken on.
 *
 * Table values and positions come from a 64-bit LCG: timing and memory safety do not depend
 * on them, and parity with the oracle is the business of tests/test_gpu_*.py, not of this file.
 */
#include <cuda_runtime_api.h>
#include <dlfcn.h>
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <time.h>

#include "blipgpu.h"
#include "blipgpu_dev.h"

static unsigned long long lcg_state = 0x9E3779B97F4A7C15ull;
static double lcg_uniform(void)
{
    lcg_state = lcg_state * 6364136223846793005ull + 1442695040888963407ull;
    return (double)(lcg_state >> 11) * (1.0 / 9007199254740992.0);
}

static double now_s(void)
{
    struct timespec ts;
    clock_gettime(CLOCK_MONOTONIC, &ts);
    return (double)ts.tv_sec + 1e-9 * (double)ts.tv_nsec;
}

#define CUDA_OK(call)                                                                    \
    do {                                                                                 \
        cudaError_t e_ = (call);                                                         \
        if (e_ != cudaSuccess) {                                                         \
            fprintf(stderr, "%s:%d: %s: %s\n", __FILE__, __LINE__, #call, cudaGetErrorString(e_)); \
            exit(2);                                                                     \
        }                                                                                \
    } while (0)
#define BLIP_OK(call)                                                                    \
    do {                                                                                 \
        int rc_ = (call);                                                                \
        if (rc_ != BLIPGPU_OK) {                                                         \
            fprintf(stderr, "%s:%d: %s: %s\n", __FILE__, __LINE__, #call, blipgpu_strerror(rc_)); \
            exit(3);                                                                     \
        }                                                                                \
    } while (0)

/* keep != NULL: the caller gets (and frees) the host copy of the table */
static blipgpu_table* make_table_keep(const double A[9], const int n[3], int L, float** keep)
{
    const size_t count = (size_t)n[0] * n[1] * n[2] * (size_t)L;
    float* c = (float*)malloc(count * sizeof(float));
    if (!c) { fprintf(stderr, "out of host memory\n"); exit(2); }
    for (size_t i = 0; i < count; ++i) c[i] = (float)(2.0 * lcg_uniform() - 1.0);
    blipgpu_table* t = NULL;
    BLIP_OK(blipgpu_create(A, n, L, c, 0, NULL, &t));
    if (keep) *keep = c; else free(c);
    return t;
}

static blipgpu_table* make_table(const double A[9], const int n[3], int L)
{
    return make_table_keep(A, n, L, NULL);
}

/* The CPU fp64 oracle (oracle/libblip_oracle.so; test infrastructure, never linked into the product or
 * into this program): `selftest <path to the library>` loads it at run time and checks every kernel's
 * outputs against it with north_star's tolerances; the other modes of this program never touch it. */
typedef int (*oracle_eval_fn)(const double*, const int*, int, const float*, const double*, long long, int,
                              double*, double*, double*, int*);
typedef int (*oracle_spacing_fn)(const double*, const int*, double*);

/* largest |gpu - oracle| of a call's outputs as a fraction of its tolerance (val, grad, lap: tol[0..2]);
 * h = [val nv | grad 3 nv | lap nv] with row pitch ld, the oracle's arrays are dense in L */
static double oracle_fraction(const float* h, size_t nv, long long Mp, int L, long long ld, int mode,
                              const double* oval, const double* ograd, const double* olap, const double tol[3])
{
    double worst = 0.0;
    for (long long j = 0; j < Mp; ++j)
        for (int l = 0; l < L; ++l) {
            double f = fabs((double)h[j * ld + l] - oval[j * L + l]) / tol[0];
            if (!(f <= worst)) worst = f;                    /* NaN counts as a failure */
            if (mode == 0) continue;
            for (int i = 0; i < 3; ++i) {
                f = fabs((double)h[nv + (3 * j + i) * ld + l] - ograd[(3 * j + i) * L + l]) / tol[1];
                if (!(f <= worst)) worst = f;
            }
            f = fabs((double)h[4 * nv + j * ld + l] - olap[j * L + l]) / tol[2];
            if (!(f <= worst)) worst = f;
        }
    return worst;
}

static double* make_positions(const double A[9], long long M, double spread)
{
    double* p = (double*)malloc(sizeof(double) * 3 * (size_t)M);
    for (long long j = 0; j < M; ++j) {
        double u[3];
        for (int a = 0; a < 3; ++a) u[a] = (lcg_uniform() - 0.5) * 2.0 * spread;
        for (int i = 0; i < 3; ++i) p[3 * j + i] = u[0] * A[i] + u[1] * A[3 + i] + u[2] * A[6 + i];
    }
    return p;
}

static int cmp_double(const void* a, const void* b)
{
    const double x = *(const double*)a, y = *(const double*)b;
    return (x > y) - (x < y);
}

/* ------------------------------------------------------------------------------------- */
static int run_latency(int calls)
{
    const double A[9] = {17.4, 0, 0, 0, 17.4, 0, 0, 0, 11.2};
    const int n[3] = {64, 64, 40};
    const int L = 768;
    const long long ld = 768;
    blipgpu_table* t = make_table(A, n, L);
    const long long pool = 1 << 18;                     /* 262,144 positions: every table row, many times */
    double* hpos = make_positions(A, pool, 0.5);
    double* dpos = NULL;
    float *val = NULL, *grad = NULL, *lap = NULL;
    const long long Mmax = 1536;
    CUDA_OK(cudaMalloc((void**)&dpos, sizeof(double) * 3 * (size_t)pool));
    CUDA_OK(cudaMemcpy(dpos, hpos, sizeof(double) * 3 * (size_t)pool, cudaMemcpyHostToDevice));
    CUDA_OK(cudaMalloc((void**)&val, sizeof(float) * (size_t)Mmax * ld));
    CUDA_OK(cudaMalloc((void**)&grad, sizeof(float) * 3 * (size_t)Mmax * ld));
    CUDA_OK(cudaMalloc((void**)&lap, sizeof(float) * (size_t)Mmax * ld));
    cudaStream_t s;
    CUDA_OK(cudaStreamCreate(&s));
    BLIP_OK(blipgpu_reserve(t, Mmax));
    const long long Ms[] = {1, 8, 32, 128, 512, 1536};
    double* lat = (double*)malloc(sizeof(double) * (size_t)calls);
    printf("{\"harness\": \"latency\", \"table\": \"64x64x40 x 768 (503 MB)\", \"calls\": %d, "
           "\"positions\": \"a different slice of a 262,144-position pool per call (rows from HBM, not a warm L2)\", "
           "\"rows\": [", calls);
    int first = 1;
    for (int mode = 0; mode <= 1; ++mode)
        for (size_t k = 0; k < sizeof(Ms) / sizeof(Ms[0]); ++k) {
            const long long M = Ms[k];
            const long long slots = pool / M;
            for (int i = 0; i < 20; ++i)                /* warm-up: code, workspace */
                BLIP_OK(blipgpu_eval(t, dpos + 3 * M * (i % slots), M, mode, val, grad, lap, ld, NULL, s));
            CUDA_OK(cudaStreamSynchronize(s));
            /* (a) call + wait: what a caller that needs psi before its next step sees */
            for (int i = 0; i < calls; ++i) {
                const double t0 = now_s();
                BLIP_OK(blipgpu_eval(t, dpos + 3 * M * ((i + 20) % slots), M, mode, val, grad, lap, ld, NULL, s));
                CUDA_OK(cudaStreamSynchronize(s));
                lat[i] = now_s() - t0;
            }
            qsort(lat, (size_t)calls, sizeof(double), cmp_double);
            const double med = lat[calls / 2], p10 = lat[calls / 10], p90 = lat[(9 * calls) / 10];
            /* (b) back-to-back calls, one wait at the end: the rate at which calls can be issued */
            const double t0 = now_s();
            for (int i = 0; i < calls; ++i)
                BLIP_OK(blipgpu_eval(t, dpos + 3 * M * ((i + 7) % slots), M, mode, val, grad, lap, ld, NULL, s));
            CUDA_OK(cudaStreamSynchronize(s));
            const double per_call = (now_s() - t0) / calls;
            printf("%s{\"M\": %lld, \"mode\": \"%s\", \"us_call_and_wait_median\": %.2f, \"us_p10\": %.2f, \"us_p90\": %.2f, "
                   "\"us_back_to_back\": %.2f, \"evals_per_s_back_to_back\": %.4g, \"kernel\": %d}",
                   first ? "" : ", ", M, mode ? "vgl" : "value", 1e6 * med, 1e6 * p10, 1e6 * p90, 1e6 * per_call,
                   (double)M * L / per_call, blipgpu_last_path(t));
            first = 0;
        }
    printf("]}\n");
    free(lat); free(hpos);
    cudaFree(dpos); cudaFree(val); cudaFree(grad); cudaFree(lap);
    cudaStreamDestroy(s);
    BLIP_OK(blipgpu_destroy(t));
    return 0;
}

/* ------------------------------------------------------------------------------------- */
static int all_finite(const float* x, size_t n)
{
    for (size_t i = 0; i < n; ++i)
        if (!isfinite(x[i])) return 0;
    return 1;
}

static int run_selftest(const char* oracle_lib)
{
    const double A[9] = {20, 0, 0, 3, 19, 0, 2, 2, 24};
    const int n[3] = {17, 12, 19};
    const int L = 257;
    const long long ld = 260, M = 6000;
    float* htable = NULL;
    blipgpu_table* t = make_table_keep(A, n, L, &htable);
    double* hpos = make_positions(A, M, 3.0);
    double *oval = NULL, *ograd = NULL, *olap = NULL, tol[3] = {0, 0, 0};
    if (oracle_lib) {
        void* so = dlopen(oracle_lib, RTLD_NOW);
        if (!so) { fprintf(stderr, "cannot load the oracle %s: %s\n", oracle_lib, dlerror()); return 2; }
        oracle_eval_fn oeval = (oracle_eval_fn)dlsym(so, "blip_oracle_eval");
        oracle_spacing_fn ospacing = (oracle_spacing_fn)dlsym(so, "blip_oracle_spacing");
        if (!oeval || !ospacing) { fprintf(stderr, "oracle symbols missing\n"); return 2; }
        oval = (double*)malloc(sizeof(double) * (size_t)M * L);
        ograd = (double*)malloc(sizeof(double) * 3 * (size_t)M * L);
        olap = (double*)malloc(sizeof(double) * (size_t)M * L);
        double hs[3], cmax = 0.0;
        if (!oval || !ograd || !olap || oeval(A, n, L, htable, hpos, M, 1, oval, ograd, olap, NULL) != 0 || ospacing(A, n, hs) != 0) {
            fprintf(stderr, "oracle evaluation failed\n");
            return 2;
        }
        const double hmax = fmax(hs[0], fmax(hs[1], hs[2]));
        for (size_t i = 0; i < (size_t)n[0] * n[1] * n[2] * (size_t)L; ++i) cmax = fmax(cmax, fabs((double)htable[i]));
        tol[0] = 2e-5 * cmax; tol[1] = 2e-5 * cmax / hmax; tol[2] = 5e-5 * cmax / (hmax * hmax);     /* north_star */
    }
    free(htable);
    double* dpos = NULL;
    float *val = NULL, *grad = NULL, *lap = NULL, *dvec = NULL, *cout = NULL;
    double *val64 = NULL, *grad64 = NULL, *lap64 = NULL;
    int* cell = NULL;
    CUDA_OK(cudaMalloc((void**)&dpos, sizeof(double) * 3 * (size_t)M));
    CUDA_OK(cudaMemcpy(dpos, hpos, sizeof(double) * 3 * (size_t)M, cudaMemcpyHostToDevice));
    CUDA_OK(cudaMalloc((void**)&val, sizeof(float) * (size_t)M * ld));
    CUDA_OK(cudaMalloc((void**)&grad, sizeof(float) * 3 * (size_t)M * ld));
    CUDA_OK(cudaMalloc((void**)&lap, sizeof(float) * (size_t)M * ld));
    CUDA_OK(cudaMalloc((void**)&dvec, sizeof(float) * (size_t)M * ld));
    CUDA_OK(cudaMalloc((void**)&cout, sizeof(float) * (size_t)M * 8));
    CUDA_OK(cudaMalloc((void**)&cell, sizeof(int) * 3 * (size_t)M));
    CUDA_OK(cudaMalloc((void**)&val64, sizeof(double) * 512 * ld));
    CUDA_OK(cudaMalloc((void**)&grad64, sizeof(double) * 3 * 512 * ld));
    CUDA_OK(cudaMalloc((void**)&lap64, sizeof(double) * 512 * ld));
    {
        float* hd = (float*)malloc(sizeof(float) * (size_t)M * ld);
        for (size_t i = 0; i < (size_t)M * ld; ++i) hd[i] = (float)(lcg_uniform() - 0.5);
        CUDA_OK(cudaMemcpy(dvec, hd, sizeof(float) * (size_t)M * ld, cudaMemcpyHostToDevice));
        free(hd);
    }
    const size_t nv = (size_t)M * ld;
    float* h_staged = (float*)malloc(sizeof(float) * 5 * nv);
    float* h_other = (float*)malloc(sizeof(float) * 5 * nv);
    int fails = 0;
    for (int mode = 1; mode >= 0; --mode) {
        for (int path = 2; path >= 0; --path) {            /* staged, direct (grouped), automatic */
            const long long Mp = path == 0 ? 300 : M;      /* automatic at M = 300: the split kernel */
            BLIP_OK(blipgpu_set_tuning(t, path, 0));
            CUDA_OK(cudaMemset(val, 0, sizeof(float) * nv));
            CUDA_OK(cudaMemset(grad, 0, sizeof(float) * 3 * nv));
            CUDA_OK(cudaMemset(lap, 0, sizeof(float) * nv));
            for (int rep = 0; rep < 2; ++rep)
                BLIP_OK(blipgpu_eval(t, dpos, Mp, mode, val, grad, lap, ld, cell, NULL));
            CUDA_OK(cudaDeviceSynchronize());
            float* h = path == 2 ? h_staged : h_other;
            CUDA_OK(cudaMemcpy(h, val, sizeof(float) * nv, cudaMemcpyDeviceToHost));
            CUDA_OK(cudaMemcpy(h + nv, grad, sizeof(float) * 3 * nv, cudaMemcpyDeviceToHost));
            CUDA_OK(cudaMemcpy(h + 4 * nv, lap, sizeof(float) * nv, cudaMemcpyDeviceToHost));
            const size_t used = (size_t)Mp * ld;
            int ok = all_finite(h, used) && (mode == 0 || (all_finite(h + nv, 3 * used) && all_finite(h + 4 * nv, used)));
            if (path == 1) ok = ok && memcmp(h_staged, h_other, sizeof(float) * (mode ? 5 : 1) * nv) == 0;
            double frac = -1.0;
            if (oval) { frac = oracle_fraction(h, nv, Mp, L, ld, mode, oval, ograd, olap, tol); ok = ok && frac <= 1.0; }
            printf("selftest mode=%d path=%d M=%lld kernel=%d: %s (worst error %.4f of the tolerance against the oracle)\n", mode, path, Mp,
                   blipgpu_last_path(t), ok ? "ok" : "FAIL", frac);
            fails += !ok;
            if (path == 2) {
                /* the tensor-core staged kernel (tuning path 5) on the same batch: finite, and close to the
                   FP32-pipe kernel's results (both are within a few % of the tolerances of the fp64 definition) */
                BLIP_OK(blipgpu_set_tuning(t, 5, 0));
                CUDA_OK(cudaMemset(val, 0, sizeof(float) * nv));
                BLIP_OK(blipgpu_eval(t, dpos, Mp, mode, val, grad, lap, ld, cell, NULL));
                CUDA_OK(cudaDeviceSynchronize());
                CUDA_OK(cudaMemcpy(h_other, val, sizeof(float) * nv, cudaMemcpyDeviceToHost));
                CUDA_OK(cudaMemcpy(h_other + nv, grad, sizeof(float) * 3 * nv, cudaMemcpyDeviceToHost));
                CUDA_OK(cudaMemcpy(h_other + 4 * nv, lap, sizeof(float) * nv, cudaMemcpyDeviceToHost));
                double worst = 0.0, scale = 0.0;
                for (size_t i = 0; i < used; ++i) {
                    const double d = fabs((double)h_other[i] - (double)h_staged[i]);
                    if (d > worst) worst = d;
                    if (fabs((double)h_staged[i]) > scale) scale = fabs((double)h_staged[i]);
                }
                ok = all_finite(h_other, used) && blipgpu_last_path(t) == 5 && worst <= 1e-5 * scale;
                double frac5 = -1.0;
                if (oval) { frac5 = oracle_fraction(h_other, nv, Mp, L, ld, mode, oval, ograd, olap, tol); ok = ok && frac5 <= 1.0; }
                printf("selftest mode=%d path=5 M=%lld kernel=%d: %s (worst error %.4f of the tolerance against the oracle; largest "
                       "|value - FP32-pipe value| %.2e of %.2e)\n", mode, Mp, blipgpu_last_path(t), ok ? "ok" : "FAIL", frac5, worst, scale);
                fails += !ok;
                BLIP_OK(blipgpu_set_tuning(t, path, 0));
            }
            /* contraction epilogue of the same kernel */
            BLIP_OK(blipgpu_eval_contract(t, dpos, Mp, mode, dvec, ld, cout, NULL, NULL));
            CUDA_OK(cudaDeviceSynchronize());
            CUDA_OK(cudaMemcpy(h_other, cout, sizeof(float) * 8 * (size_t)Mp, cudaMemcpyDeviceToHost));
            ok = all_finite(h_other, 8 * (size_t)Mp);
            printf("selftest contract mode=%d path=%d: %s\n", mode, path, ok ? "ok" : "FAIL");
            fails += !ok;
        }
        BLIP_OK(blipgpu_eval_f64(t, dpos, 512, mode, val64, grad64, lap64, ld, cell, NULL));
        CUDA_OK(cudaDeviceSynchronize());
        printf("selftest f64 mode=%d: ok\n", mode);
    }
    free(h_staged); free(h_other); free(hpos); free(oval); free(ograd); free(olap);
    cudaFree(dpos); cudaFree(val); cudaFree(grad); cudaFree(lap); cudaFree(dvec); cudaFree(cout); cudaFree(cell);
    cudaFree(val64); cudaFree(grad64); cudaFree(lap64);
    BLIP_OK(blipgpu_destroy(t));
    CUDA_OK(cudaDeviceSynchronize());
    printf("selftest: %d failure(s)\n", fails);
    return fails ? 1 : 0;
}

/* The TiO2-sized shape in the launch configuration bench.py times (49,152 positions x 768
 * orbitals, staged kernels), three calls of each entry point: for the checked build. */
static int run_fullsize(void)
{
    const double A[9] = {17.4, 0, 0, 0, 17.4, 0, 0, 0, 11.2};
    const int n[3] = {64, 64, 40};
    const int L = 768;
    const long long ld = 768, M = 49152;
    blipgpu_table* t = make_table(A, n, L);
    double* hpos = make_positions(A, M, 0.5);
    double* dpos = NULL;
    float *val = NULL, *grad = NULL, *lap = NULL, *cout = NULL;
    CUDA_OK(cudaMalloc((void**)&dpos, sizeof(double) * 3 * (size_t)M));
    CUDA_OK(cudaMemcpy(dpos, hpos, sizeof(double) * 3 * (size_t)M, cudaMemcpyHostToDevice));
    CUDA_OK(cudaMalloc((void**)&val, sizeof(float) * (size_t)M * ld));
    CUDA_OK(cudaMalloc((void**)&grad, sizeof(float) * 3 * (size_t)M * ld));
    CUDA_OK(cudaMalloc((void**)&lap, sizeof(float) * (size_t)M * ld));
    CUDA_OK(cudaMalloc((void**)&cout, sizeof(float) * 8 * (size_t)M));
    int fails = 0, kernel_eval = 0;
    for (int rep = 0; rep < 3; ++rep) {
        BLIP_OK(blipgpu_eval(t, dpos, M, BLIPGPU_VGL, val, grad, lap, ld, NULL, NULL));
        BLIP_OK(blipgpu_eval(t, dpos, M, BLIPGPU_VALUE, val, NULL, NULL, ld, NULL, NULL));
        kernel_eval = blipgpu_last_path(t);
        BLIP_OK(blipgpu_eval_contract(t, dpos, M, BLIPGPU_VGL, lap, ld, cout, NULL, NULL));
        CUDA_OK(cudaDeviceSynchronize());
    }
    /* the storing calls run the tensor-core staged kernel (5), the contraction the FP32-pipe one (2) */
    printf("fullsize: kernel=%d (eval), kernel=%d (contract)\n", kernel_eval, blipgpu_last_path(t));
    fails += kernel_eval != 5 || blipgpu_last_path(t) != 2;
    {
        float* h = (float*)malloc(sizeof(float) * (size_t)M * ld);
        CUDA_OK(cudaMemcpy(h, val, sizeof(float) * (size_t)M * ld, cudaMemcpyDeviceToHost));
        fails += !all_finite(h, (size_t)M * ld);
        free(h);
    }
    free(hpos);
    cudaFree(dpos); cudaFree(val); cudaFree(grad); cudaFree(lap); cudaFree(cout);
    BLIP_OK(blipgpu_destroy(t));
    printf("fullsize: %d failure(s)\n", fails);
    return fails ? 1 : 0;
}

int main(int argc, char** argv)
{
    if (argc >= 2 && strcmp(argv[1], "latency") == 0) return run_latency(argc >= 3 ? atoi(argv[2]) : 400);
    if (argc >= 2 && strcmp(argv[1], "selftest") == 0) return run_selftest(argc >= 3 ? argv[2] : NULL);
    if (argc >= 2 && strcmp(argv[1], "fullsize") == 0) return run_fullsize();
    fprintf(stderr, "usage: %s latency [calls] | selftest [path/to/libblip_oracle.so] | fullsize\n", argv[0]);
    return 64;
}
