// blipgpu_dev.cu — developer / benchmark instrumentation declared in include/blipgpu_dev.h.
// Not part of the boundary of SURVEY.md §8(b): nothing here is on the evaluation path.  It
// forces a kernel (tests), counts launches and times the kernels of a call (bench.py's
// `gpu_launches` and `roofline` keys) and measures the device's packed-FP32 rate (the FP32
// roofline denominator, measured in the same run as the kernel it is compared with).
#include "blipgpu.h"
#include "blipgpu_dev.h"
#include "blip_host.h"

int blip_default_nq(int pitch4);     // blipgpu.cu

namespace blip {
typedef unsigned long long u64;
static __device__ __forceinline__ u64 dup2(float w)
{
    u64 r; asm("mov.b64 %0, {%1, %1};" : "=l"(r) : "f"(w)); return r;
}
static __device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c)
{
    u64 d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d;
}
static __device__ __forceinline__ float2 unpack2(u64 v)
{
    float2 r; asm("mov.b64 {%0, %1}, %2;" : "=f"(r.x), "=f"(r.y) : "l"(v)); return r;
}

// FP32 peak probe (the FP32 roofline is measured in the same run): every thread
// runs `iters` rounds of 4 x 16 independent packed FMAs on registers.
__global__ void __launch_bounds__(512)
fp32_probe_kernel(float* __restrict__ out, int iters, float seed)
{
    u64 acc[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) acc[i] = dup2(seed * (float)(i + 1 + threadIdx.x));
    const u64 x = dup2(0.999f);
    const float w = 1.0f + seed;
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
            for (int i = 0; i < 16; ++i) acc[i] = fma2(acc[i], dup2(w), x);
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 16; ++i) { const float2 v = unpack2(acc[i]); s += v.x + v.y; }
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}
}  // namespace blip

extern "C" int blipgpu_set_profiling(blipgpu_table* t, int on)
{
    if (!t) return BLIPGPU_EINVAL;
    if (on)
        for (int k = 0; k < 3; ++k)
            if (!t->pe[k]) CK(t, cudaEventCreate(&t->pe[k]));
    t->profiling = on ? 1 : 0;
    return BLIPGPU_OK;
}

extern "C" int blipgpu_last_kernel_ms(blipgpu_table* t, float* group_ms, float* eval_ms)
{
    if (!t || !t->profiling || !t->pe[2]) return BLIPGPU_EINVAL;
    CK(t, cudaEventSynchronize(t->pe[2]));
    float a = 0.f, b = 0.f;
    CK(t, cudaEventElapsedTime(&a, t->pe[0], t->pe[1]));
    CK(t, cudaEventElapsedTime(&b, t->pe[1], t->pe[2]));
    if (group_ms) *group_ms = a;
    if (eval_ms) *eval_ms = b;
    return BLIPGPU_OK;
}

extern "C" int blipgpu_set_tuning(blipgpu_table* t, int path, int nq)
{
    if (!t || path < 0 || (path > 2 && path != 5) || nq < 0 || nq > 3) return BLIPGPU_EINVAL;
    if (path == 2 && !t->staged_ok) return BLIPGPU_EINVAL;
    if (path == 5 && !(t->staged_ok && t->tc_ok)) return BLIPGPU_EINVAL;
    t->path = path;
    t->nq = nq ? nq : blip_default_nq(t->g.pitch4);
    return BLIPGPU_OK;
}

extern "C" int blipgpu_probe_fp32(blipgpu_table* t, double* tflops, void* stream)
{
    if (!t || !tflops) return BLIPGPU_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    const int blocks = t->nsm * 4, threads = 512, iters = 4096;
    float* out = nullptr;
    CK(t, cudaMalloc(&out, sizeof(float) * (size_t)blocks * threads));
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    int rc = BLIPGPU_OK;
    float ms = 0.f;
    cudaError_t e = cudaEventCreate(&e0);
    if (e == cudaSuccess) e = cudaEventCreate(&e1);
    for (int rep = 0; rep < 3 && e == cudaSuccess; ++rep) {          // the last of three runs is timed
        e = cudaEventRecord(e0, s);
        blip::fp32_probe_kernel<<<blocks, threads, 0, s>>>(out, iters, 1e-9f);
        if (e == cudaSuccess) e = cudaGetLastError();
        if (e == cudaSuccess) e = cudaEventRecord(e1, s);
        if (e == cudaSuccess) e = cudaEventSynchronize(e1);
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    }
    if (e != cudaSuccess) { t->last_cuda = (int)e; (void)cudaGetLastError(); rc = BLIPGPU_ECUDA; }
    else *tflops = 2.0 * 2.0 * 64.0 * (double)iters * (double)blocks * threads / (ms * 1e-3) / 1e12;
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaFree(out);
    t->launches += 3;
    return rc;
}

extern "C" int blipgpu_last_path(const blipgpu_table* t) { return t ? t->last_path : 0; }

extern "C" long long blipgpu_launch_count(const blipgpu_table* t) { return t ? t->launches : 0; }
