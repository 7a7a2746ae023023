// tcgen05_check.cu — the tcgen05 / tensor-memory facts blip::eval_tc_kernel (csrc/blip_tc.cuh) is built on,
// checked on the device against a host loop (no library code involved; tests/test_gpu_tc.py builds
// and runs it).  None of them is spelled out in the guides this repository was written from; they
// were found with this program:
//   * A operand in tensor memory ("TS" form of tcgen05.mma, kind::f16 and kind::tf32): lane = row m,
//     column = k; a 32-bit column holds ONE tf32 or TWO fp16 (k = 2c in the low half, 2c + 1 in
//     the high half); written with tcgen05.st.32x32b (a warp owns the lane quarter 32 (warp % 4));
//   * the A operand may start at any column that is a multiple of 4 (other offsets fault with
//     "misaligned address") — hence a table row of 8 fp16 z sites = 4 columns in blip_tc.cuh;
//   * B operand from shared memory, K-major, no swizzle: core matrices of 8 N-rows x 16 bytes, the
//     K halves of one MMA `leading byte offset` apart, the N halves `stride byte offset` apart;
//     descriptor = (addr >> 4) | (LBO >> 4) << 16 | (SBO >> 4) << 32 | 1 << 46;
//   * instruction descriptor: D fp32 (1 << 4), A/B format (0 fp16, 2 tf32) at bits 7 and 10,
//     N >> 3 at bit 17, M >> 4 at bit 24; the predicate operand selects accumulate / overwrite;
//   * tcgen05.commit -> mbarrier, tcgen05.ld.32x32b of the fp32 accumulator (lane = m, column = n).
// Exit code 0 when every case matches.
#include <cstdio>
#include <cstdlib>
#include <cstdint>
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <vector>
#include <cmath>

#define CK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) { printf("CUDA error %s at %d\n", cudaGetErrorString(e_), __LINE__); exit(1); } } while (0)

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ uint64_t make_bdesc(unsigned addr, unsigned lbo, unsigned sbo)
{
    uint64_t d = 0;
    d |= (uint64_t)((addr >> 4) & 0x3fff);
    d |= (uint64_t)((lbo >> 4) & 0x3fff) << 16;
    d |= (uint64_t)((sbo >> 4) & 0x3fff) << 32;
    d |= (uint64_t)1 << 46;          // version 1 (Blackwell)
    return d;                         // layout type 0 (no swizzle), base offset 0
}

// kind: 0 = f16 (K = 16 per MMA, 2 per column), 1 = tf32 (K = 8, one per column)
__global__ void __launch_bounds__(128) tc1(float* out, int kind, int acol, int nmma, int astep)
{
    __shared__ alignas(128) unsigned char bt[4096];
    __shared__ unsigned tbase_s;
    __shared__ alignas(8) unsigned long long bar;
    const int tid = threadIdx.x, warp = tid >> 5;
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 128;" :: "r"(smem_u32(&tbase_s)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    if (tid == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" :: "r"(smem_u32(&bar)) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const unsigned tbase = tbase_s;
    const int m = tid;                 // TMEM lane = row of A and D
    // ---- A: 64 columns.  f16: column c holds k = 2c (low half), 2c+1 (high half); tf32: column c holds k = c
    {
        unsigned v[64];
        for (int c = 0; c < 64; ++c) {
            if (kind == 0) {
                const __half lo = __float2half((float)((m & 15) + 16 * ((2 * c) & 63)) * 0.25f);
                const __half hi = __float2half((float)((m & 15) + 16 * ((2 * c + 1) & 63)) * 0.25f);
                v[c] = (unsigned)__half_as_ushort(lo) | ((unsigned)__half_as_ushort(hi) << 16);
            } else {
                v[c] = __float_as_uint((float)((m & 15) + 16 * (c & 63)) * 0.25f);
            }
        }
        const unsigned ta = tbase + ((unsigned)(warp * 32) << 16);
#pragma unroll
        for (int c = 0; c < 64; c += 8)
            asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};"
                         :: "r"(ta + c), "r"(v[c]), "r"(v[c + 1]), "r"(v[c + 2]), "r"(v[c + 3]), "r"(v[c + 4]), "r"(v[c + 5]),
                            "r"(v[c + 6]), "r"(v[c + 7]) : "memory");
        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
    }
    // ---- B tiles: nmma tiles of [K][N = 16], K-major core matrices (8 n x 16 bytes), tile j selects
    // B[k][n] = (k == n + ... ) pattern: B_j[k][n] = 1 if k == n (f16: K = 16; tf32: K = 8, n < 8) scaled by (j + 1)
    const int K = kind == 0 ? 16 : 8, esz = kind == 0 ? 2 : 4, kpc = 16 / esz;   // k per 16-byte row of a core matrix
    const unsigned tile_bytes = 16 * K * esz;                 // 512 (f16) or 512 (tf32)
    for (int i = tid; i < nmma * 16 * K; i += 128) {
        const int j = i / (16 * K), r = i % (16 * K), n = r / K, k = r % K;
        const float val = (k == n) ? (float)(j + 1) : 0.f;
        const unsigned off = j * tile_bytes + ((n / 8) * (K / kpc) + (k / kpc)) * 128 + (n % 8) * 16 + (k % kpc) * esz;
        if (kind == 0) *reinterpret_cast<__half*>(bt + off) = __float2half(val);
        else *reinterpret_cast<float*>(bt + off) = val;
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const unsigned dcol = 64;          // D: columns 64..79
    if (tid == 0) {
        const unsigned idesc = (1u << 4) | ((kind == 0 ? 0u : 2u) << 7) | ((kind == 0 ? 0u : 2u) << 10) | ((16u >> 3) << 17) | ((128u >> 4) << 24);
        for (int j = 0; j < nmma; ++j) {
            const uint64_t bd = make_bdesc(smem_u32(bt) + j * tile_bytes, 128, (K / kpc) * 128);
            const unsigned acc = j > 0;
            if (kind == 0)
                asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                             "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}"
                             :: "r"(tbase + dcol), "r"(tbase + (unsigned)(acol + j * astep)), "l"(bd), "r"(idesc), "r"(acc) : "memory");
            else
                asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                             "tcgen05.mma.cta_group::1.kind::tf32 [%0], [%1], %2, %3, p;\n\t}"
                             :: "r"(tbase + dcol), "r"(tbase + (unsigned)(acol + j * astep)), "l"(bd), "r"(idesc), "r"(acc) : "memory");
        }
        asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" :: "r"(smem_u32(&bar)) : "memory");
    }
    // wait for the MMAs
    {
        unsigned done = 0;
        while (!done)
            asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                         : "=r"(done) : "r"(smem_u32(&bar)) : "memory");
    }
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    {
        unsigned r[16];
        const unsigned ta = tbase + ((unsigned)(warp * 32) << 16) + dcol;
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
                     : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
                       "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
                     : "r"(ta) : "memory");
        asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
        for (int n = 0; n < 16; ++n) out[m * 16 + n] = __uint_as_float(r[n]);
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 128;" :: "r"(tbase) : "memory");
}

static float a_val(int kind, int m, int k)     // A[m][k] as the kernel fills it (k = global k index from column 0)
{
    return (float)((m & 15) + 16 * (k & 63)) * 0.25f;
}

int main()
{
    float* d; CK(cudaMalloc(&d, 128 * 16 * 4));
    std::vector<float> h(128 * 16);
    int failures = 0;
    struct Case { int kind, acol, nmma, astep; };
    const Case cases[] = {{0, 0, 1, 0}, {0, 8, 1, 0}, {0, 4, 1, 0}, {0, 4, 3, 8}, {0, 0, 4, 4},
                          {1, 0, 1, 0}, {1, 8, 1, 0}, {1, 4, 1, 0}, {1, 4, 3, 8}};
    for (const Case& c : cases) {
        CK(cudaMemset(d, 0xff, 128 * 16 * 4));
        tc1<<<1, 128>>>(d, c.kind, c.acol, c.nmma, c.astep);
        CK(cudaDeviceSynchronize());
        CK(cudaMemcpy(h.data(), d, 128 * 16 * 4, cudaMemcpyDeviceToHost));
        const int K = c.kind == 0 ? 16 : 8, kpcol = c.kind == 0 ? 2 : 1;
        int bad = 0; double maxerr = 0;
        for (int m = 0; m < 128; ++m)
            for (int n = 0; n < 16; ++n) {
                double ex = 0;
                for (int j = 0; j < c.nmma; ++j)
                    if (n < K) ex += (double)(j + 1) * a_val(c.kind, m, (c.acol + j * c.astep) * kpcol + n);
                const double err = fabs(h[m * 16 + n] - ex);
                if (err > maxerr) maxerr = err;
                if (err > 1e-3 * fmax(1.0, fabs(ex))) ++bad;
            }
        printf("kind=%s A column %d, %d MMA(s) %d columns apart: %d of 2048 accumulators differ (largest error %g)\n", c.kind ? "tf32" : "f16", c.acol,
               c.nmma, c.astep, bad, maxerr);
        failures += bad != 0;
    }
    printf("tcgen05_check: %d failure(s)\n", failures);
    return failures ? 1 : 0;
}
