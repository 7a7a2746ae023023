// mma_sync_probe.cuh — timing probe for the tensor-core recast of the gather + FMA step
// (§VI.E, Eq. 13-15: psi = A(r_j) . Theta is a matrix
// product, rejected by the paper because A changes with r_j).  A settled experiment, kept as a
// harness program (tests/harness/mma_sync_probe.cu) outside the shipped library: the mma.sync
// form lost to packed FP32 FMAs (profiles/r2_v1.md), the tcgen05 form of csrc/blip_tc.cuh won.
// Its outputs are not orbitals.
//
// What it times.  One "unit" of the staged kernel is one electron x 128 orbitals: the 64 site
// rows of the electron's 4x4x4 block, already in shared memory, against 5 weight vectors
// (value, 3 gradient components, Laplacian).  Per unit that is the product
//       D[128 orbitals][5] = C^T[128][64 sites] . W[64][5]
// — K = 64, per electron, no padding to the 196 rows of a plane.  Both forms below run it from
// the same shared-memory tile with the same launch shape as the staged kernel (one CTA per SM,
// 16 warps, each warp a stream of units), without TMA traffic or plane hand-offs: the question
// is only which pipe does the arithmetic faster.
//   form 0  packed FP32 FMAs exactly as the shipped kernel issues them: z axis contracted
//           first, 18 FMAs per column and orbital (MODE 2), 64 LDS.128 per unit.
//   form 1  mma.sync.m16n8k8 tf32 with the 3-term hi/lo split (A_hi B_hi + A_lo B_hi + A_hi B_lo;
//           a single tf32 pass carries 11 bits = 5e-4, against a tolerance of 2e-5): M = 16
//           orbitals, N = 8 (5 quantities used), K = 8 sites -> 8 x 8 MMAs per term, 192 per
//           unit.  The coefficient tile is read with one LDS.32 per fragment register from a
//           tile padded to 136 floats per row (conflict-free; the TMA tile of the real kernel
//           has 128-float rows and would 4-way conflict here, so this is the recast's best
//           case), split with LOP3 + FADD per element; the weights are split once per unit.
//           The D fragments go through shared memory to get back to orbital-contiguous rows.
//   form 2  form 1 with a single tf32 term (64 MMAs per unit, no split): the tensor-pipe floor
//           of the recast if precision were not an issue.
#pragma once
#include <cuda_runtime.h>

namespace blip_probe {

constexpr int kProbeWarps = 16;
constexpr int kProbePitch = 136;                               // floats per site row of the padded tile

__device__ __forceinline__ void mma_tf32(float (&d)[4], const unsigned (&a)[4], unsigned b0, unsigned b1)
{
    asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}

struct ProbeSmem {
    float tile[64 * kProbePitch];                               // 64 site rows x 128 orbitals (+ 8 pad)
    float wts[kProbeWarps][3][3][4];                            // per warp: per-axis w, w', w'' at the 4 sites
    float dfrag[kProbeWarps][8][16 * 9];                        // per warp: D of one orbital tile, [16 orbitals][8 + 1 pad]
};

template <int FORM>
__global__ void __launch_bounds__(kProbeWarps * 32, 1)
mma_sync_probe_kernel(float* __restrict__ out, int units_per_warp, float seed)
{
    extern __shared__ __align__(16) unsigned char probe_raw[];
    ProbeSmem& sm = *reinterpret_cast<ProbeSmem*>(probe_raw);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int i = threadIdx.x; i < 64 * kProbePitch; i += blockDim.x) sm.tile[i] = seed * (float)((i * 2654435761u) >> 20);
    if (lane < 12) for (int k = 0; k < 3; ++k) sm.wts[warp][lane >> 2][k][lane & 3] = seed * (float)(lane + 3 * k + 1);
    __syncthreads();
    float* orow = out + ((size_t)blockIdx.x * kProbeWarps + warp) * 5 * 128;      // one unit's worth of output rows, rewritten
    float drift = 0.f;
    if (FORM == 0) {
        // ---- packed FP32 form: lane owns 4 orbitals; 16 columns x (4 LDS.128 + 36 FFMA2)
        typedef unsigned long long u64;
        auto dup2 = [](float w) { u64 r; asm("mov.b64 %0, {%1, %1};" : "=l"(r) : "f"(w)); return r; };
        auto fma2 = [](u64 a, u64 b, u64 c) { u64 d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d; };
        auto mul2 = [](u64 a, u64 b) { u64 d; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; };
        const unsigned base = (unsigned)__cvta_generic_to_shared(&sm.tile[0]) + lane * 16;
#pragma unroll 1
        for (int u = 0; u < units_per_warp; ++u) {
            float wz[3][4];
#pragma unroll
            for (int k = 0; k < 3; ++k)
#pragma unroll
                for (int m = 0; m < 4; ++m) wz[k][m] = sm.wts[warp][2][k][m] + drift;
            u64 acc[2][5];
#pragma unroll
            for (int p = 0; p < 2; ++p)
#pragma unroll
                for (int q = 0; q < 5; ++q) acc[p][q] = 0ull;
#pragma unroll
            for (int col = 0; col < 16; ++col) {
                const float p00 = sm.wts[warp][0][0][col >> 2] * sm.wts[warp][1][0][col & 3];
                const float p10 = sm.wts[warp][0][1][col >> 2], p01 = sm.wts[warp][1][1][col & 3], la = sm.wts[warp][0][2][col >> 2];
                ulonglong2 c[4];
#pragma unroll
                for (int m = 0; m < 4; ++m)
                    asm volatile("ld.shared.v2.b64 {%0, %1}, [%2];" : "=l"(c[m].x), "=l"(c[m].y) : "r"(base + (4 * col + m) * (kProbePitch * 4)));
#pragma unroll
                for (int p = 0; p < 2; ++p) {
                    const u64 c0 = p ? c[0].y : c[0].x, c1 = p ? c[1].y : c[1].x, c2 = p ? c[2].y : c[2].x, c3 = p ? c[3].y : c[3].x;
                    u64 a = mul2(c0, dup2(wz[0][0])); a = fma2(c1, dup2(wz[0][1]), a); a = fma2(c2, dup2(wz[0][2]), a); a = fma2(c3, dup2(wz[0][3]), a);
                    u64 b = mul2(c0, dup2(wz[1][0])); b = fma2(c1, dup2(wz[1][1]), b); b = fma2(c2, dup2(wz[1][2]), b); b = fma2(c3, dup2(wz[1][3]), b);
                    u64 d = mul2(c0, dup2(wz[2][0])); d = fma2(c1, dup2(wz[2][1]), d); d = fma2(c2, dup2(wz[2][2]), d); d = fma2(c3, dup2(wz[2][3]), d);
                    acc[p][0] = fma2(a, dup2(p00), acc[p][0]);
                    acc[p][1] = fma2(a, dup2(p10), acc[p][1]);
                    acc[p][2] = fma2(a, dup2(p01), acc[p][2]);
                    acc[p][3] = fma2(b, dup2(p00), acc[p][3]);
                    acc[p][4] = fma2(d, dup2(p00), fma2(a, dup2(la), acc[p][4]));
                }
            }
#pragma unroll
            for (int q = 0; q < 5; ++q) {
                float2 x, y;
                asm("mov.b64 {%0, %1}, %2;" : "=f"(x.x), "=f"(x.y) : "l"(acc[0][q]));
                asm("mov.b64 {%0, %1}, %2;" : "=f"(y.x), "=f"(y.y) : "l"(acc[1][q]));
                asm volatile("st.global.cs.v4.f32 [%0], {%1, %2, %3, %4};" :: "l"(orow + q * 128 + 4 * lane), "f"(x.x), "f"(x.y), "f"(y.x), "f"(y.y) : "memory");
                drift += x.x * 1e-30f;
            }
        }
    } else {
        // ---- tensor-core form.  Fragment coordinates of m16n8k8: g = lane / 4, t = lane % 4.
        const int g = lane >> 2, t = lane & 3;
        constexpr int NTERM = FORM == 1 ? 3 : 1;
#pragma unroll 1
        for (int u = 0; u < units_per_warp; ++u) {
            // B fragments: W[site][quantity], quantity = g (5 used), sites t and t + 4 of each k-step
            // (site s = 16 m1 + 4 m2 + m3): product of three per-axis factors, split into hi + lo
            unsigned bhi[8][2], blo[8][2];
#pragma unroll
            for (int ks = 0; ks < 8; ++ks)
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const int s = 8 * ks + t + 4 * h;
                    const int kx = (g == 1) ? 1 : (g == 4 ? 2 : 0), ky = (g == 2) ? 1 : 0, kz = (g == 3) ? 1 : 0;
                    float w = sm.wts[warp][0][kx][s >> 4] * sm.wts[warp][1][ky][(s >> 2) & 3] * (sm.wts[warp][2][kz][s & 3] + drift);
                    if (g >= 5) w = 0.f;
                    const unsigned hi = __float_as_uint(w) & 0xffffe000u;
                    bhi[ks][h] = hi;
                    blo[ks][h] = __float_as_uint(w - __uint_as_float(hi));
                }
#pragma unroll 1
            for (int ot = 0; ot < 8; ++ot) {                 // 16 orbitals per tile
                float d[4] = {0.f, 0.f, 0.f, 0.f};
                const float* col = &sm.tile[16 * ot + g];
#pragma unroll
                for (int ks = 0; ks < 8; ++ks) {
                    // A fragment: C^T[orbital][site]: (g, t), (g + 8, t), (g, t + 4), (g + 8, t + 4)
                    const float x0 = col[(8 * ks + t) * kProbePitch], x1 = col[(8 * ks + t) * kProbePitch + 8];
                    const float x2 = col[(8 * ks + t + 4) * kProbePitch], x3 = col[(8 * ks + t + 4) * kProbePitch + 8];
                    unsigned ahi[4] = {__float_as_uint(x0) & 0xffffe000u, __float_as_uint(x1) & 0xffffe000u,
                                       __float_as_uint(x2) & 0xffffe000u, __float_as_uint(x3) & 0xffffe000u};
                    mma_tf32(d, ahi, bhi[ks][0], bhi[ks][1]);
                    if (NTERM == 3) {
                        unsigned alo[4] = {__float_as_uint(x0 - __uint_as_float(ahi[0])), __float_as_uint(x1 - __uint_as_float(ahi[1])),
                                           __float_as_uint(x2 - __uint_as_float(ahi[2])), __float_as_uint(x3 - __uint_as_float(ahi[3]))};
                        mma_tf32(d, alo, bhi[ks][0], bhi[ks][1]);
                        mma_tf32(d, ahi, blo[ks][0], blo[ks][1]);
                    }
                }
                // D fragment: (orbital g, quantities 2t, 2t+1), (orbital g + 8, same) -> shared memory
                float* df = &sm.dfrag[warp][ot][0];
                df[g * 9 + 2 * t] = d[0]; df[g * 9 + 2 * t + 1] = d[1];
                df[(g + 8) * 9 + 2 * t] = d[2]; df[(g + 8) * 9 + 2 * t + 1] = d[3];
            }
            __syncwarp();
            // back to orbital-contiguous rows: lane owns orbitals 4 lane .. 4 lane + 3
#pragma unroll
            for (int q = 0; q < 5; ++q) {
                const float* df = &sm.dfrag[warp][lane >> 2][0];
                const int o = (4 * lane) & 15;
                const float a = df[o * 9 + q], b = df[(o + 1) * 9 + q], c = df[(o + 2) * 9 + q], e = df[(o + 3) * 9 + q];
                asm volatile("st.global.cs.v4.f32 [%0], {%1, %2, %3, %4};" :: "l"(orow + q * 128 + 4 * lane), "f"(a), "f"(b), "f"(c), "f"(e) : "memory");
                drift += a * 1e-30f;
            }
            __syncwarp();
        }
    }
    if (drift == 123.456f) out[0] = drift;
}

}  // namespace blip_probe
