// blip_kernels.cuh — sm_100a device code of the blip orbital evaluator (product path).
//
// Steps of the hot path, all on the GPU:
//   a-1 cell map       r -> (i_a, f_a)          PAPER.md:98-102 (Eq. 8); fp64, pinned sequence
//   a-2 weights        f_a -> w, w', w'' -> 64 x {W, Gx, Gy, Gz, Lam}   PAPER.md:84-86 (Eq. 7)
//   a-3 gather + FMA   64 coefficient rows x 5 weights per orbital     PAPER.md:78-80 (Eq. 6)
//   a-4 grouping       counting sort of electrons by brick of cells (not in the paper)
//   a-5 output         val/grad/lap in caller order, orbital index innermost
//
// Shares nothing with oracle/ (the CPU fp64 checker): the weight polynomials below are
// written in the symmetric B(x) form, the oracle uses the expanded per-site pieces.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace blip {

constexpr int kWarpsPerBlock = 8;          // eval kernel: one warp = one electron x 128 orbitals
constexpr int kBrick = 4;                  // grouping: bricks of 4x4x4 cells
constexpr int kScanThreads = 1024;

struct Geom {
    double G[9];        // inverse lattice, u = r.G (row vector), fp64 for the index map
    int n[3];           // grid points per axis
    int nb[3];          // bricks per axis
    float J[9];         // J[a][i] = n_a G[i][a] = d t_a / d r_i
    float Q[6];         // (J J^T): Q00 Q11 Q22 Q01 Q02 Q12
    int L;              // orbitals
    int pitch4;         // table row pitch in float4 (= ceil(L/4))
};

// ---------------------------------------------------------------------------------------
// a-1: cell map.  The IEEE sequence is pinned so that the integer
// cell index is a pure function of the caller's bits: no FMA contraction (__dmul_rn /
// __dadd_rn), wrap by u - floor(u), fold the u -> 1.0 rounding case back to cell 0.
// Returns false for a non-finite position.
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ bool cell_map_axis(const Geom& g, int a, double x, double y, double z,
                                              int& i, float& f)
{
    double u = __dadd_rn(__dadd_rn(__dmul_rn(x, g.G[a]), __dmul_rn(y, g.G[3 + a])),
                         __dmul_rn(z, g.G[6 + a]));
    if (!isfinite(u)) { i = -1; f = __int_as_float(0x7fc00000); return false; }
    u = __dsub_rn(u, floor(u));
    double t = __dmul_rn(u, (double)g.n[a]);
    int ia = (int)floor(t);
    if (ia >= g.n[a]) { ia -= g.n[a]; t = __dsub_rn(t, (double)g.n[a]); }
    i = ia;
    f = (float)__dsub_rn(t, (double)ia);
    return true;
}

__device__ __forceinline__ int brick_of(const Geom& g, int i0, int i1, int i2)
{
    return ((i0 / kBrick) * g.nb[1] + (i1 / kBrick)) * g.nb[2] + (i2 / kBrick);
}

// ---------------------------------------------------------------------------------------
// a-4 (1/3): one thread per electron: cell -> brick bin, histogram, optional cell output.
// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
bin_kernel(Geom g, const double* __restrict__ pos, long long M,
           int* __restrict__ bin, unsigned* __restrict__ hist, int* __restrict__ cell)
{
    long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= M) return;
    double x = pos[3 * e], y = pos[3 * e + 1], z = pos[3 * e + 2];
    int i0, i1, i2; float f;
    bool ok = cell_map_axis(g, 0, x, y, z, i0, f);
    ok = cell_map_axis(g, 1, x, y, z, i1, f) && ok;
    ok = cell_map_axis(g, 2, x, y, z, i2, f) && ok;
    if (!ok) i0 = i1 = i2 = -1;
    if (cell) { cell[3 * e] = i0; cell[3 * e + 1] = i1; cell[3 * e + 2] = i2; }
    int b = ok ? brick_of(g, i0, i1, i2) : 0;
    bin[e] = b;
    atomicAdd(&hist[b], 1u);
}

// a-4 (2/3): exclusive scan of the histogram, in place, one CTA.
__global__ void __launch_bounds__(kScanThreads)
scan_kernel(unsigned* __restrict__ hist, int nbins)
{
    __shared__ unsigned part[kScanThreads];
    const int tid = threadIdx.x;
    const int per = (nbins + kScanThreads - 1) / kScanThreads;
    const int lo = min(tid * per, nbins), hi = min(lo + per, nbins);
    unsigned s = 0;
    for (int b = lo; b < hi; ++b) s += hist[b];
    part[tid] = s;
    __syncthreads();
    for (int d = 1; d < kScanThreads; d <<= 1) {            // Hillis-Steele inclusive scan
        unsigned v = (tid >= d) ? part[tid - d] : 0u;
        __syncthreads();
        part[tid] += v;
        __syncthreads();
    }
    unsigned run = part[tid] - s;                            // exclusive prefix of this segment
    for (int b = lo; b < hi; ++b) { unsigned c = hist[b]; hist[b] = run; run += c; }
}

// a-4 (3/3): scatter electron ids into brick order (order inside a brick is arbitrary; the
// results do not depend on it because every electron is evaluated independently).
__global__ void __launch_bounds__(256)
scatter_kernel(const int* __restrict__ bin, unsigned* __restrict__ offs, long long M,
               int* __restrict__ perm)
{
    long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= M) return;
    unsigned slot = atomicAdd(&offs[bin[e]], 1u);
    perm[slot] = (int)e;
}

// ---------------------------------------------------------------------------------------
// a-2: the 1-D factor phi (cardinal cubic B-spline) at the 4 sites i-1..i+2 as a function of
// f = t - i, written through the distance x to the site's own end of the cell:
//   outer sites (m = 0, 3):  B = x^3/6,               x = 1-f (m=0) or f (m=3)
//   inner sites (m = 1, 2):  B = 2/3 - x^2 (1 - x/2),  x = f (m=1) or 1-f (m=2)
// d/dt picks up a minus sign when x = 1-f.  [Not printed in the paper: PAPER.md:98 only says
// "polynomial"; readings R1-R3.]
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ void phi_site(float f, int m, float& w, float& d1, float& d2)
{
    const bool mirrored = (m == 0) || (m == 2);
    const float x = mirrored ? 1.0f - f : f;
    const float sg = mirrored ? -1.0f : 1.0f;
    if (m == 0 || m == 3) {
        w = x * x * x * (1.0f / 6.0f);
        d1 = sg * 0.5f * x * x;
        d2 = x;
    } else {
        w = (2.0f / 3.0f) - x * x * (1.0f - 0.5f * x);
        d1 = sg * x * (1.5f * x - 2.0f);
        d2 = 3.0f * x - 2.0f;
    }
}

__device__ __forceinline__ int wrap_site(int k, int n)
{
    return k < 0 ? k + n : (k >= n ? k - n : k);
}

// Per-warp shared scratch: per-axis factors, then the 64 folded weight sets + row indices.
struct WarpScratch {
    float ax[3][3][4];          // [axis][w, w', w''][m]
    int   k[3][4];              // wrapped site index per axis
    float4 wg[64];              // {W, Gx, Gy, Gz} per site
    float2 lr[64];              // {Lam, row index (int bits)} per site
};

// Computes the cell, the per-axis factors and the 64 folded weights of electron `e` into
// this warp's scratch.  All 32 lanes call it.  Returns false for a non-finite position.
template <int MODE>
__device__ __forceinline__ bool warp_prepare(const Geom& g, const double* __restrict__ pos,
                                             long long e, WarpScratch& ws, int lane,
                                             int* __restrict__ cell_out)
{
    const double x = pos[3 * e], y = pos[3 * e + 1], z = pos[3 * e + 2];
    int ia = 0; float fa = 0.f; bool ok = true;
    if (lane < 12) {
        const int a = lane >> 2, m = lane & 3;
        ok = cell_map_axis(g, a, x, y, z, ia, fa);
        float w, d1, d2;
        phi_site(fa, m, w, d1, d2);
        ws.ax[a][0][m] = w; ws.ax[a][1][m] = d1; ws.ax[a][2][m] = d2;
        ws.k[a][m] = wrap_site(ia - 1 + m, g.n[a]);
        if (cell_out && m == 0) cell_out[3 * e + a] = ok ? ia : -1;
    }
    ok = __all_sync(0xffffffffu, ok);
    __syncwarp();
    if (!ok) return false;
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        const int s = lane + 32 * h;
        const int m0 = s >> 4, m1 = (s >> 2) & 3, m2 = s & 3;
        const float a0 = ws.ax[0][0][m0], a1 = ws.ax[1][0][m1], a2 = ws.ax[2][0][m2];
        const int row = (ws.k[0][m0] * g.n[1] + ws.k[1][m1]) * g.n[2] + ws.k[2][m2];
        const float W = a0 * a1 * a2;
        if (MODE == 0) {
            ws.lr[s] = make_float2(W, __int_as_float(row));
        } else {
            const float b0 = ws.ax[0][1][m0], b1 = ws.ax[1][1][m1], b2 = ws.ax[2][1][m2];
            const float c0 = ws.ax[0][2][m0], c1 = ws.ax[1][2][m1], c2 = ws.ax[2][2][m2];
            const float a12 = a1 * a2, a02 = a0 * a2, a01 = a0 * a1;
            const float T0 = b0 * a12, T1 = b1 * a02, T2 = b2 * a01;         // dS/dt_a weights
            const float gx = g.J[0] * T0 + g.J[3] * T1 + g.J[6] * T2;
            const float gy = g.J[1] * T0 + g.J[4] * T1 + g.J[7] * T2;
            const float gz = g.J[2] * T0 + g.J[5] * T1 + g.J[8] * T2;
            const float lam = g.Q[0] * (c0 * a12) + g.Q[1] * (c1 * a02) + g.Q[2] * (c2 * a01)
                            + 2.0f * (g.Q[3] * (b0 * b1 * a2) + g.Q[4] * (b0 * b2 * a1)
                                      + g.Q[5] * (b1 * b2 * a0));
            ws.wg[s] = make_float4(W, gx, gy, gz);
            ws.lr[s] = make_float2(lam, __int_as_float(row));
        }
    }
    __syncwarp();
    return true;
}

__device__ __forceinline__ void st_stream(float4* p, const float4& v)
{
    asm volatile("st.global.cs.v4.f32 [%0], {%1, %2, %3, %4};"
                 :: "l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}

// ---------------------------------------------------------------------------------------
// a-3 + a-5, v0: warp = (electron, chunk of 128 orbitals), lane = 4 consecutive orbitals.
// grid.x = groups of kWarpsPerBlock electrons in grouped order, grid.y = orbital chunk, so
// that the CTAs in flight share one 512-byte column of the table rows (L1/L2 locality).
// 64 x LDG.128 per lane, coalesced across the warp (l is the sequential
// index), 5 FMAs per coefficient, streaming 128-bit stores.
// ---------------------------------------------------------------------------------------
template <int MODE>
__global__ void __launch_bounds__(kWarpsPerBlock * 32)
eval_kernel(Geom g, const float4* __restrict__ table, const double* __restrict__ pos,
            const int* __restrict__ perm, long long M,
            float* __restrict__ val, float* __restrict__ grad, float* __restrict__ lap,
            long long ld, int* __restrict__ cell_out)
{
    __shared__ WarpScratch scratch[kWarpsPerBlock];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long long sidx = (long long)blockIdx.x * kWarpsPerBlock + warp;
    if (sidx >= M) return;                                   // warp-uniform; no block barrier below
    const long long e = perm ? (long long)perm[sidx] : sidx;
    WarpScratch& ws = scratch[warp];
    const int quad = blockIdx.y * 32 + lane;
    const bool active = quad < g.pitch4;
    const bool ok = warp_prepare<MODE>(g, pos, e, ws, lane, blockIdx.y == 0 ? cell_out : nullptr);

    float4 v = make_float4(0.f, 0.f, 0.f, 0.f), gx = v, gy = v, gz = v, lp = v;
    if (ok && active) {
        const float4* __restrict__ col = table + quad;
        constexpr int U = 8;
#pragma unroll 1
        for (int s0 = 0; s0 < 64; s0 += U) {
            float4 c[U];
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int row = __float_as_int(ws.lr[s0 + u].y);
                c[u] = __ldg(col + (size_t)row * (size_t)g.pitch4);
            }
#pragma unroll
            for (int u = 0; u < U; ++u) {
                if (MODE == 0) {
                    const float W = ws.lr[s0 + u].x;
                    v.x = fmaf(W, c[u].x, v.x); v.y = fmaf(W, c[u].y, v.y);
                    v.z = fmaf(W, c[u].z, v.z); v.w = fmaf(W, c[u].w, v.w);
                } else {
                    const float4 w = ws.wg[s0 + u];
                    const float lam = ws.lr[s0 + u].x;
                    v.x = fmaf(w.x, c[u].x, v.x); v.y = fmaf(w.x, c[u].y, v.y);
                    v.z = fmaf(w.x, c[u].z, v.z); v.w = fmaf(w.x, c[u].w, v.w);
                    gx.x = fmaf(w.y, c[u].x, gx.x); gx.y = fmaf(w.y, c[u].y, gx.y);
                    gx.z = fmaf(w.y, c[u].z, gx.z); gx.w = fmaf(w.y, c[u].w, gx.w);
                    gy.x = fmaf(w.z, c[u].x, gy.x); gy.y = fmaf(w.z, c[u].y, gy.y);
                    gy.z = fmaf(w.z, c[u].z, gy.z); gy.w = fmaf(w.z, c[u].w, gy.w);
                    gz.x = fmaf(w.w, c[u].x, gz.x); gz.y = fmaf(w.w, c[u].y, gz.y);
                    gz.z = fmaf(w.w, c[u].z, gz.z); gz.w = fmaf(w.w, c[u].w, gz.w);
                    lp.x = fmaf(lam, c[u].x, lp.x); lp.y = fmaf(lam, c[u].y, lp.y);
                    lp.z = fmaf(lam, c[u].z, lp.z); lp.w = fmaf(lam, c[u].w, lp.w);
                }
            }
        }
    }
    if (!active) return;
    if (!ok) {
        const float nan = __int_as_float(0x7fc00000);
        v = make_float4(nan, nan, nan, nan); gx = gy = gz = lp = v;
    }
    const size_t o = (size_t)e * (size_t)ld + 4 * (size_t)quad;
    st_stream(reinterpret_cast<float4*>(val + o), v);
    if (MODE != 0) {
        const size_t og = (size_t)e * 3 * (size_t)ld + 4 * (size_t)quad;
        st_stream(reinterpret_cast<float4*>(grad + og), gx);
        st_stream(reinterpret_cast<float4*>(grad + og + ld), gy);
        st_stream(reinterpret_cast<float4*>(grad + og + 2 * ld), gz);
        st_stream(reinterpret_cast<float4*>(lap + o), lp);
    }
}

}  // namespace blip
