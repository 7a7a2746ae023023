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

// Per-warp shared scratch: per-axis factors, then the weights of the 16 (m1, m2) columns.
struct WarpScratch {
    float ax[3][3][4];          // [axis][w, w', w''][m]
    int   k[3][4];              // wrapped site index per axis
    float4 cw[16];              // column (m1,m2): {P00, P10, P01, La}  (see warp_prepare)
    float  lb[16];              // column (m1,m2): Lb
    int    rb[16];              // column (m1,m2): first table row of the column, (k1*n2 + k2)*n3
};

// Computes the cell and the per-axis factors of electron `e`, then the column weights, into
// this warp's scratch.  All 32 lanes call it.  Returns false for a non-finite position.
//
// With S the spline in grid coordinates t, T_a = dS/dt_a and H_ab = d2S/dt_a dt_b, the z axis
// (k3, contiguous table rows) is contracted first: for column (m1, m2)
//     a = sum_m3 w3[m3] c,   b = sum_m3 w3'[m3] c,   d = sum_m3 (Q22 w3''[m3]) c
// and the column is folded into 5 accumulators with 5 per-column weights
//     val += P00 a                     P00 = w1 w2
//     T1  += P10 a                     P10 = w1' w2
//     T2  += P01 a                     P01 = w1 w2'
//     T3  += P00 b
//     lap += La a + Lb b + P00 d       La = Q00 w1'' w2 + Q11 w1 w2'' + 2 Q01 w1' w2'
//                                      Lb = 2 (Q02 w1' w2 + Q12 w1 w2')
// (lap = sum_ab Q_ab H_ab, Q = J J^T).  19 FMAs per column and orbital for any lattice; the
// Cartesian gradient grad_i = sum_a J[a][i] T_a is formed once per orbital in the epilogue.
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
    if (lane < 16) {
        const int m1 = lane >> 2, m2 = lane & 3;
        const float a0 = ws.ax[0][0][m1], b0 = ws.ax[0][1][m1], c0 = ws.ax[0][2][m1];
        const float a1 = ws.ax[1][0][m2], b1 = ws.ax[1][1][m2], c1 = ws.ax[1][2][m2];
        const float la = g.Q[0] * (c0 * a1) + g.Q[1] * (a0 * c1) + 2.0f * g.Q[3] * (b0 * b1);
        ws.cw[lane] = make_float4(a0 * a1, b0 * a1, a0 * b1, la);
        ws.lb[lane] = 2.0f * (g.Q[4] * (b0 * a1) + g.Q[5] * (a0 * b1));
        ws.rb[lane] = (ws.k[0][m1] * g.n[1] + ws.k[1][m2]) * g.n[2];
    }
    __syncwarp();
    return true;
}

__device__ __forceinline__ void st_stream(float4* p, const float4& v)
{
    asm volatile("st.global.cs.v4.f32 [%0], {%1, %2, %3, %4};"
                 :: "l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}

// Packed fp32 pairs (sm_100 FFMA2 / FMUL2: two FMAs per issue slot at the same FP32-pipe
// rate).  A pair is two consecutive orbitals; a weight is broadcast to both halves (ptxas
// folds the {w, w} move into the instruction's scalar-operand form).
typedef unsigned long long u64;
__device__ __forceinline__ u64 dup2(float w)
{
    u64 r; asm("mov.b64 %0, {%1, %1};" : "=l"(r) : "f"(w)); return r;
}
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c)
{
    u64 d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d;
}
__device__ __forceinline__ u64 mul2(u64 a, u64 b)
{
    u64 d; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d;
}
__device__ __forceinline__ float2 unpack2(u64 v)
{
    float2 r; asm("mov.b64 {%0, %1}, %2;" : "=f"(r.x), "=f"(r.y) : "l"(v)); return r;
}

// ---------------------------------------------------------------------------------------
// a-3 + a-5: warp = (electron, chunk of NQ*128 orbitals); lane owns NQ quads of 4 consecutive
// orbitals, quad q = (chunk*NQ + j)*32 + lane.  grid.x = groups of kWarpsPerBlock electrons in
// grouped order, grid.y = orbital chunk (chunk-major launch order: the CTAs in flight share
// one column slab of the table, which streams through L2 once).  Per column (m1, m2): 4*NQ
// LDG.128, coalesced across the warp (l is the sequential index), prefetched
// one column ahead of the FMAs that consume them; streaming 128-bit stores.
// ---------------------------------------------------------------------------------------
template <int MODE, int NQ>
struct EvalAcc {
    u64 val[2 * NQ], t1[2 * NQ], t2[2 * NQ], t3[2 * NQ], lp[2 * NQ];
};

template <int NQ>
__device__ __forceinline__ void load_column(const ulonglong2* __restrict__ table, const int (&quad)[NQ],
                                            const Geom& g, const WarpScratch& ws, int c,
                                            const int (&zoff)[4], ulonglong2 (&buf)[4 * NQ])
{
    const ulonglong2* base = table + (size_t)ws.rb[c] * (size_t)g.pitch4;
#pragma unroll
    for (int m = 0; m < 4; ++m)
#pragma unroll
        for (int j = 0; j < NQ; ++j) buf[m * NQ + j] = __ldg(base + zoff[m] + quad[j]);
}

template <int MODE, int NQ>
__device__ __forceinline__ void fold_column(const WarpScratch& ws, int c, const float (&wz)[3][4],
                                            const ulonglong2 (&buf)[4 * NQ], EvalAcc<MODE, NQ>& acc)
{
    const float4 w = ws.cw[c];
    const float lb = ws.lb[c];
#pragma unroll
    for (int j = 0; j < NQ; ++j)
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const u64 c0 = h ? buf[0 * NQ + j].y : buf[0 * NQ + j].x;
            const u64 c1 = h ? buf[1 * NQ + j].y : buf[1 * NQ + j].x;
            const u64 c2 = h ? buf[2 * NQ + j].y : buf[2 * NQ + j].x;
            const u64 c3 = h ? buf[3 * NQ + j].y : buf[3 * NQ + j].x;
            const int p = 2 * j + h;
            u64 a = mul2(c0, dup2(wz[0][0]));
            a = fma2(c1, dup2(wz[0][1]), a); a = fma2(c2, dup2(wz[0][2]), a); a = fma2(c3, dup2(wz[0][3]), a);
            acc.val[p] = fma2(a, dup2(w.x), acc.val[p]);
            if (MODE != 0) {
                u64 b = mul2(c0, dup2(wz[1][0]));
                b = fma2(c1, dup2(wz[1][1]), b); b = fma2(c2, dup2(wz[1][2]), b); b = fma2(c3, dup2(wz[1][3]), b);
                u64 d = mul2(c0, dup2(wz[2][0]));
                d = fma2(c1, dup2(wz[2][1]), d); d = fma2(c2, dup2(wz[2][2]), d); d = fma2(c3, dup2(wz[2][3]), d);
                acc.t1[p] = fma2(a, dup2(w.y), acc.t1[p]);
                acc.t2[p] = fma2(a, dup2(w.z), acc.t2[p]);
                acc.t3[p] = fma2(b, dup2(w.x), acc.t3[p]);
                u64 l = fma2(a, dup2(w.w), acc.lp[p]);
                l = fma2(b, dup2(lb), l);
                acc.lp[p] = fma2(d, dup2(w.x), l);
            }
        }
}

template <int MODE, int NQ>
__global__ void __launch_bounds__(kWarpsPerBlock * 32)
eval_kernel(Geom g, const float4* __restrict__ table4, const double* __restrict__ pos,
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
    const ulonglong2* __restrict__ table = reinterpret_cast<const ulonglong2*>(table4);
    int quad[NQ], lquad[NQ];
#pragma unroll
    for (int j = 0; j < NQ; ++j) {
        quad[j] = (blockIdx.y * NQ + j) * 32 + lane;
        lquad[j] = min(quad[j], g.pitch4 - 1);               // lanes past the row end re-read its last quad
    }
    const bool ok = warp_prepare(g, pos, e, ws, lane, blockIdx.y == 0 ? cell_out : nullptr);

    EvalAcc<MODE, NQ> acc;
#pragma unroll
    for (int p = 0; p < 2 * NQ; ++p) acc.val[p] = acc.t1[p] = acc.t2[p] = acc.t3[p] = acc.lp[p] = 0ull;
    if (ok) {
        float wz[3][4]; int zoff[4];
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            wz[0][m] = ws.ax[2][0][m]; wz[1][m] = ws.ax[2][1][m]; wz[2][m] = g.Q[2] * ws.ax[2][2][m];
            zoff[m] = ws.k[2][m] * g.pitch4;
        }
        ulonglong2 buf0[4 * NQ], buf1[4 * NQ];
        load_column<NQ>(table, lquad, g, ws, 0, zoff, buf0);
#pragma unroll 1
        for (int c = 0; c < 16; c += 2) {
            load_column<NQ>(table, lquad, g, ws, c + 1, zoff, buf1);
            fold_column<MODE, NQ>(ws, c, wz, buf0, acc);
            if (c + 2 < 16) load_column<NQ>(table, lquad, g, ws, c + 2, zoff, buf0);
            fold_column<MODE, NQ>(ws, c + 1, wz, buf1, acc);
        }
    }
    const float nan = __int_as_float(0x7fc00000);
#pragma unroll
    for (int j = 0; j < NQ; ++j) {
        if (quad[j] >= g.pitch4) continue;
        float4 v, gx, gy, gz, lp;
        if (ok) {
            const float2 v0 = unpack2(acc.val[2 * j]), v1 = unpack2(acc.val[2 * j + 1]);
            v = make_float4(v0.x, v0.y, v1.x, v1.y);
            if (MODE != 0) {
                const float2 a0 = unpack2(acc.t1[2 * j]), a1 = unpack2(acc.t1[2 * j + 1]);
                const float2 b0 = unpack2(acc.t2[2 * j]), b1 = unpack2(acc.t2[2 * j + 1]);
                const float2 c0 = unpack2(acc.t3[2 * j]), c1 = unpack2(acc.t3[2 * j + 1]);
                const float2 l0 = unpack2(acc.lp[2 * j]), l1 = unpack2(acc.lp[2 * j + 1]);
                const float4 T1 = make_float4(a0.x, a0.y, a1.x, a1.y);
                const float4 T2 = make_float4(b0.x, b0.y, b1.x, b1.y);
                const float4 T3 = make_float4(c0.x, c0.y, c1.x, c1.y);
#define BLIP_GRAD(i, out)                                                                       \
                out.x = fmaf(g.J[i], T1.x, fmaf(g.J[3 + i], T2.x, g.J[6 + i] * T3.x));         \
                out.y = fmaf(g.J[i], T1.y, fmaf(g.J[3 + i], T2.y, g.J[6 + i] * T3.y));         \
                out.z = fmaf(g.J[i], T1.z, fmaf(g.J[3 + i], T2.z, g.J[6 + i] * T3.z));         \
                out.w = fmaf(g.J[i], T1.w, fmaf(g.J[3 + i], T2.w, g.J[6 + i] * T3.w));
                BLIP_GRAD(0, gx) BLIP_GRAD(1, gy) BLIP_GRAD(2, gz)
#undef BLIP_GRAD
                lp = make_float4(l0.x, l0.y, l1.x, l1.y);
            }
        } else {
            v = make_float4(nan, nan, nan, nan); gx = gy = gz = lp = v;
        }
        const size_t o = (size_t)e * (size_t)ld + 4 * (size_t)quad[j];
        st_stream(reinterpret_cast<float4*>(val + o), v);
        if (MODE != 0) {
            const size_t og = (size_t)e * 3 * (size_t)ld + 4 * (size_t)quad[j];
            st_stream(reinterpret_cast<float4*>(grad + og), gx);
            st_stream(reinterpret_cast<float4*>(grad + og + ld), gy);
            st_stream(reinterpret_cast<float4*>(grad + og + 2 * ld), gz);
            st_stream(reinterpret_cast<float4*>(lap + o), lp);
        }
    }
}

}  // namespace blip
