// blip_kernels.cuh — sm_100a device code of the blip orbital evaluator (product path).
//
// Steps of the hot path, all on the GPU:
//   a-1 cell map       r -> (i_a, f_a)          PAPER.md:98-102 (Eq. 8); fp64, pinned sequence
//   a-2 weights        f_a -> w, w', w'' -> per-column weights          PAPER.md:84-86 (Eq. 7)
//   a-3 gather + FMA   64 coefficient rows per orbital                  PAPER.md:78-80 (Eq. 6)
//   a-4 grouping       counting sort of electrons by cell group (not in the paper)
//   a-5 output         val/grad/lap in caller order, orbital index innermost
//
// Two evaluation kernels share the arithmetic (fold_pair below):
//   eval_direct_kernel  warp = electron x NQ*128 orbitals, coefficient rows gathered straight
//                       from L2/HBM into registers; for sparse batches (few electrons per cell)
//   eval_staged_kernel  CTA = pencil of cells x 128 (or 64) orbitals; the planes of the table
//                       the pencil touches slide through shared memory by TMA, every electron
//                       of the pencil is evaluated from shared memory; for dense batches
//
// The table is stored ghost-padded: T[p1][p2][p3][l] = c[(p1-1) mod n1][(p2-1) mod n2]
// [(p3-1) mod n3][l], p_a in [0, n_a+3), so that the 4x4x4 block of an electron in cell i is
// the box p_a = i_a .. i_a+3 with no wrap-around (one TMA box per plane, contiguous z rows).
//
// Shares nothing with oracle/ (the CPU fp64 checker): the weight polynomials below are
// written in the symmetric B(x) form and the sum is contracted z axis first, the oracle uses
// the expanded per-site pieces and keeps all 10 grid-space accumulators.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace blip {

constexpr int kWarpsPerBlock = 8;          // direct kernel: 8 electrons per CTA
constexpr int kBrick = 4;                  // direct path grouping: bricks of 4x4x4 cells
constexpr int kScanThreads = 1024;
constexpr int kRecFloats = 96;             // per-electron record (ElecRec), 384 bytes

struct Geom {
    double G[9];        // inverse lattice, u = r.G (row vector), fp64 for the index map
    int n[3];           // grid points per axis
    int np[3];          // padded table extent per axis, n + 3
    int nb[3];          // direct path: bricks per axis
    float J[9];         // J[a][i] = n_a G[i][a] = d t_a / d r_i
    float Q[6];         // (J J^T): Q00 Q11 Q22 Q01 Q02 Q12
    int L;              // orbitals
    int pitch4;         // table row pitch in float4 (= ceil(L/4))
};

// Geometry of the staged path: pencils of BY x BZ cells running along axis 1, cut into
// segments of `seg` cell planes.  Sort key of an electron = (pencil, i1).
struct StagedGeom {
    int by, bz;         // cross-section of a pencil in cells (template constants of the kernel)
    int nby, nbz;       // pencils per axis
    int seg;            // cell planes per segment
    int nseg;           // segments per pencil = ceil(n1 / seg)
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

__device__ __forceinline__ int staged_key(const Geom& g, const StagedGeom& sg, int i0, int i1, int i2)
{
    return ((i1 / sg.by) * sg.nbz + (i2 / sg.bz)) * g.n[0] + i0;
}

// ---------------------------------------------------------------------------------------
// a-4 (1/3): one thread per electron: cell -> bin, histogram, optional cell output.
// staged != 0: bin = (pencil, i1); else bin = 4x4x4 brick.
// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
bin_kernel(Geom g, StagedGeom sg, int staged, const double* __restrict__ pos, long long M,
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
    int b = 0;
    if (ok) b = staged ? staged_key(g, sg, i0, i1, i2) : brick_of(g, i0, i1, i2);
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

// a-4 (3/3): scatter electron ids into bin order (order inside a bin is arbitrary; the
// results do not depend on it because every electron is evaluated independently).  On return
// offs[b] is the END of bin b in the sorted order.
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
// Table set-up: ghost-padded copy of the caller's [n1][n2][n3][L] table, one thread per
// float4 of the destination, pad columns L..pitch-1 zero.
// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
pad_kernel(Geom g, const float* __restrict__ src, float4* __restrict__ dst, long long total4)
{
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= total4) return;
    const int q = (int)(idx % g.pitch4);
    long long prow = idx / g.pitch4;
    const int p3 = (int)(prow % g.np[2]); prow /= g.np[2];
    const int p2 = (int)(prow % g.np[1]);
    const int p1 = (int)(prow / g.np[1]);
    const int k1 = (p1 + g.n[0] - 1) % g.n[0], k2 = (p2 + g.n[1] - 1) % g.n[1], k3 = (p3 + g.n[2] - 1) % g.n[2];
    const float* s = src + (((size_t)k1 * g.n[1] + k2) * g.n[2] + k3) * (size_t)g.L;
    float v[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) v[j] = (4 * q + j < g.L) ? __ldg(s + 4 * q + j) : 0.0f;
    dst[idx] = make_float4(v[0], v[1], v[2], v[3]);
}

// ---------------------------------------------------------------------------------------
// a-2: the 1-D factor phi (cardinal cubic B-spline) at the 4 sites i-1..i+2 as a function of
// f = t - i, written through the distance x to the site's own end of the cell:
//   outer sites (m = 0, 3):  B = x^3/6,               x = 1-f (m=0) or f (m=3)
//   inner sites (m = 1, 2):  B = 2/3 - x^2 (1 - x/2),  x = f (m=1) or 1-f (m=2)
// d/dt picks up a minus sign when x = 1-f.  [Not printed in the paper: PAPER.md:98 only says
// "polynomial"; readings R1-R3.]  Explicit rounding intrinsics: the direct and the
// staged path must produce bit-identical weights.
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ void phi_site(float f, int m, float& w, float& d1, float& d2)
{
    const bool mirrored = (m == 0) || (m == 2);
    const float x = mirrored ? __fsub_rn(1.0f, f) : f;
    const float sg = mirrored ? -1.0f : 1.0f;
    const float x2 = __fmul_rn(x, x);
    if (m == 0 || m == 3) {
        w = __fmul_rn(__fmul_rn(x2, x), 1.0f / 6.0f);
        d1 = __fmul_rn(sg, __fmul_rn(0.5f, x2));
        d2 = x;
    } else {
        w = __fsub_rn(2.0f / 3.0f, __fmul_rn(x2, __fmaf_rn(-0.5f, x, 1.0f)));
        d1 = __fmul_rn(sg, __fmul_rn(x, __fmaf_rn(1.5f, x, -2.0f)));
        d2 = __fmaf_rn(3.0f, x, -2.0f);
    }
}

// Per-electron record: everything the gather + FMA loop needs, 96 floats.
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
struct ElecRec {
    float4 cw[16];      // column (m1,m2) = 4 m1 + m2: {P00, P10, P01, La}
    float  lb[16];      // column: Lb
    float  wz[3][4];    // w3, w3', Q22 w3''
    int    i[3];        // cell index (i1, i2, i3); -1 for a non-finite position
    int    e;           // electron id in the caller's order
};
static_assert(sizeof(ElecRec) == kRecFloats * 4, "ElecRec is 96 floats");

// Column weights of column `col` from the per-axis factors ax[axis][w, w', w''][m].
template <typename AX>
__device__ __forceinline__ void column_weights(const Geom& g, const AX& ax, int col, float4& cw, float& lb)
{
    const int m1 = col >> 2, m2 = col & 3;
    const float a0 = ax[0][0][m1], b0 = ax[0][1][m1], c0 = ax[0][2][m1];
    const float a1 = ax[1][0][m2], b1 = ax[1][1][m2], c1 = ax[1][2][m2];
    const float p00 = __fmul_rn(a0, a1), p10 = __fmul_rn(b0, a1), p01 = __fmul_rn(a0, b1);
    float la = __fmul_rn(g.Q[0], __fmul_rn(c0, a1));
    la = __fmaf_rn(g.Q[1], __fmul_rn(a0, c1), la);
    la = __fmaf_rn(__fmul_rn(2.0f, g.Q[3]), __fmul_rn(b0, b1), la);
    cw = make_float4(p00, p10, p01, la);
    lb = __fmul_rn(2.0f, __fmaf_rn(g.Q[4], p10, __fmul_rn(g.Q[5], p01)));
}

// Warp-cooperative a-1 + a-2 for electron `e` into `rec` (shared memory).  `ax` is per-warp
// scratch.  All 32 lanes call it.
__device__ __forceinline__ void warp_prepare(const Geom& g, const double* __restrict__ pos, int e,
                                             float (&ax)[3][3][4], ElecRec& rec, int lane)
{
    const double x = pos[3 * (size_t)e], y = pos[3 * (size_t)e + 1], z = pos[3 * (size_t)e + 2];
    if (lane < 12) {
        const int a = lane >> 2, m = lane & 3;
        int ia; float fa;
        const bool ok = cell_map_axis(g, a, x, y, z, ia, fa);
        float w, d1, d2;
        phi_site(fa, m, w, d1, d2);
        ax[a][0][m] = w; ax[a][1][m] = d1; ax[a][2][m] = d2;
        if (m == 0) rec.i[a] = ok ? ia : -1;
    }
    if (lane == 12) rec.e = e;
    __syncwarp();
    if (lane < 16) {
        float4 cw; float lb;
        column_weights(g, ax, lane, cw, lb);
        rec.cw[lane] = cw; rec.lb[lane] = lb;
    } else if (lane < 28) {
        const int k = (lane - 16) >> 2, m = lane & 3;
        rec.wz[k][m] = (k == 2) ? __fmul_rn(g.Q[2], ax[2][2][m]) : ax[2][k][m];
    }
    __syncwarp();
}

// a-1 + a-2 for the staged path: one thread per electron of the sorted order, records to
// global memory (384 B each; read back through L2 by the staged kernel once per orbital chunk).
__global__ void __launch_bounds__(128)
prep_kernel(Geom g, const double* __restrict__ pos, const int* __restrict__ perm, long long M,
            float4* __restrict__ recs)
{
    const long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= M) return;
    const int e = perm[s];
    const double x = pos[3 * (size_t)e], y = pos[3 * (size_t)e + 1], z = pos[3 * (size_t)e + 2];
    float ax[3][3][4]; int ic[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        int ia; float fa;
        const bool ok = cell_map_axis(g, a, x, y, z, ia, fa);
        ic[a] = ok ? ia : -1;
#pragma unroll
        for (int m = 0; m < 4; ++m) phi_site(fa, m, ax[a][0][m], ax[a][1][m], ax[a][2][m]);
    }
    float4* out = recs + (size_t)s * (kRecFloats / 4);
    float lb[16];
#pragma unroll
    for (int col = 0; col < 16; ++col) {
        float4 cw;
        column_weights(g, ax, col, cw, lb[col]);
        out[col] = cw;
    }
#pragma unroll
    for (int k = 0; k < 4; ++k) out[16 + k] = make_float4(lb[4 * k], lb[4 * k + 1], lb[4 * k + 2], lb[4 * k + 3]);
    out[20] = make_float4(ax[2][0][0], ax[2][0][1], ax[2][0][2], ax[2][0][3]);
    out[21] = make_float4(ax[2][1][0], ax[2][1][1], ax[2][1][2], ax[2][1][3]);
    out[22] = make_float4(__fmul_rn(g.Q[2], ax[2][2][0]), __fmul_rn(g.Q[2], ax[2][2][1]),
                          __fmul_rn(g.Q[2], ax[2][2][2]), __fmul_rn(g.Q[2], ax[2][2][3]));
    out[23] = make_float4(__int_as_float(ic[0]), __int_as_float(ic[1]), __int_as_float(ic[2]),
                          __int_as_float(e));
}

// ---------------------------------------------------------------------------------------
// Packed fp32 pairs (sm_100 FFMA2 / FMUL2: two FMAs per issue slot at the same FP32-pipe
// rate).  A pair is two consecutive orbitals; a weight is broadcast to both halves (ptxas
// folds the {w, w} move into the instruction's scalar-operand form).
// ---------------------------------------------------------------------------------------
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

// Accumulators of one pair of orbitals.
struct PairAcc { u64 val, t1, t2, t3, lp; };

// a-3 for one column (m1, m2) and one pair of orbitals: c0..c3 are the coefficient pairs of
// the 4 z sites.  Both kernels call this with the same operands in the same order, so their
// results are bit-identical.
template <int MODE>
__device__ __forceinline__ void fold_pair(u64 c0, u64 c1, u64 c2, u64 c3, const float (&wz)[3][4],
                                          const float4& w, float lb, PairAcc& acc)
{
    u64 a = mul2(c0, dup2(wz[0][0]));
    a = fma2(c1, dup2(wz[0][1]), a); a = fma2(c2, dup2(wz[0][2]), a); a = fma2(c3, dup2(wz[0][3]), a);
    acc.val = fma2(a, dup2(w.x), acc.val);
    if (MODE != 0) {
        u64 b = mul2(c0, dup2(wz[1][0]));
        b = fma2(c1, dup2(wz[1][1]), b); b = fma2(c2, dup2(wz[1][2]), b); b = fma2(c3, dup2(wz[1][3]), b);
        u64 d = mul2(c0, dup2(wz[2][0]));
        d = fma2(c1, dup2(wz[2][1]), d); d = fma2(c2, dup2(wz[2][2]), d); d = fma2(c3, dup2(wz[2][3]), d);
        acc.t1 = fma2(a, dup2(w.y), acc.t1);
        acc.t2 = fma2(a, dup2(w.z), acc.t2);
        acc.t3 = fma2(b, dup2(w.x), acc.t3);
        u64 l = fma2(a, dup2(w.w), acc.lp);
        l = fma2(b, dup2(lb), l);
        acc.lp = fma2(d, dup2(w.x), l);
    }
}

__device__ __forceinline__ void st_stream4(float* p, float a, float b, float c, float d)
{
    asm volatile("st.global.cs.v4.f32 [%0], {%1, %2, %3, %4};"
                 :: "l"(p), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}
__device__ __forceinline__ void st_stream2(float* p, float a, float b)
{
    asm volatile("st.global.cs.v2.f32 [%0], {%1, %2};" :: "l"(p), "f"(a), "f"(b) : "memory");
}

// a-5 for NP consecutive pairs (NP = 1: 2 orbitals, NP = 2: 4 orbitals) starting at orbital
// column `col0` of electron `e`: Cartesian gradient from the grid-space one, streaming stores
// (evict-first: outputs are never re-read and must not push table rows out of L2).
template <int MODE, int NP>
__device__ __forceinline__ void store_pairs(const Geom& g, const PairAcc (&acc)[NP], bool ok, int e,
                                            int col0, float* __restrict__ val, float* __restrict__ grad,
                                            float* __restrict__ lap, long long ld)
{
    const float nan = __int_as_float(0x7fc00000);
    float v[2 * NP], gx[2 * NP], gy[2 * NP], gz[2 * NP], lp[2 * NP];
#pragma unroll
    for (int p = 0; p < NP; ++p) {
        const float2 s = unpack2(acc[p].val);
        v[2 * p] = ok ? s.x : nan; v[2 * p + 1] = ok ? s.y : nan;
        if (MODE != 0) {
            const float2 a = unpack2(acc[p].t1), b = unpack2(acc[p].t2), c = unpack2(acc[p].t3);
            const float2 l = unpack2(acc[p].lp);
            const float ta[2] = {a.x, a.y}, tb[2] = {b.x, b.y}, tc[2] = {c.x, c.y};
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const float x = __fmaf_rn(g.J[0], ta[h], __fmaf_rn(g.J[3], tb[h], __fmul_rn(g.J[6], tc[h])));
                const float y = __fmaf_rn(g.J[1], ta[h], __fmaf_rn(g.J[4], tb[h], __fmul_rn(g.J[7], tc[h])));
                const float z = __fmaf_rn(g.J[2], ta[h], __fmaf_rn(g.J[5], tb[h], __fmul_rn(g.J[8], tc[h])));
                gx[2 * p + h] = ok ? x : nan; gy[2 * p + h] = ok ? y : nan; gz[2 * p + h] = ok ? z : nan;
            }
            lp[2 * p] = ok ? l.x : nan; lp[2 * p + 1] = ok ? l.y : nan;
        }
    }
    const size_t o = (size_t)e * (size_t)ld + (size_t)col0;
    const size_t og = (size_t)e * 3 * (size_t)ld + (size_t)col0;
    if (NP == 2) {
        st_stream4(val + o, v[0], v[1], v[2], v[3]);
        if (MODE != 0) {
            st_stream4(grad + og, gx[0], gx[1], gx[2], gx[3]);
            st_stream4(grad + og + ld, gy[0], gy[1], gy[2], gy[3]);
            st_stream4(grad + og + 2 * ld, gz[0], gz[1], gz[2], gz[3]);
            st_stream4(lap + o, lp[0], lp[1], lp[2], lp[3]);
        }
    } else {
        st_stream2(val + o, v[0], v[1]);
        if (MODE != 0) {
            st_stream2(grad + og, gx[0], gx[1]);
            st_stream2(grad + og + ld, gy[0], gy[1]);
            st_stream2(grad + og + 2 * ld, gz[0], gz[1]);
            st_stream2(lap + o, lp[0], lp[1]);
        }
    }
}

// ---------------------------------------------------------------------------------------
// Direct kernel: warp = (electron, chunk of NQ*128 orbitals); lane owns NQ quads of 4
// consecutive orbitals, quad q = (chunk*NQ + j)*32 + lane.  grid.x = groups of kWarpsPerBlock
// electrons in grouped order, grid.y = orbital chunk (chunk-major launch order: the CTAs in
// flight share one column slab of the table).  Per column (m1, m2): 4*NQ LDG.128, coalesced
// across the warp (l is the sequential index), prefetched one column ahead
// of the FMAs that consume them.
// ---------------------------------------------------------------------------------------
struct DirectScratch {
    ElecRec rec;
    float ax[3][3][4];
};

template <int NQ>
__device__ __forceinline__ void load_column(const ulonglong2* __restrict__ table, const unsigned (&off)[NQ],
                                            unsigned colrow, int pitch4, ulonglong2 (&buf)[4 * NQ])
{
    const unsigned base = colrow * (unsigned)pitch4;
#pragma unroll
    for (int m = 0; m < 4; ++m)
#pragma unroll
        for (int j = 0; j < NQ; ++j) buf[m * NQ + j] = __ldg(table + (base + m * (unsigned)pitch4 + off[j]));
}

template <int MODE, int NQ>
__device__ __forceinline__ void fold_column(const ElecRec& rec, int c, const float (&wz)[3][4],
                                            const ulonglong2 (&buf)[4 * NQ], PairAcc (&acc)[NQ][2])
{
    const float4 w = rec.cw[c];
    const float lb = rec.lb[c];
#pragma unroll
    for (int j = 0; j < NQ; ++j) {
        fold_pair<MODE>(buf[0 * NQ + j].x, buf[1 * NQ + j].x, buf[2 * NQ + j].x, buf[3 * NQ + j].x, wz, w, lb, acc[j][0]);
        fold_pair<MODE>(buf[0 * NQ + j].y, buf[1 * NQ + j].y, buf[2 * NQ + j].y, buf[3 * NQ + j].y, wz, w, lb, acc[j][1]);
    }
}

template <int MODE, int NQ>
__global__ void __launch_bounds__(kWarpsPerBlock * 32)
eval_direct_kernel(Geom g, const float4* __restrict__ table4, const double* __restrict__ pos,
                   const int* __restrict__ perm, long long M,
                   float* __restrict__ val, float* __restrict__ grad, float* __restrict__ lap,
                   long long ld, int* __restrict__ cell_out)
{
    __shared__ DirectScratch scratch[kWarpsPerBlock];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long long sidx = (long long)blockIdx.x * kWarpsPerBlock + warp;
    if (sidx >= M) return;                                   // warp-uniform; no block barrier below
    const int e = perm ? perm[sidx] : (int)sidx;
    DirectScratch& ws = scratch[warp];
    const ulonglong2* __restrict__ table = reinterpret_cast<const ulonglong2*>(table4);
    int quad[NQ]; unsigned off[NQ];
#pragma unroll
    for (int j = 0; j < NQ; ++j) {
        quad[j] = (blockIdx.y * NQ + j) * 32 + lane;
        off[j] = (unsigned)min(quad[j], g.pitch4 - 1);       // lanes past the row end re-read its last quad
    }
    warp_prepare(g, pos, e, ws.ax, ws.rec, lane);
    const int i1 = ws.rec.i[0], i2 = ws.rec.i[1], i3 = ws.rec.i[2];
    const bool ok = (i1 | i2 | i3) >= 0;
    if (cell_out && blockIdx.y == 0 && lane < 3) cell_out[3 * (size_t)e + lane] = ok ? ws.rec.i[lane] : -1;

    PairAcc acc[NQ][2];
#pragma unroll
    for (int j = 0; j < NQ; ++j)
#pragma unroll
        for (int h = 0; h < 2; ++h) acc[j][h].val = acc[j][h].t1 = acc[j][h].t2 = acc[j][h].t3 = acc[j][h].lp = 0ull;
    if (ok) {
        float wz[3][4];
#pragma unroll
        for (int k = 0; k < 3; ++k)
#pragma unroll
            for (int m = 0; m < 4; ++m) wz[k][m] = ws.rec.wz[k][m];
        // padded row of site (m1, m2, m3 = 0): ((i1 + m1) np2 + (i2 + m2)) np3 + i3
        const unsigned row0 = ((unsigned)i1 * g.np[1] + i2) * g.np[2] + i3;
        const unsigned s1 = (unsigned)g.np[1] * g.np[2], s2 = (unsigned)g.np[2];
        ulonglong2 buf0[4 * NQ], buf1[4 * NQ];
        load_column<NQ>(table, off, row0, g.pitch4, buf0);
#pragma unroll 1
        for (int c = 0; c < 16; c += 2) {
            const unsigned r1 = row0 + (c >> 2) * s1 + ((c + 1) & 3) * s2;
            load_column<NQ>(table, off, r1, g.pitch4, buf1);
            fold_column<MODE, NQ>(ws.rec, c, wz, buf0, acc);
            if (c + 2 < 16) {
                const unsigned r2 = row0 + ((c + 2) >> 2) * s1 + ((c + 2) & 3) * s2;
                load_column<NQ>(table, off, r2, g.pitch4, buf0);
            }
            fold_column<MODE, NQ>(ws.rec, c + 1, wz, buf1, acc);
        }
    }
#pragma unroll
    for (int j = 0; j < NQ; ++j)
        if (quad[j] < g.pitch4) store_pairs<MODE, 2>(g, acc[j], ok, e, 4 * quad[j], val, grad, lap, ld);
}

// ---------------------------------------------------------------------------------------
// Staged kernel.  Work item (blockIdx.x = pencil segment, blockIdx.y = orbital chunk of C =
// 32*VEC orbitals): the electrons of the segment, sorted by cell plane i1, are the units; the
// table planes p1 = lo .. hi+3 of the pencil's (BY+3) x (BZ+3) cross-section slide through a
// ring of R shared-memory slots.  One producer warp issues one TMA box per plane; NW consumer
// warps take units from a shared counter.  A consumer at plane i1 waits for planes i1..i1+3
// (full barriers) and, when it moves past plane s, releases it (empty barriers, NW arrivals),
// which lets the producer overwrite the slot of plane s with plane s+R.
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" :: "r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}"
        :: "r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_4d(unsigned dst, const CUtensorMap* tmap, int c0, int c1, int c2, int c3,
                                            unsigned bar)
{
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes "
        "[%0], [%1, {%2, %3, %4, %5}], [%6];"
        :: "r"(dst), "l"(reinterpret_cast<uint64_t>(tmap)), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(bar)
        : "memory");
}

template <int VEC, int BY, int BZ, int R, int NW>
struct StagedCfg {
    static constexpr int C = 32 * VEC;                       // orbitals per tile row
    static constexpr int PY = BY + 3, PZ = BZ + 3;
    static constexpr int PLANE_FLOATS = PY * PZ * C;
    static constexpr int PLANE_BYTES = PLANE_FLOATS * 4;
    static constexpr int THREADS = (NW + 1) * 32;
    struct Smem {
        alignas(128) float plane[R][PLANE_FLOATS];
        alignas(16) ElecRec rec[NW][2];
        alignas(8) u64 full[R];
        alignas(8) u64 empty[R];
        int counter;
    };
};

template <int MODE, int VEC, int BY, int BZ, int R, int NW>
__global__ void __launch_bounds__((NW + 1) * 32, 1)
eval_staged_kernel(const __grid_constant__ CUtensorMap tmap, Geom g, StagedGeom sg,
                   const float4* __restrict__ recs, const unsigned* __restrict__ bin_end,
                   float* __restrict__ val, float* __restrict__ grad, float* __restrict__ lap, long long ld)
{
    using Cfg = StagedCfg<VEC, BY, BZ, R, NW>;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    typename Cfg::Smem& sm = *reinterpret_cast<typename Cfg::Smem*>(smem_raw);
    constexpr int NP = VEC / 2;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int pencil = blockIdx.x / sg.nseg, segi = blockIdx.x - pencil * sg.nseg;
    const int lo = segi * sg.seg, hi = min(lo + sg.seg, g.n[0]) - 1;         // cell planes of this segment
    const int bin0 = pencil * g.n[0] + lo, bin1 = pencil * g.n[0] + hi;
    const unsigned u0 = bin0 ? bin_end[bin0 - 1] : 0u, u1 = bin_end[bin1];
    if (u0 == u1) return;                                                    // no electrons here
    const int chunk = blockIdx.y;
    const int by = pencil / sg.nbz, bz = pencil - by * sg.nbz;

    if (threadIdx.x == 0) {
        for (int s = 0; s < R; ++s) { mbar_init(smem_u32(&sm.full[s]), 1); mbar_init(smem_u32(&sm.empty[s]), NW); }
        sm.counter = 0;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();

    if (warp == NW) {
        // ---- producer: one TMA box {C, PZ, PY, 1} per table plane, in plane order; before
        // leaving, wait until the last planes have landed (no copy may outlive the CTA)
        if (lane == 0) {
            const int nplanes = hi + 4 - lo;
            for (int k = 0; k < nplanes; ++k) {
                const int slot = k % R, round = k / R;
                if (round > 0) mbar_wait(smem_u32(&sm.empty[slot]), (unsigned)((round & 1) ^ 1));
                const unsigned bar = smem_u32(&sm.full[slot]);
                mbar_expect_tx(bar, Cfg::PLANE_BYTES);
                tma_load_4d(smem_u32(&sm.plane[slot][0]), &tmap, chunk * Cfg::C, bz * BZ, by * BY, lo + k, bar);
            }
            for (int k = max(0, nplanes - R); k < nplanes; ++k)
                mbar_wait(smem_u32(&sm.full[k % R]), (unsigned)((k / R) & 1));
        }
        return;
    }

    // ---- consumers
    const unsigned nunits = u1 - u0;
    const float4* __restrict__ rsrc = recs + (size_t)u0 * (kRecFloats / 4);
    // Every warp walks through the planes in order: it waits for plane q only after releasing
    // plane q-R (whose slot plane q reuses), and releases a plane only after having waited for
    // it, so that its NW arrivals on an empty barrier always belong to the barrier's current phase.
    int released = lo;                 // planes < released have been released by this warp
    int waited = lo - 1;               // planes <= waited have been waited for by this warp
    auto advance = [&](int need_upto, int release_below) {
        for (int q = waited + 1; q <= need_upto; ++q) {
            for (; released <= q - R; ++released)
                if (lane == 0) mbar_arrive(smem_u32(&sm.empty[(released - lo) % R]));
            mbar_wait(smem_u32(&sm.full[(q - lo) % R]), (unsigned)(((q - lo) / R) & 1));
        }
        waited = max(waited, need_upto);
        for (; released < release_below; ++released)
            if (lane == 0) mbar_arrive(smem_u32(&sm.empty[(released - lo) % R]));
    };
    auto grab = [&]() -> unsigned {
        unsigned u = 0;
        if (lane == 0) u = (unsigned)atomicAdd(&sm.counter, 1);
        return __shfl_sync(0xffffffffu, u, 0);
    };
    unsigned u = grab();
    int cur = 0;
    if (u < nunits) {
        if (lane < kRecFloats / 4)
            reinterpret_cast<float4*>(&sm.rec[warp][0])[lane] = __ldg(rsrc + (size_t)u * (kRecFloats / 4) + lane);
        __syncwarp();
    }
    while (u < nunits) {
        const unsigned un = grab();
        float4 pre = make_float4(0.f, 0.f, 0.f, 0.f);
        if (un < nunits && lane < kRecFloats / 4) pre = __ldg(rsrc + (size_t)un * (kRecFloats / 4) + lane);

        const ElecRec& rec = sm.rec[warp][cur];
        const int i1 = rec.i[0], i2 = rec.i[1], i3 = rec.i[2], e = rec.e;
        const bool ok = i1 >= 0;                             // non-finite positions (bin 0) touch no plane
        const int pl = i1;
        PairAcc acc[NP];
#pragma unroll
        for (int p = 0; p < NP; ++p) acc[p].val = acc[p].t1 = acc[p].t2 = acc[p].t3 = acc[p].lp = 0ull;
        if (ok) {
            advance(pl + 3, pl);                             // planes pl..pl+3 resident, planes < pl released
            float wz[3][4];
#pragma unroll
            for (int k = 0; k < 3; ++k)
#pragma unroll
                for (int m = 0; m < 4; ++m) wz[k][m] = rec.wz[k][m];
            const int r23 = ((i2 - by * BY) * Cfg::PZ + (i3 - bz * BZ)) * Cfg::C + lane * VEC;
#pragma unroll
            for (int m1 = 0; m1 < 4; ++m1) {
                const float* pp = &sm.plane[(pl + m1 - lo) % R][r23];
#pragma unroll
                for (int m2 = 0; m2 < 4; ++m2) {
                    const float* cp = pp + m2 * Cfg::PZ * Cfg::C;
                    const float4 w = rec.cw[4 * m1 + m2];
                    const float lb = rec.lb[4 * m1 + m2];
                    if (VEC == 4) {
                        const ulonglong2 c0 = *reinterpret_cast<const ulonglong2*>(cp);
                        const ulonglong2 c1 = *reinterpret_cast<const ulonglong2*>(cp + Cfg::C);
                        const ulonglong2 c2 = *reinterpret_cast<const ulonglong2*>(cp + 2 * Cfg::C);
                        const ulonglong2 c3 = *reinterpret_cast<const ulonglong2*>(cp + 3 * Cfg::C);
                        fold_pair<MODE>(c0.x, c1.x, c2.x, c3.x, wz, w, lb, acc[0]);
                        fold_pair<MODE>(c0.y, c1.y, c2.y, c3.y, wz, w, lb, acc[NP - 1]);
                    } else {
                        const u64 c0 = *reinterpret_cast<const u64*>(cp);
                        const u64 c1 = *reinterpret_cast<const u64*>(cp + Cfg::C);
                        const u64 c2 = *reinterpret_cast<const u64*>(cp + 2 * Cfg::C);
                        const u64 c3 = *reinterpret_cast<const u64*>(cp + 3 * Cfg::C);
                        fold_pair<MODE>(c0, c1, c2, c3, wz, w, lb, acc[0]);
                    }
                }
            }
        }
        const int col0 = chunk * Cfg::C + lane * VEC;
        if (col0 < 4 * g.pitch4) store_pairs<MODE, NP>(g, acc, ok, e, col0, val, grad, lap, ld);

        if (un < nunits && lane < kRecFloats / 4) reinterpret_cast<float4*>(&sm.rec[warp][cur ^ 1])[lane] = pre;
        __syncwarp();
        cur ^= 1;
        u = un;
    }
    __syncwarp();
    advance(hi, hi + 1);
}

}  // namespace blip
