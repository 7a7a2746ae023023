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
#include "blip_types.h"

namespace blip {

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

// First statement of every kernel of a call: with programmatic stream serialization the kernel
// may already be resident while its predecessor runs; this returns when the predecessor has
// completed and flushed its writes (a no-op for a plain launch).
__device__ __forceinline__ void wait_for_predecessor()
{
    asm volatile("griddepcontrol.wait;" ::: "memory");
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
    wait_for_predecessor();
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

// Work items of the staged kernel (pencil segments), ordered by decreasing electron count — the
// persistent staged kernel takes items from a shared counter, so heavy items first keeps the
// tail short (longest-processing-time-first) — and the reset of that counter.  One CTA of
// kScanThreads threads; `start[b]` = first sorted unit of bin b (global or shared memory),
// `keybuf` = kScanChunk words of shared memory, *nonempty = 0 on entry (shared memory).
__device__ __forceinline__ void order_items(const unsigned* start, int nbins, long long M, const Geom& g, const StagedGeom& sg,
                                            int4* __restrict__ order, int* __restrict__ meta, unsigned* keybuf, int* nonempty)
{
    const int tid = threadIdx.x;
    const unsigned* offs = start;
    if (tid == 0) meta[1] = 0;
    const int nps = sg.nps;
    auto units_of = [&](int i, unsigned& u0, unsigned& u1) {
        const int pencil = i / sg.nseg, segi = i - pencil * sg.nseg;
        const int p0 = segi * sg.seg, p1 = min(p0 + sg.seg, g.n[0]);
        const int bin0 = pencil * g.n[0] + p0, bin1 = pencil * g.n[0] + p1;         // [bin0, bin1)
        u0 = offs[bin0];
        u1 = (bin1 < nbins) ? offs[bin1] : (unsigned)M;
    };
    if (nps > kMaxSortedItems) {
        for (int i = tid; i < nps; i += kScanThreads) {
            unsigned u0, u1;
            units_of(i, u0, u1);
            order[i] = make_int4(i, (int)u0, (int)(u1 - u0), 0);
        }
        if (tid == 0) meta[0] = nps;
        return;
    }
    unsigned* keys = keybuf;
    int n2 = 1;
    while (n2 < nps) n2 <<= 1;
    int mine = 0;
    for (int i = tid; i < n2; i += kScanThreads) {
        unsigned key = 0;
        if (i < nps) {
            unsigned u0, u1;
            units_of(i, u0, u1);
            // sort key: (segment index along the pencil, ascending — with up to 4 segments per pencil),
            // then electron count, descending.  All CTAs then work in the same stretch of the table
            // at a time — neighbouring pencils find each other's halo rows in L2 — and take the
            // heaviest items of that stretch first.
            const unsigned raw = u1 - u0;
            unsigned cnt, pri = 0;
            if (sg.nseg <= 4) { cnt = min(raw, (1u << 17) - 1u); pri = raw ? 3u - (unsigned)(i % sg.nseg) : 0u; }   // empty items stay last
            else cnt = min(raw, (1u << 19) - 1u);
            key = (pri << 30) | (cnt << 13) | (unsigned)i;
            mine += (raw != 0);
        }
        keys[i] = key;
    }
    if (mine) atomicAdd(nonempty, mine);
    __syncthreads();
    if (nps <= kScanThreads) {
        // rank sort: keys are distinct (they end in the item id), so the number of larger keys
        // is the item's place; every thread reads the same key at the same time (a broadcast)
        if (tid < nps) {
            const unsigned key = keys[tid];
            int rank = 0;
            for (int j = 0; j < nps; ++j) rank += (keys[j] > key);
            const int id = (int)(key & 8191u);
            unsigned u0, u1;
            units_of(id, u0, u1);
            order[rank] = make_int4(id, (int)u0, (int)(u1 - u0), 0);
        }
    } else {
        for (int k = 2; k <= n2; k <<= 1)                     // bitonic sort, descending
            for (int j = k >> 1; j > 0; j >>= 1) {
                for (int i = tid; i < n2; i += kScanThreads) {
                    const int x = i ^ j;
                    if (x > i) {
                        const unsigned a = keys[i], b = keys[x];
                        const bool desc = (i & k) == 0;
                        if ((a < b) == desc) { keys[i] = b; keys[x] = a; }
                    }
                }
                __syncthreads();
            }
        for (int i = tid; i < nps; i += kScanThreads) {
            const int id = (int)(keys[i] & 8191u);
            unsigned u0, u1;
            units_of(id, u0, u1);
            order[i] = make_int4(id, (int)u0, (int)(u1 - u0), 0);
        }
    }
    if (tid == 0) meta[0] = *nonempty;
}

// a-4 (2/3): exclusive scan of the histogram into `offs`, one CTA.  `hist` is all zero on entry
// to every call (blipgpu_create clears it once) and this kernel, its only reader, puts it back
// to zero as it reads it: a call leaves no state behind for the next one, so a call captured
// in a CUDA graph can be replayed any number of times.  For the staged path it also orders
// the work items (pencil segments) by decreasing electron count — the persistent staged kernel
// takes items from a shared counter, so heavy items first keeps the tail short
// (longest-processing-time-first) — and resets that counter.
//   offs[b]           start of bin b in the sorted order (the scatter kernels advance it)
//   order[0 .. nps)   {pencil segment id, first unit, units, 0}; units are indices into the
//                     sorted records; heaviest first, in id order if nps > kMaxSortedItems
//   meta[0]           number of leading entries of `order` that hold electrons
//   meta[1]           work counter of the staged kernel, reset to 0
constexpr int kScanChunk = 8 * kScanThreads;                 // bins scanned per pass through shared memory
__global__ void __launch_bounds__(kScanThreads)
scan_kernel(unsigned* __restrict__ hist, unsigned* __restrict__ offs, int nbins, long long M, int staged,
            Geom g, StagedGeom sg, int4* __restrict__ order, int* __restrict__ meta)
{
    __shared__ unsigned buf[kScanChunk];                     // one chunk of the histogram; later the sort keys
    __shared__ unsigned wsum[kScanThreads / 32];
    __shared__ unsigned carry_s;
    __shared__ int nonempty;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    wait_for_predecessor();
    if (tid == 0) { carry_s = 0; nonempty = 0; }
    __syncthreads();
    for (int base = 0; base < nbins; base += kScanChunk) {
        const int n = min(kScanChunk, nbins - base);
#pragma unroll
        for (int k = 0; k < 8; ++k) {                        // coalesced, 8 independent loads per thread
            const int i = tid + k * kScanThreads;
            unsigned v = 0u;
            if (i < n) { v = hist[base + i]; hist[base + i] = 0u; }
            buf[i] = v;
        }
        __syncthreads();
        unsigned v[8], s = 0;
#pragma unroll
        for (int k = 0; k < 8; ++k) { v[k] = buf[8 * tid + k]; s += v[k]; }
        unsigned inc = s;                                    // inclusive scan of the per-thread sums
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const unsigned t = __shfl_up_sync(0xffffffffu, inc, d);
            if (lane >= d) inc += t;
        }
        if (lane == 31) wsum[wid] = inc;
        __syncthreads();
        if (wid == 0) {
            unsigned w = wsum[lane], winc = w;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const unsigned t = __shfl_up_sync(0xffffffffu, winc, d);
                if (lane >= d) winc += t;
            }
            wsum[lane] = winc - w;                           // exclusive prefix of each warp
        }
        __syncthreads();
        unsigned run = carry_s + wsum[wid] + inc - s;        // exclusive prefix of this thread's 8 bins
#pragma unroll
        for (int k = 0; k < 8; ++k) { buf[8 * tid + k] = run; run += v[k]; }
        __syncthreads();
        if (tid == kScanThreads - 1) carry_s = run;
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const int i = tid + k * kScanThreads;
            if (i < n) offs[base + i] = buf[i];
        }
        __syncthreads();
    }
    if (!staged) return;
    // offs[b] = start of bin b (written above by this block, visible after the barrier)
    order_items(offs, nbins, M, g, sg, order, meta, buf, &nonempty);
}

// a-4 (3/3): scatter electron ids into bin order (order inside a bin is arbitrary; the
// results do not depend on it because every electron is evaluated independently).  On return
// offs[b] is the END of bin b in the sorted order.
__global__ void __launch_bounds__(256)
scatter_kernel(const int* __restrict__ bin, unsigned* __restrict__ offs, long long M,
               int* __restrict__ perm)
{
    wait_for_predecessor();
    long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= M) return;
    unsigned slot = atomicAdd(&offs[bin[e]], 1u);
    BLIP_ASSERT((long long)slot < M);
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

// The same record as the staged kernel reads it: instead of the cell index it carries where
// the electron's 4x4x4 block starts in the staged planes of its work item.
struct StagedRec {
    float4 cw[16];
    float  lb[16];
    float  wz[3][4];
    int4   loc;         // {i1 - first plane of the pencil segment (-1: non-finite position),
                        //  byte offset of row (i2, i3) in a staged plane, (i2 % BY) << 8 | (i3 % BZ), electron id}
};
static_assert(sizeof(StagedRec) == sizeof(ElecRec), "one record layout");

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
    lb = __fmul_rn(2.0f, __fmaf_rn(g.Q[4], p10, __fmul_rn(g.Q[5], p01)));
    // diagonal J (MODE 2, where Lb = 0): the gradient weights carry J, so that the accumulators
    // are the Cartesian components and the epilogue has nothing left to multiply
    cw = g.diag ? make_float4(p00, __fmul_rn(g.J[0], p10), __fmul_rn(g.J[4], p01), la) : make_float4(p00, p10, p01, la);
}

// Warp-cooperative a-2 for electron `e` into `rec` (shared memory) from its cell map: lanes
// 0..11 hold (axis a = lane / 4, site m = lane % 4) and are given i_a, f_a of their axis.  `ax`
// is per-warp scratch.  All 32 lanes call it.
__device__ __forceinline__ void warp_weights(const Geom& g, int e, int ia, float fa, bool ok,
                                             float (&ax)[3][3][4], ElecRec& rec, int lane)
{
    if (lane < 12) {
        const int a = lane >> 2, m = lane & 3;
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
        rec.wz[k][m] = (k == 2) ? __fmul_rn(g.Q[2], ax[2][2][m])
                     : (k == 1 && g.diag) ? __fmul_rn(g.J[8], ax[2][1][m]) : ax[2][k][m];
    }
    __syncwarp();
}

// Warp-cooperative a-1 + a-2 for electron `e` into `rec` (shared memory).  All 32 lanes call it.
__device__ __forceinline__ void warp_prepare(const Geom& g, const double* __restrict__ pos, int e,
                                             float (&ax)[3][3][4], ElecRec& rec, int lane)
{
    const double x = pos[3 * (size_t)e], y = pos[3 * (size_t)e + 1], z = pos[3 * (size_t)e + 2];
    int ia = 0; float fa = 0.f; bool ok = true;
    if (lane < 12) ok = cell_map_axis(g, lane >> 2, x, y, z, ia, fa);
    warp_weights(g, e, ia, fa, ok, ax, rec, lane);
}

// a-1 + a-2 for the staged path: the record of electron e (384 B; read back through L2 by the
// staged kernel once per orbital chunk), written to slot s of the sorted order.
__device__ __forceinline__ void write_staged_record(const Geom& g, const StagedGeom& sg, int tile_floats,
                                                    const double* __restrict__ pos, int e, unsigned s,
                                                    float4* recs, int pitch4 = kRecFloats / 4)
{
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
    float4* out = recs + (size_t)s * pitch4;
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
    const float jz = g.diag ? g.J[8] : 1.0f;                 // see column_weights
    out[21] = g.diag ? make_float4(__fmul_rn(jz, ax[2][1][0]), __fmul_rn(jz, ax[2][1][1]), __fmul_rn(jz, ax[2][1][2]),
                                   __fmul_rn(jz, ax[2][1][3]))
                     : make_float4(ax[2][1][0], ax[2][1][1], ax[2][1][2], ax[2][1][3]);
    out[22] = make_float4(__fmul_rn(g.Q[2], ax[2][2][0]), __fmul_rn(g.Q[2], ax[2][2][1]),
                          __fmul_rn(g.Q[2], ax[2][2][2]), __fmul_rn(g.Q[2], ax[2][2][3]));
    // StagedRec::loc: plane within the pencil segment, byte offset of row (i2, i3) in a plane of
    // (by+3) x (bz+3) rows of tile_floats floats
    int pl = -1, off = 0, yz = 0;
    if (ic[0] >= 0 && ic[1] >= 0 && ic[2] >= 0) {            // finite on every axis, as bin_of / bin_kernel decide it
        pl = ic[0] % sg.seg;
        const int y0 = ic[1] % sg.by, z0 = ic[2] % sg.bz;
        off = (y0 * (sg.bz + 3) + z0) * tile_floats * 4;
        yz = (y0 << 8) | z0;                                 // the cell's offset in its pencil, for the tensor-core kernel
    }
    out[23] = make_float4(__int_as_float(pl), __int_as_float(off), __int_as_float(yz), __int_as_float(e));
}

// a-4 (3/3) for the staged path, three-kernel form: one thread per electron takes its slot in
// bin order and writes the electron's record there.  On return offs[b] is the END of bin b.
__global__ void __launch_bounds__(128)
scatter_prep_kernel(Geom g, StagedGeom sg, int tile_floats, const double* __restrict__ pos,
                    const int* __restrict__ bin, unsigned* __restrict__ offs, long long M,
                    float4* __restrict__ recs)
{
    wait_for_predecessor();
    const long long el = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (el >= M) return;
    const int e = (int)el;
    const unsigned s = atomicAdd(&offs[bin[e]], 1u);
    BLIP_ASSERT((long long)s < M);
    write_staged_record(g, sg, tile_floats, pos, e, s, recs);
}

// ---------------------------------------------------------------------------------------
// a-4 in ONE launch (cooperative: every CTA is resident, so the CTAs can wait for one another):
//   phase 1   every electron: cell -> bin, count[bin] += 1 (and the optional cell output);
//   barrier   over the grid (arrival counter + generation word in global memory);
//   phase 2   every CTA scans the whole histogram into its own shared memory (a few thousand
//             bins: cheaper than a second barrier around a one-CTA scan), then every electron
//             takes slot start[bin] + cursor[bin]++ and writes its record (staged path) or its
//             index (direct path) there; CTA 0 orders the work items instead.
// The three launches of the other form (bin, scan, scatter: ~31 us of a 480 us TiO2 step, mostly
// launch-to-launch latency) become one of ~12 us.
//
// State between calls, all on the device, so that a captured call can be replayed: the counter
// arrays come in two groups {count, cursor}; a call uses the group selected by the parity of
// the barrier generation, which it finds all zero, and zeroes the other group, which the
// previous call left dirty.  gstate = {arrivals, generation}.
// Shared memory: (nbins + 1) words for the scan, dynamic.
// ---------------------------------------------------------------------------------------
template <bool STAGED>
__global__ void __launch_bounds__(kScanThreads, 1)
group_kernel(Geom g, StagedGeom sg, int tile_floats, const double* __restrict__ pos, long long M,
             unsigned* __restrict__ counters /* [4][nalloc] */, int nalloc, int nbins, unsigned* __restrict__ gstate,
             int4* __restrict__ order, int* __restrict__ meta, float4* __restrict__ recs, int* __restrict__ perm,
             int* __restrict__ cell, int nstage)
{
    extern __shared__ __align__(16) unsigned start[];        // [nbins + 1] exclusive scan of the counts, then record staging
    __shared__ unsigned wsum[kScanThreads / 32];
    __shared__ unsigned keybuf[STAGED ? kScanChunk : 1];   // CTA 0 of the staged form sorts the work items here
    __shared__ int nonempty;
    __shared__ unsigned gen_s;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    if (tid == 0) { gen_s = *reinterpret_cast<volatile unsigned*>(gstate + 1); nonempty = 0; }
    __syncthreads();
    const unsigned gen = gen_s;
    unsigned* count = counters + (size_t)(2 * (gen & 1u)) * nalloc;
    unsigned* cursor = count + nalloc;
    unsigned* stale = counters + (size_t)(2 * ((gen & 1u) ^ 1u)) * nalloc;     // both arrays of the other group
    const long long nthreads = (long long)gridDim.x * kScanThreads;
    const long long gtid = (long long)blockIdx.x * kScanThreads + tid;

    auto bin_of = [&](long long e, int (&ic)[3]) -> int {
        const double x = pos[3 * e], y = pos[3 * e + 1], z = pos[3 * e + 2];
        float f;
        bool ok = cell_map_axis(g, 0, x, y, z, ic[0], f);
        ok = cell_map_axis(g, 1, x, y, z, ic[1], f) && ok;
        ok = cell_map_axis(g, 2, x, y, z, ic[2], f) && ok;
        if (!ok) { ic[0] = ic[1] = ic[2] = -1; return 0; }
        return STAGED ? staged_key(g, sg, ic[0], ic[1], ic[2]) : brick_of(g, ic[0], ic[1], ic[2]);
    };
    // ---- phase 1 (an equal share of the electrons per CTA)
    {
        const long long share1 = (M + gridDim.x - 1) / gridDim.x;
        const long long a0 = (long long)blockIdx.x * share1, a1 = min(a0 + share1, M);
        for (long long e = a0 + tid; e < a1; e += kScanThreads) {
            int ic[3];
            const int b = bin_of(e, ic);
            BLIP_ASSERT(b >= 0 && b < nbins);
            if (cell) { cell[3 * e] = ic[0]; cell[3 * e + 1] = ic[1]; cell[3 * e + 2] = ic[2]; }
            atomicAdd(&count[b], 1u);
        }
    }
    for (long long i = gtid; i < 2LL * nalloc; i += nthreads) stale[i] = 0u;
    // ---- grid barrier
    __syncthreads();
    if (tid == 0) {
        __threadfence();
        const unsigned arrived = atomicAdd(gstate, 1u);
        if (arrived == gridDim.x - 1) {
            *reinterpret_cast<volatile unsigned*>(gstate) = 0u;
            __threadfence();
            atomicAdd(gstate + 1, 1u);
        } else {
            while (*reinterpret_cast<volatile unsigned*>(gstate + 1) == gen) __nanosleep(40);
        }
        __threadfence();
    }
    __syncthreads();
    // ---- phase 2: exclusive scan of count[0 .. nbins) into shared memory (every CTA, redundantly)
    for (int base = 0; base < nbins; base += 8 * kScanThreads) {      // 8 independent loads per thread in flight
        unsigned v[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const int i = base + tid + k * kScanThreads;
            v[k] = (i < nbins) ? __ldcg(count + i) : 0u;
        }
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const int i = base + tid + k * kScanThreads;
            if (i < nbins) start[i] = v[k];
        }
    }
    __syncthreads();
    const int per = ((nbins + kScanThreads - 1) / kScanThreads) | 1;     // odd: consecutive threads start in different banks
    const int b0 = min(tid * per, nbins), b1 = min(b0 + per, nbins);
    unsigned sum = 0;
    for (int b = b0; b < b1; ++b) { const unsigned v = start[b]; start[b] = sum; sum += v; }
    unsigned inc = sum;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const unsigned t = __shfl_up_sync(0xffffffffu, inc, d);
        if (lane >= d) inc += t;
    }
    if (lane == 31) wsum[wid] = inc;
    __syncthreads();
    if (wid == 0) {
        unsigned w = wsum[lane], winc = w;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const unsigned t = __shfl_up_sync(0xffffffffu, winc, d);
            if (lane >= d) winc += t;
        }
        wsum[lane] = winc - w;
    }
    __syncthreads();
    const unsigned toff = wsum[wid] + inc - sum;
    for (int b = b0; b < b1; ++b) start[b] += toff;
    if (tid == 0) start[nbins] = (unsigned)M;
    __syncthreads();
    if (STAGED && blockIdx.x == 0) {                         // CTA 0: the work items of the staged kernel
        order_items(start, nbins + 1, M, g, sg, order, meta, keybuf, &nonempty);
        if (gridDim.x > 1) return;
    }
    // ---- phase 2: scatter (CTAs 1.. when CTA 0 orders the items), an equal share of the electrons per CTA
    const int first = (STAGED && gridDim.x > 1) ? 1 : 0;
    const long long nc = (long long)gridDim.x - first;
    const long long share = (M + nc - 1) / nc;
    const long long e0 = (long long)(blockIdx.x - first) * share, e1 = min(e0 + share, M);
    if (STAGED) {
        // A thread per electron (position load, fp64 cell map, slot atomic, weights: every electron
        // of the round in flight at once) builds its record in shared memory — 24 float4 per thread
        // straight to global memory would be 24 stores of 32 scattered 16-byte pieces per warp, and
        // took 9 us — and then the whole CTA copies the records out, 384 contiguous bytes each.
        constexpr int RW = kRecFloats / 4 + 1;               // float4 per staged record: 24 + 1 pad (bank spread)
        float4* stage = reinterpret_cast<float4*>(start + (((size_t)nbins + 1 + 3) & ~(size_t)3));
        unsigned* slots = reinterpret_cast<unsigned*>(stage + (size_t)nstage * RW);
        for (long long r0 = e0; r0 < e1; r0 += nstage) {
            const int nr = (int)min((long long)nstage, e1 - r0);
            for (int r = tid; r < nr; r += kScanThreads) {
                const long long e = r0 + r;
                int ic[3];
                const int b = bin_of(e, ic);
                const unsigned slot = start[b] + atomicAdd(&cursor[b], 1u);
                BLIP_ASSERT(slot < start[b + 1] && (long long)slot < M);
                slots[r] = slot;
                write_staged_record(g, sg, tile_floats, pos, (int)e, (unsigned)r, stage, RW);
            }
            __syncthreads();
            for (int i = tid; i < nr * (kRecFloats / 4); i += kScanThreads) {
                const int r = i / (kRecFloats / 4), q = i - r * (kRecFloats / 4);
                recs[(size_t)slots[r] * (kRecFloats / 4) + q] = stage[(size_t)r * RW + q];
            }
            __syncthreads();
        }
    } else {
        for (long long e = e0 + tid; e < e1; e += kScanThreads) {
            int ic[3];
            const int b = bin_of(e, ic);
            const unsigned slot = start[b] + atomicAdd(&cursor[b], 1u);
            BLIP_ASSERT(slot < start[b + 1] && (long long)slot < M);
            perm[slot] = (int)e;
        }
    }
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
__device__ __forceinline__ void set_nan(PairAcc& a)         // outputs of a non-finite position (R17)
{
    a.val = a.t1 = a.t2 = a.t3 = a.lp = 0x7fc000007fc00000ull;
}

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
        if (MODE == 1) l = fma2(b, dup2(lb), l);             // MODE 2: Q02 = Q12 = 0, so Lb = 0
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
// MODE 2: J is diagonal (lattice vectors along the Cartesian axes).
template <int MODE, int NP>
__device__ __forceinline__ void store_pairs(const Geom& g, const PairAcc (&acc)[NP], int e,
                                            int col0, float* __restrict__ val, float* __restrict__ grad,
                                            float* __restrict__ lap, long long ld)
{
    float v[2 * NP], gx[2 * NP], gy[2 * NP], gz[2 * NP], lp[2 * NP];
#pragma unroll
    for (int p = 0; p < NP; ++p) {
        const float2 s = unpack2(acc[p].val);
        v[2 * p] = s.x; v[2 * p + 1] = s.y;
        if (MODE != 0) {
            const float2 a = unpack2(acc[p].t1), b = unpack2(acc[p].t2), c = unpack2(acc[p].t3);
            const float2 l = unpack2(acc[p].lp);
            const float ta[2] = {a.x, a.y}, tb[2] = {b.x, b.y}, tc[2] = {c.x, c.y};
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                if (MODE == 2) {                             // J is already in the weights
                    gx[2 * p + h] = ta[h];
                    gy[2 * p + h] = tb[h];
                    gz[2 * p + h] = tc[h];
                } else {
                    gx[2 * p + h] = __fmaf_rn(g.J[0], ta[h], __fmaf_rn(g.J[3], tb[h], __fmul_rn(g.J[6], tc[h])));
                    gy[2 * p + h] = __fmaf_rn(g.J[1], ta[h], __fmaf_rn(g.J[4], tb[h], __fmul_rn(g.J[7], tc[h])));
                    gz[2 * p + h] = __fmaf_rn(g.J[2], ta[h], __fmaf_rn(g.J[5], tb[h], __fmul_rn(g.J[8], tc[h])));
                }
            }
            lp[2 * p] = l.x; lp[2 * p + 1] = l.y;
        }
    }
    const size_t o = (size_t)e * (size_t)ld + (size_t)col0;
    const size_t og = (size_t)e * 3 * (size_t)ld + (size_t)col0;
    BLIP_ASSERT(e >= 0 && (long long)e < g.M && col0 >= 0 && (long long)col0 + 2 * NP <= ld);
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

// a-5 for complex orbitals with a Bloch phase (the paper's orbitals are
// complex): real channels (2m, 2m+1) form u_m = S_2m + i S_2m+1 and the output is
//     psi_m = e^{i k_m.r} u_m,   grad psi_m = e^{i k_m.r} (grad u_m + i k_m u_m),
//     laplace psi_m = e^{i k_m.r} (laplace u_m + 2 i k_m.grad u_m - |k_m|^2 u_m)
// stored as interleaved (re, im) fp32 in the places of the two real channels.  A lane's 4
// orbitals are 2 complex ones (acc[0], acc[1]); the phase k.r is taken in fp64, brought to
// (-1, 1] half-turns exactly, and only then rounded to fp32 for sincospi, so its error does not
// grow with |k.r| (reading R8a).  Once per electron x complex orbital.
__device__ __forceinline__ void bloch_phase(const double* __restrict__ pos, const double* __restrict__ kvec, int e, int m,
                                            int ncomplex, float& c, float& s, float (&kf)[3], float& k2)
{
    double k0 = 0.0, k1 = 0.0, k2d = 0.0;
    if (m < ncomplex) { k0 = __ldg(kvec + 3 * (size_t)m); k1 = __ldg(kvec + 3 * (size_t)m + 1); k2d = __ldg(kvec + 3 * (size_t)m + 2); }
    const double x = __ldg(pos + 3 * (size_t)e), y = __ldg(pos + 3 * (size_t)e + 1), z = __ldg(pos + 3 * (size_t)e + 2);
    const double theta = fma(k2d, z, fma(k1, y, k0 * x));
    double t = theta * 0.31830988618379067154;              // half-turns: theta / pi
    t = fma(-2.0, rint(0.5 * t), t);                         // exact: t in [-1, 1]
    sincospif((float)t, &s, &c);
    kf[0] = (float)k0; kf[1] = (float)k1; kf[2] = (float)k2d;
    k2 = (float)fma(k2d, k2d, fma(k1, k1, k0 * k0));
}

template <int MODE>
__device__ __forceinline__ void store_pairs_complex(const Geom& g, const PairAcc (&acc)[2], int e, int col0,
                                                    const double* __restrict__ pos, const double* __restrict__ kvec,
                                                    float* __restrict__ val, float* __restrict__ grad,
                                                    float* __restrict__ lap, long long ld)
{
    float v[4], gx[4], gy[4], gz[4], lp[4];
#pragma unroll
    for (int p = 0; p < 2; ++p) {
        float c, s, k[3], k2;
        bloch_phase(pos, kvec, e, (col0 >> 1) + p, g.L >> 1, c, s, k, k2);
        const float2 u = unpack2(acc[p].val);                // u = u.x + i u.y
        v[2 * p] = __fmaf_rn(c, u.x, -__fmul_rn(s, u.y));
        v[2 * p + 1] = __fmaf_rn(s, u.x, __fmul_rn(c, u.y));
        if (MODE != 0) {
            const float2 a = unpack2(acc[p].t1), b = unpack2(acc[p].t2), d = unpack2(acc[p].t3), l = unpack2(acc[p].lp);
            float gr[3], gi[3];                              // Cartesian gradient of u: real and imaginary channel
            if (MODE == 2) {
                gr[0] = a.x; gr[1] = b.x; gr[2] = d.x; gi[0] = a.y; gi[1] = b.y; gi[2] = d.y;
            } else {
#pragma unroll
                for (int i = 0; i < 3; ++i) {
                    gr[i] = __fmaf_rn(g.J[i], a.x, __fmaf_rn(g.J[3 + i], b.x, __fmul_rn(g.J[6 + i], d.x)));
                    gi[i] = __fmaf_rn(g.J[i], a.y, __fmaf_rn(g.J[3 + i], b.y, __fmul_rn(g.J[6 + i], d.y)));
                }
            }
            float* const out[3] = {gx, gy, gz};
#pragma unroll
            for (int i = 0; i < 3; ++i) {                    // grad u + i k u
                const float re = __fmaf_rn(-k[i], u.y, gr[i]), im = __fmaf_rn(k[i], u.x, gi[i]);
                out[i][2 * p] = __fmaf_rn(c, re, -__fmul_rn(s, im));
                out[i][2 * p + 1] = __fmaf_rn(s, re, __fmul_rn(c, im));
            }
            const float kgr = __fmaf_rn(k[0], gr[0], __fmaf_rn(k[1], gr[1], __fmul_rn(k[2], gr[2])));
            const float kgi = __fmaf_rn(k[0], gi[0], __fmaf_rn(k[1], gi[1], __fmul_rn(k[2], gi[2])));
            const float re = __fmaf_rn(-k2, u.x, __fmaf_rn(-2.0f, kgi, l.x));      // laplace u + 2 i k.grad u - k^2 u
            const float im = __fmaf_rn(-k2, u.y, __fmaf_rn(2.0f, kgr, l.y));
            lp[2 * p] = __fmaf_rn(c, re, -__fmul_rn(s, im));
            lp[2 * p + 1] = __fmaf_rn(s, re, __fmul_rn(c, im));
        }
    }
    const size_t o = (size_t)e * (size_t)ld + (size_t)col0;
    const size_t og = (size_t)e * 3 * (size_t)ld + (size_t)col0;
    BLIP_ASSERT(e >= 0 && (long long)e < g.M && col0 >= 0 && (long long)col0 + 4 <= ld);
    st_stream4(val + o, v[0], v[1], v[2], v[3]);
    if (MODE != 0) {
        st_stream4(grad + og, gx[0], gx[1], gx[2], gx[3]);
        st_stream4(grad + og + ld, gy[0], gy[1], gy[2], gy[3]);
        st_stream4(grad + og + 2 * ld, gz[0], gz[1], gz[2], gz[3]);
        st_stream4(lap + o, lp[0], lp[1], lp[2], lp[3]);
    }
}

// Contraction epilogue (§VI.D, Eq. 11): instead of
// storing the orbitals of electron e, contract them with the caller's vector d_e (column of
// the inverse Slater matrix in the paper's use):
//     out[e][0] += sum_l psi_l d_l,  out[e][1..3] += sum_l grad psi_l d_l,  out[e][4] += sum_l lap psi_l d_l
// over the 2 NP orbitals of this lane (dq: their d values, zero past the last orbital), then
// over the warp; one atomic add per quantity and (electron, orbital tile).
template <int MODE, int NP>
__device__ __forceinline__ void contract_pairs(const Geom& g, const PairAcc (&acc)[NP], const float (&dq)[2 * NP],
                                               float (&sum)[5])
{
#pragma unroll
    for (int p = 0; p < NP; ++p) {
        const float2 v = unpack2(acc[p].val);
        sum[0] = __fmaf_rn(v.x, dq[2 * p], __fmaf_rn(v.y, dq[2 * p + 1], sum[0]));
        if (MODE != 0) {
            const float2 a = unpack2(acc[p].t1), b = unpack2(acc[p].t2), c = unpack2(acc[p].t3), l = unpack2(acc[p].lp);
            sum[1] = __fmaf_rn(a.x, dq[2 * p], __fmaf_rn(a.y, dq[2 * p + 1], sum[1]));
            sum[2] = __fmaf_rn(b.x, dq[2 * p], __fmaf_rn(b.y, dq[2 * p + 1], sum[2]));
            sum[3] = __fmaf_rn(c.x, dq[2 * p], __fmaf_rn(c.y, dq[2 * p + 1], sum[3]));
            sum[4] = __fmaf_rn(l.x, dq[2 * p], __fmaf_rn(l.y, dq[2 * p + 1], sum[4]));
        }
    }
}
// Grid-space gradient -> Cartesian on the lane's partial sums (linear, so it commutes with the
// sums over lanes and tiles), then the five sums are added over the warp with 9 shuffles: at
// each of the first three steps a lane hands half of its values to its partner and keeps the
// other half, so that lane 4 q ends up with the warp total of quantity q; one atomic add per
// quantity into out[e][0..4].
template <int MODE>
__device__ __forceinline__ void contract_flush(const Geom& g, float (&sum)[5], int e, float* __restrict__ out, int lane)
{
    if (MODE == 0) {
        float r = sum[0];
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) r += __shfl_xor_sync(0xffffffffu, r, d);
        if (lane == 0) atomicAdd(out + 8 * (size_t)e, r);
        return;
    }
    float v[8];
    v[0] = sum[0];
    if (MODE == 2) {                                         // J is already in the weights
        v[1] = sum[1]; v[2] = sum[2]; v[3] = sum[3];
    } else {
        v[1] = __fmaf_rn(g.J[0], sum[1], __fmaf_rn(g.J[3], sum[2], __fmul_rn(g.J[6], sum[3])));
        v[2] = __fmaf_rn(g.J[1], sum[1], __fmaf_rn(g.J[4], sum[2], __fmul_rn(g.J[7], sum[3])));
        v[3] = __fmaf_rn(g.J[2], sum[1], __fmaf_rn(g.J[5], sum[2], __fmul_rn(g.J[8], sum[3])));
    }
    v[4] = sum[4]; v[5] = v[6] = v[7] = 0.f;
    const bool h16 = lane & 16, h8 = lane & 8, h4 = lane & 4;
    float w[4], x[2];
#pragma unroll
    for (int k = 0; k < 4; ++k) {                            // keep quantity k + 4 [lane bit 4]
        const float give = h16 ? v[k] : v[k + 4], keep = h16 ? v[k + 4] : v[k];
        w[k] = keep + __shfl_xor_sync(0xffffffffu, give, 16);
    }
#pragma unroll
    for (int k = 0; k < 2; ++k) {                            // ... + 2 [bit 3]
        const float give = h8 ? w[k] : w[k + 2], keep = h8 ? w[k + 2] : w[k];
        x[k] = keep + __shfl_xor_sync(0xffffffffu, give, 8);
    }
    const float give = h4 ? x[0] : x[1], keep = h4 ? x[1] : x[0];
    float r = keep + __shfl_xor_sync(0xffffffffu, give, 4);  // ... + [bit 2]: quantity lane >> 2
    r += __shfl_xor_sync(0xffffffffu, r, 2);
    r += __shfl_xor_sync(0xffffffffu, r, 1);
    if ((lane & 3) == 0 && lane < 20) atomicAdd(out + 8 * (size_t)e + (lane >> 2), r);
}
// d values of the 4 orbitals starting at column col0 of electron e, zero at and past column L
__device__ __forceinline__ float4 ldg_dvec(const float* __restrict__ dvec, long long ldd, int e, int col0)
{
    return __ldg(reinterpret_cast<const float4*>(dvec + (size_t)e * (size_t)ldd + col0));
}
__device__ __forceinline__ void mask_dvec(const float4& v, int col0, int L, float (&dq)[4])
{
    dq[0] = col0 < L ? v.x : 0.f; dq[1] = col0 + 1 < L ? v.y : 0.f;
    dq[2] = col0 + 2 < L ? v.z : 0.f; dq[3] = col0 + 3 < L ? v.w : 0.f;
}
__device__ __forceinline__ void load_dvec(const float* __restrict__ dvec, long long ldd, int e, int col0, int L,
                                          float (&dq)[4])
{
    mask_dvec(ldg_dvec(dvec, ldd, e, col0), col0, L, dq);
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
                                            unsigned colrow, int pitch4, ulonglong2 (&buf)[4 * NQ],
                                            long long nrows_checked = 0)
{
    const unsigned base = colrow * (unsigned)pitch4;
    BLIP_ASSERT((unsigned long long)colrow + 3 < (unsigned long long)nrows_checked);
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
                   long long ld, const float* __restrict__ dvec, long long ldd, float* __restrict__ cout,
                   int* __restrict__ cell_out, const double* __restrict__ kvec)
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
    if (!ok) {
#pragma unroll
        for (int j = 0; j < NQ; ++j) { set_nan(acc[j][0]); set_nan(acc[j][1]); }
    } else {
        float wz[3][4];
#pragma unroll
        for (int k = 0; k < 3; ++k)
#pragma unroll
            for (int m = 0; m < 4; ++m) wz[k][m] = ws.rec.wz[k][m];
        // padded row of site (m1, m2, m3 = 0): ((i1 + m1) np2 + (i2 + m2)) np3 + i3
        const unsigned row0 = ((unsigned)i1 * g.np[1] + i2) * g.np[2] + i3;
        const unsigned s1 = (unsigned)g.np[1] * g.np[2], s2 = (unsigned)g.np[2];
        ulonglong2 buf0[4 * NQ], buf1[4 * NQ];
        load_column<NQ>(table, off, row0, g.pitch4, buf0, (long long)g.np[0] * g.np[1] * g.np[2]);
#pragma unroll 1
        for (int c = 0; c < 16; c += 2) {
            const unsigned r1 = row0 + (c >> 2) * s1 + ((c + 1) & 3) * s2;
            load_column<NQ>(table, off, r1, g.pitch4, buf1, (long long)g.np[0] * g.np[1] * g.np[2]);
            fold_column<MODE, NQ>(ws.rec, c, wz, buf0, acc);
            if (c + 2 < 16) {
                const unsigned r2 = row0 + ((c + 2) >> 2) * s1 + ((c + 2) & 3) * s2;
                load_column<NQ>(table, off, r2, g.pitch4, buf0, (long long)g.np[0] * g.np[1] * g.np[2]);
            }
            fold_column<MODE, NQ>(ws.rec, c + 1, wz, buf1, acc);
        }
    }
    if (dvec) {
        float sum[5] = {0.f, 0.f, 0.f, 0.f, 0.f};
#pragma unroll
        for (int j = 0; j < NQ; ++j)
            if (quad[j] < g.pitch4) {
                float dq[4];
                load_dvec(dvec, ldd, e, 4 * quad[j], g.L, dq);
                contract_pairs<MODE, 2>(g, acc[j], dq, sum);
            }
        contract_flush<MODE>(g, sum, e, cout, lane);
        return;
    }
    if (kvec) {                                              // complex orbitals (blipgpu_eval_complex)
#pragma unroll
        for (int j = 0; j < NQ; ++j)
            if (quad[j] < g.pitch4) store_pairs_complex<MODE>(g, acc[j], e, 4 * quad[j], pos, kvec, val, grad, lap, ld);
        return;
    }
#pragma unroll
    for (int j = 0; j < NQ; ++j)
        if (quad[j] < g.pitch4) store_pairs<MODE, 2>(g, acc[j], e, 4 * quad[j], val, grad, lap, ld);
}

// ---------------------------------------------------------------------------------------
// Split kernel, for small batches (the paper's particle-by-particle end of the sweep,
// PAPER.md:268 kernel (1), where a call is a handful of electrons and the cost is latency):
// CTA = (electron, 128 orbitals), 4 warps; warp m1 takes the 16 rows of plane i1 + m1.  Every
// warp maps the position to its cell itself (a-1, fp64) and issues its 16 loads at once — one
// memory round trip, started as early as possible — and only then computes the weights (a-2),
// while the loads are in flight; the four partial sums are added in plane order through shared
// memory.  One block barrier per CTA.
// ---------------------------------------------------------------------------------------
template <int MODE>
__global__ void __launch_bounds__(128)
eval_split_kernel(Geom g, const float4* __restrict__ table4, const double* __restrict__ pos,
                  const int* __restrict__ perm, long long M, float* __restrict__ val, float* __restrict__ grad, float* __restrict__ lap,
                  long long ld, const float* __restrict__ dvec, long long ldd, float* __restrict__ cout,
                  int* __restrict__ cell_out, const double* __restrict__ kvec)
{
    __shared__ DirectScratch wsw[4];                         // one per warp
    __shared__ u64 part[3][5 * 2][32];                       // partial sums of warps 1..3
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int e = perm ? perm[blockIdx.x] : (int)blockIdx.x;
    const ulonglong2* __restrict__ table = reinterpret_cast<const ulonglong2*>(table4);
    const int quad = blockIdx.y * 32 + lane;
    const unsigned off[1] = {(unsigned)min(quad, g.pitch4 - 1)};
    DirectScratch& ws = wsw[warp];
    // a-1: lanes 0..11 = (axis lane / 4, site lane % 4); lanes 0, 4, 8 hold the three cell indices
    const double x = pos[3 * (size_t)e], y = pos[3 * (size_t)e + 1], z = pos[3 * (size_t)e + 2];
    int ia = 0; float fa = 0.f; bool okl = true;
    if (lane < 12) okl = cell_map_axis(g, lane >> 2, x, y, z, ia, fa);
    const int i1 = __shfl_sync(0xffffffffu, ia, 0), i2 = __shfl_sync(0xffffffffu, ia, 4), i3 = __shfl_sync(0xffffffffu, ia, 8);
    const bool ok = (i1 | i2 | i3) >= 0;
    if (cell_out && blockIdx.y == 0 && warp == 0 && lane < 12 && (lane & 3) == 0) cell_out[3 * (size_t)e + (lane >> 2)] = ok ? ia : -1;

    PairAcc acc[1][2];
#pragma unroll
    for (int h = 0; h < 2; ++h) acc[0][h].val = acc[0][h].t1 = acc[0][h].t2 = acc[0][h].t3 = acc[0][h].lp = 0ull;
    ulonglong2 buf[4][4];
    if (ok) {                                                // all 16 rows of plane i1 + warp in flight
        const unsigned s2 = (unsigned)g.np[2];
        const unsigned row0 = ((unsigned)(i1 + warp) * g.np[1] + i2) * g.np[2] + i3;
#pragma unroll
        for (int m2 = 0; m2 < 4; ++m2) load_column<1>(table, off, row0 + m2 * s2, g.pitch4, buf[m2], (long long)g.np[0] * g.np[1] * g.np[2]);
    }
    warp_weights(g, e, ia, fa, okl, ws.ax, ws.rec, lane);    // a-2, while the loads are in flight
    if (ok) {
        float wz[3][4];
#pragma unroll
        for (int k = 0; k < 3; ++k)
#pragma unroll
            for (int m = 0; m < 4; ++m) wz[k][m] = ws.rec.wz[k][m];
#pragma unroll
        for (int m2 = 0; m2 < 4; ++m2) fold_column<MODE, 1>(ws.rec, 4 * warp + m2, wz, buf[m2], acc);
    }
    if (warp > 0) {
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            part[warp - 1][5 * h + 0][lane] = acc[0][h].val;
            if (MODE != 0) {
                part[warp - 1][5 * h + 1][lane] = acc[0][h].t1; part[warp - 1][5 * h + 2][lane] = acc[0][h].t2;
                part[warp - 1][5 * h + 3][lane] = acc[0][h].t3; part[warp - 1][5 * h + 4][lane] = acc[0][h].lp;
            }
        }
    }
    __syncthreads();
    if (warp != 0) return;
    if (!ok) { set_nan(acc[0][0]); set_nan(acc[0][1]); }
    else {
        const u64 one = dup2(1.0f);
#pragma unroll
        for (int w = 0; w < 3; ++w)
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                acc[0][h].val = fma2(part[w][5 * h + 0][lane], one, acc[0][h].val);
                if (MODE != 0) {
                    acc[0][h].t1 = fma2(part[w][5 * h + 1][lane], one, acc[0][h].t1);
                    acc[0][h].t2 = fma2(part[w][5 * h + 2][lane], one, acc[0][h].t2);
                    acc[0][h].t3 = fma2(part[w][5 * h + 3][lane], one, acc[0][h].t3);
                    acc[0][h].lp = fma2(part[w][5 * h + 4][lane], one, acc[0][h].lp);
                }
            }
    }
    if (dvec) {
        float sum[5] = {0.f, 0.f, 0.f, 0.f, 0.f};
        if (quad < g.pitch4) {
            float dq[4];
            load_dvec(dvec, ldd, e, 4 * quad, g.L, dq);
            contract_pairs<MODE, 2>(g, acc[0], dq, sum);
        }
        contract_flush<MODE>(g, sum, e, cout, lane);
        return;
    }
    if (quad >= g.pitch4) return;
    if (kvec) store_pairs_complex<MODE>(g, acc[0], e, 4 * quad, pos, kvec, val, grad, lap, ld);
    else store_pairs<MODE, 2>(g, acc[0], e, 4 * quad, val, grad, lap, ld);
}

// ---------------------------------------------------------------------------------------
// Staged kernel (persistent: one CTA per SM).  A work item is (pencil segment, orbital chunk
// of C = 32*VEC orbitals): the electrons of the segment, sorted by cell plane i1, are its
// units; the table planes p1 = lo .. hi+3 of the pencil's (BY+3) x (BZ+3) cross-section slide
// through a ring of R shared-memory slots, one TMA box per plane.
//
//   producer warp   takes items from the global counter meta[1] (heaviest segment first:
//                   `order`), publishes their descriptors through a 3-entry queue — item k+1 as
//                   soon as the last plane of item k is issued, so that consumers can prefetch
//                   across the item boundary — and issues the planes of item after item into
//                   the ring: the planes of the next item arrive while the consumers finish
//                   the current one;
//   NW consumers    warp w takes units w, w+NW, ... of every item.  Planes carry a CTA-wide
//                   sequence number; every consumer waits for and releases every plane in
//                   sequence order (full / empty barriers, NW arrivals per plane), so barrier
//                   phases follow from the sequence number alone.
//
// What bounds it (ncu + in-kernel timers, profiles/): while the warps run the 64-row loop the
// shared-memory pipe (32 KB of coefficient reads per unit, 128 B/clk/SM) and the issue ports
// (a packed FMA holds its scheduler's port for two cycles) are both > 90 % busy; the rest of
// the time goes to waiting for planes (TMA latency under load) and per-unit bookkeeping.
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ ulonglong2 lds128(unsigned addr)
{
    ulonglong2 v; asm volatile("ld.shared.v2.b64 {%0, %1}, [%2];" : "=l"(v.x), "=l"(v.y) : "r"(addr)); return v;
}
__device__ __forceinline__ u64 lds64(unsigned addr)
{
    u64 v; asm volatile("ld.shared.b64 %0, [%1];" : "=l"(v) : "r"(addr)); return v;
}
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
// arrival by lane 0 only, predicated inside the instruction (no branch, no reconvergence point)
__device__ __forceinline__ void mbar_arrive_lane0(unsigned bar, int lane)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.eq.s32 p, %1, 0;\n\t"
        "@p mbarrier.arrive.shared::cta.b64 _, [%0];\n\t}"
        :: "r"(bar), "r"(lane) : "memory");
}
__device__ __forceinline__ bool mbar_test(unsigned bar, unsigned parity)
{
    unsigned done;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done) : "r"(bar), "r"(parity) : "memory");
    return done != 0;
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
// Producer-side wait: the producer has nothing else to do, so it backs off between polls and
// leaves the issue slots of its scheduler to the consumer warps that share it.
__device__ __forceinline__ void mbar_wait_backoff(unsigned bar, unsigned parity)
{
    unsigned done = 0;
    while (true) {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(done) : "r"(bar), "r"(parity) : "memory");
        if (done) break;
        __nanosleep(64);
    }
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

constexpr int kItemQueue = 3;              // item descriptors in flight per CTA: finishing, current, next

__device__ __forceinline__ void tma_prefetch_4d(const CUtensorMap* tmap, int c0, int c1, int c2, int c3)
{
    asm volatile("cp.async.bulk.prefetch.tensor.4d.L2.global.tile [%0, {%1, %2, %3, %4}];"
                 :: "l"(reinterpret_cast<uint64_t>(tmap)), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}

struct WorkItem {
    int nplanes;        // planes of this item (0: no electrons, -1: no more work)
    int chunk;          // orbital chunk
    int by, bz;         // pencil coordinates
    int lo;             // first cell plane
    unsigned seq0;      // CTA-wide sequence number of plane lo
    unsigned u0;        // first unit (index into the sorted records)
    unsigned nunits;
};

template <int VEC, int BY, int BZ, int R, int NW>
struct StagedCfg {
    static constexpr int C = 32 * VEC;                       // orbitals per tile row
    static constexpr int PY = BY + 3, PZ = BZ + 3;
    static constexpr int PLANE_FLOATS = PY * PZ * C;
    static constexpr int PLANE_BYTES = PLANE_FLOATS * 4;
    static constexpr int THREADS = (NW + 1) * 32;
    struct Smem {
        alignas(128) float plane[R][PLANE_FLOATS];
        alignas(16) ElecRec rec[NW];                         // one record per consumer warp; the next one waits in registers
        alignas(16) WorkItem item[kItemQueue];
        alignas(8) u64 full[R];
        alignas(8) u64 empty[R];
        alignas(8) u64 ifull[kItemQueue];
        alignas(8) u64 iempty[kItemQueue];
    };
};

// Deadlock freedom of the two queues.  The producer takes and publishes item k+1 once every
// plane of item k is issued; for that it needs ring slots, which consumers give back as they
// move through item k, and the descriptor slot of item k-2, which every consumer gives back
// when it leaves item k-2.  A consumer waits for the descriptor of item k+1 only after it has
// left item k and released all of its planes; while it still works on a unit of item k it
// only looks whether the descriptor is there yet (to prefetch its first record of item k+1).
// So whatever a consumer waits for never depends on something that consumer still holds.
// EPI: what happens to a unit's results (a-5): 0 stored, 1 contracted with d (blipgpu_eval_contract),
// 2 stored as complex orbitals with a Bloch phase (blipgpu_eval_complex).
constexpr int kEpiStore = 0, kEpiContract = 1, kEpiComplex = 2;
template <int MODE, int EPI, int VEC, int BY, int BZ, int R, int NW>
__global__ void __launch_bounds__((NW + 1) * 32, 1)
eval_staged_kernel(const __grid_constant__ CUtensorMap tmap, Geom g, StagedGeom sg,
                   const float4* __restrict__ recs, const int4* __restrict__ order, int* __restrict__ meta,
                   int nchunk, float* __restrict__ val, float* __restrict__ grad, float* __restrict__ lap,
                   long long ld, const float* __restrict__ dvec, long long ldd, float* __restrict__ cout,
                   const double* __restrict__ pos, const double* __restrict__ kvec)
{
    constexpr bool CONTRACT = EPI == kEpiContract;
    using Cfg = StagedCfg<VEC, BY, BZ, R, NW>;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    typename Cfg::Smem& sm = *reinterpret_cast<typename Cfg::Smem*>(smem_raw);
    static_assert(VEC == 4, "a lane owns 4 orbitals (one 128-bit load per row)");
    constexpr int NP = VEC / 2;
    constexpr unsigned IQ = kItemQueue;
    constexpr unsigned RU = R;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    wait_for_predecessor();
    if (threadIdx.x == 0) {
        for (int s = 0; s < R; ++s) { mbar_init(smem_u32(&sm.full[s]), 1); mbar_init(smem_u32(&sm.empty[s]), NW); }
        for (int s = 0; s < (int)IQ; ++s) { mbar_init(smem_u32(&sm.ifull[s]), 1); mbar_init(smem_u32(&sm.iempty[s]), NW); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();

    if (warp == NW) {
        // ---- producer.  It may leave as soon as everything is issued: every consumer waits
        // for every plane before it leaves, so no copy outlives the CTA.
        if (lane == 0) {
            const int nps = meta[0];
            const int nitems = nps * nchunk;
            unsigned seq_pub = 0;                            // sequence number of the next item's first plane
            struct Desc { int nplanes, chunk, by, bz, lo; };
            auto fetch = [&](unsigned k) -> Desc {           // take item k from the global queue and publish it
                const unsigned q = k % IQ;
                if (k >= IQ) mbar_wait_backoff(smem_u32(&sm.iempty[q]), ((k / IQ) & 1u) ^ 1u);
                const int w = atomicAdd(&meta[1], 1);
                WorkItem& it = sm.item[q];
                Desc d = {-1, 0, 0, 0, 0};
                if (w < nitems) {
                    // heaviest segment first, its chunks side by side
                    d.chunk = w % nchunk;
                    const int4 o = __ldg(order + w / nchunk);
                    const int pencil = o.x / sg.nseg, segi = o.x - pencil * sg.nseg;
                    d.lo = segi * sg.seg;
                    const int hi = min(d.lo + sg.seg, g.n[0]) - 1;
                    d.by = pencil / sg.nbz; d.bz = pencil - d.by * sg.nbz;
                    d.nplanes = o.z > 0 ? hi + 4 - d.lo : 0;
                    it.chunk = d.chunk; it.by = d.by; it.bz = d.bz; it.lo = d.lo; it.seq0 = seq_pub;
                    it.u0 = (unsigned)o.y; it.nunits = (unsigned)o.z;
                    seq_pub += (unsigned)d.nplanes;
                    for (int k2 = 0; k2 < min(d.nplanes, R); ++k2)       // warm L2 with the item's first planes
                        tma_prefetch_4d(&tmap, d.chunk * Cfg::C, d.bz * BZ, d.by * BY, d.lo + k2);
                }
                it.nplanes = d.nplanes;
                mbar_arrive(smem_u32(&sm.ifull[q]));
                return d;
            };
            unsigned seq = 0;
            Desc cur = fetch(0);
            for (unsigned k = 0; cur.nplanes >= 0; ++k) {
                for (int j = 0; j < cur.nplanes; ++j, ++seq) {
                    const unsigned slot = seq % RU, round = seq / RU;
                    if (j + R < cur.nplanes)
                        tma_prefetch_4d(&tmap, cur.chunk * Cfg::C, cur.bz * BZ, cur.by * BY, cur.lo + j + R);
                    if (round > 0) mbar_wait_backoff(smem_u32(&sm.empty[slot]), (round & 1u) ^ 1u);
                    const unsigned bar = smem_u32(&sm.full[slot]);
                    mbar_expect_tx(bar, Cfg::PLANE_BYTES);
                    tma_load_4d(smem_u32(&sm.plane[slot][0]), &tmap, cur.chunk * Cfg::C, cur.bz * BZ, cur.by * BY,
                                cur.lo + j, bar);
                }
                // the next item is taken from the global queue only now, when the consumers are
                // within a ring of the end of this one: a CTA never sits on a queued item while
                // another CTA runs dry
                cur = fetch(k + 1);
            }
        }
        return;
    }

    // ---- consumers.  Warp w takes units w, w + NW, ... of every item.  Planes are counted by
    // their CTA-wide sequence number; a warp waits for plane q only after releasing plane q-R
    // (whose slot plane q reuses) and releases a plane only after having waited for it, so
    // its arrival on an empty barrier always belongs to the barrier's current phase.
    //
    // The loop below is bound by instruction issue (a packed FMA holds the issue port of its
    // scheduler for two cycles, everything else for one), so the bookkeeping per unit is kept
    // short: the record carries the unit's plane number and byte offset inside a plane.
    unsigned released = 0;             // planes < released have been released by this warp
    unsigned waited = 0;               // planes < waited have been waited for by this warp
    const unsigned full0 = smem_u32(&sm.full[0]), empty0 = smem_u32(&sm.empty[0]);
    // plane q of the current unit (q - released < R, so nothing is due for release first)
    auto wait_plane = [&](unsigned q) {
        if (waited <= q) {
            mbar_wait(full0 + 8u * (q % RU), (q / RU) & 1u);
            waited = q + 1;
        }
    };
    auto release_upto = [&](unsigned release_end) {      // planes < release_end no longer needed by this warp
#pragma unroll 1
        while (released < release_end) {
            mbar_arrive_lane0(empty0 + 8u * (released % RU), lane);
            ++released;
        }
    };
    // Planes < end that this warp does not read (between two of its units, or to the end of an
    // item): each is given back as soon as it has been waited for.  Holding them until the
    // next wait forces it would let the producer issue plane q only when the consumers
    // already stand waiting for it, i.e. put the full copy latency on every plane passed.
    auto pass_upto = [&](unsigned end) {
        release_upto(min(waited, end));
        if (waited < end) {
#pragma unroll 1
            do {
                const unsigned sl = 8u * (waited % RU);
                mbar_wait(full0 + sl, (waited / RU) & 1u);
                mbar_arrive_lane0(empty0 + sl, lane);
                ++waited;
            } while (waited < end);
            released = waited;
        }
    };

    unsigned n = 0;                    // current item
    unsigned u = (unsigned)warp;       // current unit of item n
    bool have = false;                 // sm.rec[warp] already holds the record of (n, u)
    int it_nplanes, it_col0 = 0;
    unsigned it_seq0 = 0, it_nunits = 0;
    const float4* it_rsrc = recs;
    auto load_item = [&](unsigned k) {
        mbar_wait(smem_u32(&sm.ifull[k % IQ]), (k / IQ) & 1u);
        const WorkItem& it = sm.item[k % IQ];
        it_nplanes = it.nplanes;
        if (it_nplanes >= 0) {
            it_col0 = it.chunk * Cfg::C + lane * VEC;
            it_seq0 = it.seq0;
            it_nunits = it.nunits;
            it_rsrc = recs + (size_t)it.u0 * (kRecFloats / 4);
        }
    };
    load_item(0);
    const unsigned lane_off = (unsigned)lane * (VEC * 4);
    const unsigned plane0 = smem_u32(&sm.plane[0][0]);
    while (true) {
        while (it_nplanes >= 0 && u >= it_nunits) {          // leave item n: pass all its planes
            if (it_nplanes > 0) pass_upto(it_seq0 + it_nplanes);
            __syncwarp();
            if (lane == 0) mbar_arrive(smem_u32(&sm.iempty[n % IQ]));
            ++n; u = (unsigned)warp;
            load_item(n);
        }
        if (it_nplanes < 0) break;
        if (!have) {
            if (lane < kRecFloats / 4)
                reinterpret_cast<float4*>(&sm.rec[warp])[lane] = __ldg(it_rsrc + (size_t)u * (kRecFloats / 4) + lane);
            __syncwarp();
        }
        const StagedRec& rec = reinterpret_cast<const StagedRec&>(sm.rec[warp]);
        const int4 loc = rec.loc;
        BLIP_ASSERT((long long)((it_rsrc - recs) / (kRecFloats / 4)) + u < g.M && loc.w >= 0 && (long long)loc.w < g.M);
        BLIP_ASSERT(loc.x < it_nplanes - 3 && loc.y >= 0 && loc.y + 3 * (Cfg::PZ * Cfg::C * 4) + 4 * Cfg::C * 4 <= Cfg::PLANE_BYTES);                            // {plane in item or -1, byte offset in plane, -, electron}
        const bool ok = loc.x >= 0;                          // non-finite positions (bin 0) touch no plane
        const unsigned sq = it_seq0 + (unsigned)loc.x;
        // planes i1, i1+1 resident, earlier ones released; planes i1+2 and i1+3 are waited for
        // just before their quarter of the loop, which leaves the producer two more slots of the
        // ring to run ahead of the consumers
        if (ok) { pass_upto(sq); wait_plane(sq); wait_plane(sq + 1); }

        // record of this warp's next unit, in flight during the FMAs
        const float4* nsrc = nullptr;
        if (u + NW < it_nunits) nsrc = it_rsrc + (size_t)(u + NW) * (kRecFloats / 4);
        else {
            // the next item, if the producer has published it already (it does so once all planes
            // of this one are issued; waiting for it here, with this unit's planes pinned, could
            // starve the producer of ring slots)
            if (mbar_test(smem_u32(&sm.ifull[(n + 1) % IQ]), ((n + 1) / IQ) & 1u)) {
                const WorkItem& nx = sm.item[(n + 1) % IQ];
                if (nx.nplanes >= 0 && (unsigned)warp < nx.nunits)
                    nsrc = recs + (size_t)(nx.u0 + (unsigned)warp) * (kRecFloats / 4);
            }
        }
        float4 pre = make_float4(0.f, 0.f, 0.f, 0.f);
        if (nsrc && lane < kRecFloats / 4) pre = __ldg(nsrc + lane);
        float4 dv = make_float4(0.f, 0.f, 0.f, 0.f);        // contraction mode: this lane's d values, in flight during the FMAs
        if (CONTRACT && it_col0 < 4 * g.pitch4) dv = ldg_dvec(dvec, ldd, loc.w, it_col0);
        // a-5: store the unit's results, or contract them with d (blipgpu_eval_contract)
        auto emit = [&](const PairAcc (&a)[NP]) {
            if (CONTRACT) {
                float sum[5] = {0.f, 0.f, 0.f, 0.f, 0.f};
                if (it_col0 < 4 * g.pitch4) {
                    float dq[4];
                    mask_dvec(dv, it_col0, g.L, dq);
                    contract_pairs<MODE, NP>(g, a, dq, sum);
                }
                contract_flush<MODE>(g, sum, loc.w, cout, lane);
            } else if (it_col0 < 4 * g.pitch4) {
                if (EPI == kEpiComplex) store_pairs_complex<MODE>(g, a, loc.w, it_col0, pos, kvec, val, grad, lap, ld);
                else store_pairs<MODE, NP>(g, a, loc.w, it_col0, val, grad, lap, ld);
            }
        };
        if (!ok) {                                           // non-finite position (rare): NaN out, no plane touched
            PairAcc nanacc[NP];
#pragma unroll
            for (int p = 0; p < NP; ++p) set_nan(nanacc[p]);
            emit(nanacc);
        } else {
            PairAcc acc[NP];
#pragma unroll
            for (int p = 0; p < NP; ++p) acc[p].val = acc[p].t1 = acc[p].t2 = acc[p].t3 = acc[p].lp = 0ull;
            float wz[3][4];
#pragma unroll
            for (int k = 0; k < 3; ++k)
#pragma unroll
                for (int m = 0; m < 4; ++m) wz[k][m] = rec.wz[k][m];
            const unsigned off = (unsigned)loc.y + lane_off;
#pragma unroll
            for (int m1 = 0; m1 < 4; ++m1) {
                // planes i1+2, i1+3 just before their quarter of the loop
                if (m1 >= 2) wait_plane(sq + m1);
                BLIP_ASSERT(sq + m1 < waited && sq + m1 >= released && sq + m1 - released < RU);   // landed, not given back
                const unsigned pp = plane0 + ((sq + m1) % RU) * (unsigned)Cfg::PLANE_BYTES + off;
#pragma unroll
                for (int m2 = 0; m2 < 4; ++m2) {
                    const unsigned cp = pp + m2 * (Cfg::PZ * Cfg::C * 4);
                    const float4 w = rec.cw[4 * m1 + m2];
                    const float lb = (MODE == 1) ? rec.lb[4 * m1 + m2] : 0.f;
                    if (VEC == 4) {
                        const ulonglong2 c0 = lds128(cp), c1 = lds128(cp + Cfg::C * 4);
                        const ulonglong2 c2 = lds128(cp + 2 * Cfg::C * 4), c3 = lds128(cp + 3 * Cfg::C * 4);
                        fold_pair<MODE>(c0.x, c1.x, c2.x, c3.x, wz, w, lb, acc[0]);
                        fold_pair<MODE>(c0.y, c1.y, c2.y, c3.y, wz, w, lb, acc[NP - 1]);
                    } else {
                        const u64 c0 = lds64(cp), c1 = lds64(cp + Cfg::C * 4);
                        const u64 c2 = lds64(cp + 2 * Cfg::C * 4), c3 = lds64(cp + 3 * Cfg::C * 4);
                        fold_pair<MODE>(c0, c1, c2, c3, wz, w, lb, acc[0]);
                    }
                }
            }
            emit(acc);
        }

        have = nsrc != nullptr;
        __syncwarp();                                        // every lane is done with this unit's record
        if (have && lane < kRecFloats / 4) reinterpret_cast<float4*>(&sm.rec[warp])[lane] = pre;
        __syncwarp();
        u += NW;
    }
}

}  // namespace blip
