// blip_tc.cuh — the gather + FMA step (a-3) of dense batches on the 5th-generation tensor cores
// (tcgen05.mma with the coefficient operand in tensor memory), sm_100a.
//
// PAPER.md:401-419 (§VI.E, Eq. 13-15) rejects the dense matrix form psi = A Theta because the
// matrix changes with the electron position; north_star allows tensor cores "only if recasting the
// batch as a dense weights x coefficients contraction is shown to win".  The recast that does win
// keeps the contraction per electron, K = the sites of the electron's 4x4x4 block, and puts the
// COEFFICIENTS on the M side of the MMA, where the tensor core is full whatever the batch holds:
//
//     D[128 orbitals][N = 16] += A[128 orbitals][K = 16 sites] * B[K = 16 sites][N = 16]
//
//   A  one table plane of the pencil's 7 x 7-row cross-section, transposed into tensor memory
//      (lane = orbital, column = site), so that the 16 sites of an MMA — rows (y, z = 0..7) and
//      (y + 1, z = 0..7) of the plane, the z axis padded from 7 to 8 — are 8 consecutive TMEM
//      columns that start at a multiple of 4: any electron of the pencil finds its rows y0 ..
//      y0 + 3 at column 4 y0 of the plane, no copy per electron;
//   B  the electron's folded weights (W, Gamma_x,y,z, Lambda per site) in
//      shared memory, zero outside its z window z0 .. z0 + 3;
//   D  fp32 accumulators in tensor memory, read back by the epilogue warps (tcgen05.ld).
//
// Precision.  The tensor core multiplies fp16 (11 significant bits); north_star's tolerances
// need ~2^-20.  Both operands are split exactly in two fp16 halves after an exact power-of-two
// scaling: c' = c 2^k_l = c1 + c2 (c1 = rn16(c'), c2 = rn16(c' - c1): 22 bits), W' = W 2^kq =
// W1 + W2 likewise.  The coefficient scale is PER ORBITAL l (the M rows of the MMA are orbitals):
// 2^k_l max|c_l| in [2^8, 2^9), so an orbital whose amplitude is far below the table's maximum keeps
// its own 22 bits instead of falling on the fp16 subnormal floor of a table-wide scale; the epilogue
// lane that holds orbital l undoes it with one more exact multiply (reading R12a).  The B tile carries [W1 | W2] in its N dimension (columns 0..4 and 5..9), the A
// operand is issued twice (c1, c2) into the same accumulators, so that D[:, q] + D[:, 5 + q] =
// (c1 + c2)(W1 + W2) summed over the sites in fp32: all four cross terms, error ~2^-21 of
// sum |c W|.  Per electron and 128 orbitals: 4 planes x 2 row pairs x 2 halves = 16 MMAs.
//
// The scaled, split, z-paired fp16 words of A are not computed per launch: the library writes them
// once (first use of this path, or blipgpu_reserve) into a second table of its own (tc_table_kernel below; same bytes per coefficient as the
// fp32 table), so that a staged plane is moved to tensor memory word for word.
//
// Roles of the persistent CTA (one per SM), 29 warps:
//   producer (1)     work items (chunk-major: all pencils of one 128-orbital slice of the table are
//                    in flight together and find each other's halo rows in L2) and one 5-D TMA box
//                    per plane into a ring of 4 shared-memory slots — the protocol of eval_staged_kernel;
//   converters (2x4) a group per plane parity, a warp per TMEM lane quarter: the plane's 56 words per
//                    orbital from shared memory -> tcgen05.st into a ring of 8 TMEM plane slots
//                    (2 halves x 28 columns each);
//   weights (8)      one electron each: record -> 80 (column, quantity) weight vectors, scaled and
//                    split -> B tile slot (4 KB) in the canonical K-major core-matrix layout;
//   issuers (4)      one elected thread each: wait for B tile, planes and a free accumulator,
//                    issue the 16 MMAs, tcgen05.commit to free the B slot / publish D; planes are
//                    given back to the converters by commit as the units move on;
//   epilogue (2 x 4) tcgen05.ld of D, unscale, Cartesian gradient, streaming stores (a-5).
// All hand-offs are mbarriers; units are numbered CTA-wide so that slot and phase of every ring
// follow from the unit (or plane) number alone.
#pragma once
#include "blip_kernels.cuh"
#include <cuda_fp16.h>

namespace blip {

constexpr int kTcRS = 4;            // shared-memory plane slots (one TMA box each)
constexpr int kTcRT = 8;            // TMEM plane slots
constexpr int kTcPlaneCols = 56;    // TMEM columns of a plane: 2 halves x 7 rows x 4 columns (8 fp16 z sites)
constexpr int kTcND = 4;            // accumulator slots (16 columns each)
constexpr int kTcDCol0 = kTcRT * kTcPlaneCols;               // 392
constexpr int kTcNB = 16;           // B tile slots
constexpr int kTcBBytes = 4096;     // 8 tiles x 512 B
constexpr int kTcPlaneWords = 7 * 4 * 2 * 128;               // 28,672 bytes per staged plane
constexpr int kTcNInfo = 32;        // unit info ring (>= kTcNB + kTcND)
constexpr int kTcNC = 8, kTcNE = 8, kTcNW = 8, kTcNI = 4;
constexpr int kTcWarps = kTcNC + kTcNE + kTcNW + kTcNI + 1;  // 29
constexpr int kTcThreads = kTcWarps * 32;
constexpr int kTcReaders = kTcNC + kTcNE + kTcNW + kTcNI;    // warps that walk the item queue
static_assert(kTcDCol0 + 16 * kTcND <= 512, "tensor memory has 512 columns");
static_assert(kTcNInfo >= kTcNB + kTcND, "unit info must outlive the B slot until the epilogue has read it");
// An mbarrier wait names its phase by parity only, so a waiter must see EVERY phase of the barriers
// it waits on (a waiter that skips one takes the phase before its own for complete): every ring
// slot is therefore always waited for by the same warp(s) —
static_assert(kTcNC == 8 && kTcRS % 2 == 0 && kTcRT % 2 == 0, "two converter groups alternate planes: a slot must keep its plane parity");
static_assert(kTcNB % kTcNW == 0 && kTcNB % kTcNI == 0, "a B slot belongs to one weight warp and one issuer");
static_assert(kTcND % kTcNI == 0 && kTcND % 2 == 0, "an accumulator slot belongs to one issuer and one epilogue group");

struct TcScale {
    float sw[5];        // 2^kq applied to the weights of quantity q (val, T1, T2, T3, lap)
    float inv[5];       // 1 / sw[q]; the per-orbital 2^-k_l comes from the `oscale` array (tc_colscale_kernel)
};
constexpr int kTcMaxScaleExp = 100; // |k_l| <= 100: the host admits tables with max|c| < 2^100 only, and 2^-(k_l + kq) stays a normal fp32

struct TcSmem {
    alignas(128) unsigned plane[kTcRS][kTcPlaneWords];       // [y 7][z pair 4][half 2][128 orbitals], one TMA box
    alignas(128) unsigned char bt[kTcNB][kTcBBytes];
    alignas(16) float4 wrec[kTcNW][kRecFloats / 4];          // record of the unit a weight warp works on
    alignas(16) int4 info[kTcNInfo];                        // {plane sequence number or -1, y0, electron, -}
    alignas(16) WorkItem item[kItemQueue];
    alignas(8) u64 full[kTcRS], empty[kTcRS];                // shared-memory planes: TMA -> converters
    alignas(8) u64 tfull[kTcRT], tempty[kTcRT];              // TMEM planes: converters -> issuers
    alignas(8) u64 bfull[kTcNB], bempty[kTcNB];              // B tiles: weight warps -> issuers
    alignas(8) u64 dfull[kTcND], dempty[kTcND];              // accumulators: issuers -> epilogue
    alignas(8) u64 ifull[kItemQueue], iempty[kItemQueue];
    unsigned tbase;
};

__device__ __forceinline__ bool tc_elect_one()
{
    unsigned pred;
    asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(pred));
    return pred != 0;
}
constexpr unsigned kTcWaitHintNs = 100;
// wait of a role that runs ahead of / behind the issuers: the hardware may park the warp for up to
// 100 ns per poll instead of spinning in the issue slots the other roles need (1 us and sleeping
// waits were slower: the wake-up latency costs more than the polls, profiles/r2_v2.md)
__device__ __forceinline__ void mbar_wait_relaxed(unsigned bar, unsigned parity)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1, %2;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}"
        :: "r"(bar), "r"(parity), "r"(kTcWaitHintNs) : "memory");
}
__device__ __forceinline__ void tc_commit(unsigned bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" :: "r"(bar) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
// B tile descriptor: K-major, no swizzle, core matrices of 8 N-rows x 16 bytes; the two K halves
// of an MMA are 128 bytes apart (leading byte offset), the two N halves 256 (stride byte offset)
__device__ __forceinline__ uint64_t tc_bdesc(unsigned addr)
{
    return (uint64_t)((addr >> 4) & 0x3fffu) | ((uint64_t)(128u >> 4) << 16) | ((uint64_t)(256u >> 4) << 32) | ((uint64_t)1 << 46);
}
// kind::f16, A and B fp16 K-major, D fp32, M = 128, N = 16
constexpr unsigned kTcIdesc = (1u << 4) | ((16u >> 3) << 17) | ((128u >> 4) << 24);
__device__ __forceinline__ void tc_mma(unsigned d, unsigned a, uint64_t b, unsigned accumulate)
{
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}"
                 :: "r"(d), "r"(a), "l"(b), "r"(kTcIdesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ unsigned tc_pack(float lo, float hi)      // {hi, lo} -> two fp16, round to nearest
{
    unsigned r; asm("cvt.rn.f16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo)); return r;
}
__device__ __forceinline__ float2 tc_unpack(unsigned p)
{
    return __half22float2(*reinterpret_cast<const __half2*>(&p));
}
// x (already scaled) -> the two fp16 halves of a pair of values
__device__ __forceinline__ void tc_split2(float x0, float x1, unsigned& h1, unsigned& h2)
{
    h1 = tc_pack(x0, x1);
    const float2 f = tc_unpack(h1);
    h2 = tc_pack(__fsub_rn(x0, f.x), __fsub_rn(x1, f.y));
}

__device__ __forceinline__ void tma_load_5d(unsigned dst, const CUtensorMap* tmap, int c0, int c1, int c2, int c3, int c4, unsigned bar)
{
    asm volatile(
        "cp.async.bulk.tensor.5d.shared::cluster.global.tile.mbarrier::complete_tx::bytes "
        "[%0], [%1, {%2, %3, %4, %5, %6}], [%7];"
        :: "r"(dst), "l"(reinterpret_cast<uint64_t>(tmap)), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4), "r"(bar)
        : "memory");
}
__device__ __forceinline__ void tma_prefetch_5d(const CUtensorMap* tmap, int c0, int c1, int c2, int c3, int c4)
{
    asm volatile("cp.async.bulk.prefetch.tensor.5d.L2.global.tile [%0, {%1, %2, %3, %4, %5}];"
                 :: "l"(reinterpret_cast<uint64_t>(tmap)), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4) : "memory");
}

// The table of the tensor-core path (library-owned, built from the padded fp32 table when the handle
// first takes this path, or by blipgpu_reserve): the ghost-padded table with every coefficient
// scaled by 2^kc and split in its two fp16 halves, z sites in pairs, 32-bit words
//     T16[p1][p2][zp][half][l] = { c_half[p1][p2][2 zp][l], c_half[p1][p2][2 zp + 1][l] << 16 }
// — exactly the word a TMEM column of the A operand holds, so that the converter warps only move
// words from the staged plane to tensor memory.  Same bytes per coefficient as fp32.
// oscale[l] = 2^k_l, the scale of orbital l (tc_colscale_kernel).
__global__ void __launch_bounds__(256)
tc_table_kernel(Geom g, const float* __restrict__ oscale, int nzp, const float* __restrict__ padded /* [np1][np2][np3][pitch], the fp32 table */,
                unsigned* __restrict__ dst, long long total)
{
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= total) return;
    const int pitch = 4 * g.pitch4;
    const int l = (int)(idx % pitch);
    const long long r = idx / pitch;                         // (p1 np2 + p2) nzp + zp
    const int zp = (int)(r % nzp);
    const long long p12 = r / nzp;
    const float sc = __ldg(oscale + l);
    float c[2] = {0.f, 0.f};
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        const int p3 = 2 * zp + h;
        if (p3 < g.np[2]) c[h] = __fmul_rn(__ldg(padded + ((size_t)p12 * g.np[2] + p3) * (size_t)pitch + l), sc);
    }
    unsigned h1, h2;
    tc_split2(c[0], c[1], h1, h2);
    const size_t o = (size_t)r * 2 * (size_t)pitch + l;
    dst[o] = h1;
    dst[o + pitch] = h2;
}

// The B tiles of one electron (unit): lane = (column (m1, m2) = lane / 2, half = lane % 2).  Half 0
// builds the weight vectors of val, T1, T2 (P00, P10, P01 times the z weights w3), half 1 those of
// T3 (P00 w3') and lap (La w3 + Lb w3' + P00 Q22 w3''), each scaled by its power of two, split in
// two fp16 halves and placed at z sites Z0 .. Z0 + 3 of the row's 8 (zero elsewhere).
template <int Z0>
__device__ __forceinline__ uint4 tc_place(unsigned a0, unsigned a1)
{
    if (Z0 == 0) return make_uint4(a0, a1, 0u, 0u);
    if (Z0 == 2) return make_uint4(0u, a0, a1, 0u);
    const unsigned p0 = a0 << 16, p1 = __byte_perm(a0, a1, 0x5432), p2 = a1 >> 16;
    return Z0 == 1 ? make_uint4(p0, p1, p2, 0u) : make_uint4(0u, p0, p1, p2);
}
template <int Z0>
__device__ __forceinline__ void tc_store_vec(unsigned char* tile, int n, const float (&w)[4])
{
    unsigned a1[2], a2[2];
    tc_split2(w[0], w[1], a1[0], a2[0]);
    tc_split2(w[2], w[3], a1[1], a2[1]);
    const int n2 = n + 5;
    *reinterpret_cast<uint4*>(tile + n * 16) = tc_place<Z0>(a1[0], a1[1]);
    *reinterpret_cast<uint4*>(tile + (n2 >> 3) * 256 + (n2 & 7) * 16) = tc_place<Z0>(a2[0], a2[1]);
}
template <int Z0, int MODE>
__device__ __forceinline__ void tc_build_tile(const float4* rec4, const float* recf, const float (&wz)[3][4], const TcScale& scl,
                                              unsigned char* bt, int lane)
{
    const int colm = lane >> 1;
    const bool hb = lane & 1;
    if (MODE == 0 && hb) return;                             // value only: rows 1..4 and 6..9 of the tiles stay zero for the whole launch
    const float4 cw = rec4[colm];
    const int m1 = colm >> 2, m2 = colm & 3;
    unsigned char* const tile = bt + (m1 * 2 + (m2 >> 1)) * 512 + (m2 & 1) * 128;
    float w[4];
    {   // val (half 0) / T3 (half 1): P00 times w3 or w3'
        const float f = __fmul_rn(cw.x, hb ? scl.sw[3] : scl.sw[0]);
#pragma unroll
        for (int m = 0; m < 4; ++m) w[m] = __fmul_rn(f, hb ? wz[1][m] : wz[0][m]);
        tc_store_vec<Z0>(tile, hb ? 3 : 0, w);
    }
    if (MODE == 0) return;
    if (hb) {   // lap
        const float lb = recf[64 + colm];
        const float fa = __fmul_rn(cw.w, scl.sw[4]), fb = __fmul_rn(lb, scl.sw[4]), fc = __fmul_rn(cw.x, scl.sw[4]);
#pragma unroll
        for (int m = 0; m < 4; ++m) w[m] = __fmaf_rn(fc, wz[2][m], __fmaf_rn(fb, wz[1][m], __fmul_rn(fa, wz[0][m])));
        tc_store_vec<Z0>(tile, 4, w);
    } else {    // T1, T2
        const float f1 = __fmul_rn(cw.y, scl.sw[1]), f2 = __fmul_rn(cw.z, scl.sw[2]);
#pragma unroll
        for (int m = 0; m < 4; ++m) w[m] = __fmul_rn(f1, wz[0][m]);
        tc_store_vec<Z0>(tile, 1, w);
#pragma unroll
        for (int m = 0; m < 4; ++m) w[m] = __fmul_rn(f2, wz[0][m]);
        tc_store_vec<Z0>(tile, 2, w);
    }
}

template <int MODE>
__global__ void __launch_bounds__(kTcThreads, 1)
eval_tc_kernel(const __grid_constant__ CUtensorMap tmap, Geom g, StagedGeom sg, TcScale scl,
               const float4* __restrict__ recs, const int4* __restrict__ order, int* __restrict__ meta,
               int nchunk, float* __restrict__ val, float* __restrict__ grad, float* __restrict__ lap, long long ld,
               int idx32_arg /* every output element offset of this call fits 32 bits (tc_launch derives it from M and ld) */,
               const float* __restrict__ oinv /* [pitch] 2^-k_l: undoes the per-orbital scale of the fp16 table */)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    TcSmem& sm = *reinterpret_cast<TcSmem*>(smem_raw);
    constexpr unsigned IQ = kItemQueue;
    constexpr int PLANE_BYTES = kTcPlaneWords * 4;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const bool idx32 = idx32_arg != 0;
    wait_for_predecessor();
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" :: "r"(smem_u32(&sm.tbase)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    if (threadIdx.x == 32) {
        for (int s = 0; s < kTcRS; ++s) { mbar_init(smem_u32(&sm.full[s]), 1); mbar_init(smem_u32(&sm.empty[s]), 4); }
        for (int s = 0; s < kTcRT; ++s) { mbar_init(smem_u32(&sm.tfull[s]), 4); mbar_init(smem_u32(&sm.tempty[s]), kTcNI); }
        for (int s = 0; s < kTcNB; ++s) { mbar_init(smem_u32(&sm.bfull[s]), 1); mbar_init(smem_u32(&sm.bempty[s]), 1); }
        for (int s = 0; s < kTcND; ++s) { mbar_init(smem_u32(&sm.dfull[s]), 1); mbar_init(smem_u32(&sm.dempty[s]), 4); }
        for (int s = 0; s < (int)IQ; ++s) { mbar_init(smem_u32(&sm.ifull[s]), 1); mbar_init(smem_u32(&sm.iempty[s]), kTcReaders); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    // B tiles: the N rows 10..15 of every tile stay zero for the whole kernel
    for (int i = threadIdx.x; i < kTcNB * kTcBBytes / 16; i += kTcThreads)
        reinterpret_cast<uint4*>(&sm.bt[0][0])[i] = make_uint4(0u, 0u, 0u, 0u);
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const unsigned tbase = sm.tbase;

    // every reader role walks the item queue the same way
    int it_nplanes = 0, it_chunk = 0;
    unsigned it_seq0 = 0, it_nunits = 0, it_u0 = 0;
    auto load_item = [&](unsigned k) {
        mbar_wait(smem_u32(&sm.ifull[k % IQ]), (k / IQ) & 1u);
        const WorkItem& it = sm.item[k % IQ];
        it_nplanes = it.nplanes;
        if (it_nplanes >= 0) { it_chunk = it.chunk; it_seq0 = it.seq0; it_nunits = it.nunits; it_u0 = it.u0; }
    };
    auto leave_item = [&](unsigned k, bool one_thread) {
        if (!one_thread) __syncwarp();
        if (one_thread || lane == 0) mbar_arrive(smem_u32(&sm.iempty[k % IQ]));
    };

    if (warp == kTcWarps - 1) {
        // ---- producer: as in eval_staged_kernel (work queue, item descriptors, one TMA box per plane)
        if (lane == 0) {
            const int nps = meta[0];
            const int nitems = nps * nchunk;
            unsigned seq_pub = 0;
            struct Desc { int nplanes, chunk, by, bz, lo; };
            auto fetch = [&](unsigned k) -> Desc {
                const unsigned q = k % IQ;
                if (k >= IQ) mbar_wait_backoff(smem_u32(&sm.iempty[q]), ((k / IQ) & 1u) ^ 1u);
                const int w = atomicAdd(&meta[1], 1);
                WorkItem& it = sm.item[q];
                Desc d = {-1, 0, 0, 0, 0};
                if (w < nitems) {
                    // chunk-major: every pencil of one 128-orbital chunk before the next chunk, so that the CTAs
                    // in flight work on neighbouring pencils of ONE slice of the table and find each other's
                    // halo rows in L2 (the kernel is close to the DRAM bound; blip_tc.cuh header)
                    d.chunk = w / nps;
                    const int4 o = __ldg(order + (w - d.chunk * nps));
                    const int pencil = o.x / sg.nseg, segi = o.x - pencil * sg.nseg;
                    d.lo = segi * sg.seg;
                    const int hi = min(d.lo + sg.seg, g.n[0]) - 1;
                    d.by = pencil / sg.nbz; d.bz = pencil - d.by * sg.nbz;
                    d.nplanes = o.z > 0 ? hi + 4 - d.lo : 0;
                    it.chunk = d.chunk; it.by = d.by; it.bz = d.bz; it.lo = d.lo; it.seq0 = seq_pub;
                    it.u0 = (unsigned)o.y; it.nunits = (unsigned)o.z;
                    seq_pub += (unsigned)d.nplanes;
                    for (int k2 = 0; k2 < min(d.nplanes, 8); ++k2)
                        tma_prefetch_5d(&tmap, d.chunk * 128, 0, d.bz * 2, d.by * 4, d.lo + k2);
                }
                it.nplanes = d.nplanes;
                mbar_arrive(smem_u32(&sm.ifull[q]));
                return d;
            };
            unsigned seq = 0;
            Desc cur = fetch(0);
            for (unsigned k = 0; cur.nplanes >= 0; ++k) {
                for (int j = 0; j < cur.nplanes; ++j, ++seq) {
                    const unsigned slot = seq % kTcRS, round = seq / kTcRS;
                    if (j + 8 < cur.nplanes) tma_prefetch_5d(&tmap, cur.chunk * 128, 0, cur.bz * 2, cur.by * 4, cur.lo + j + 8);
                    if (round > 0) mbar_wait_backoff(smem_u32(&sm.empty[slot]), (round & 1u) ^ 1u);
                    const unsigned bar = smem_u32(&sm.full[slot]);
                    mbar_expect_tx(bar, PLANE_BYTES);
                    tma_load_5d(smem_u32(&sm.plane[slot][0]), &tmap, cur.chunk * 128, 0, cur.bz * 2, cur.by * 4, cur.lo + j, bar);
                }
                cur = fetch(k + 1);
            }
        }
    } else if (warp < kTcNC) {
        // ---- converters: lane quarter `warp` of tensor memory, thread = orbital 32 warp + lane
        const int cq = warp & 3, cg = warp >> 2;             // lane quarter; group cg converts the planes with (sequence number) % 2 == cg
        const unsigned tlane = tbase + ((unsigned)(cq * 32) << 16);
        const int orb = cq * 32 + lane;
        for (unsigned n = 0;; ++n) {
            load_item(n);
            if (it_nplanes < 0) break;
            for (int j = (int)((it_seq0 + (unsigned)cg) & 1u); j < it_nplanes; j += 2) {
                const unsigned q = it_seq0 + (unsigned)j;
                const unsigned s = q % kTcRS, t = q % kTcRT;
                mbar_wait_relaxed(smem_u32(&sm.full[s]), (q / kTcRS) & 1u);
                // rows 0..3 of the plane (32 words, all loads in flight at once) wait in registers for the
                // TMEM slot; rows 4..6 follow behind the first stores (56 words at once do not fit in the
                // 64 registers a thread of this 928-thread CTA has)
                const unsigned* src = &sm.plane[s][orb];
                const unsigned tcol = tlane + t * kTcPlaneCols;
                // word (y, z pair k, half) of this orbital; a half's 28 words are 28 consecutive TMEM columns
                auto word = [&](int y, int k, int half) { return src[((y * 4 + k) * 2 + half) * 128]; };
                unsigned a1[16], a2[16];                     // rows 0..3, halves 1 and 2
#pragma unroll
                for (int i = 0; i < 16; ++i) { a1[i] = word(i >> 2, i & 3, 0); a2[i] = word(i >> 2, i & 3, 1); }
                if (q >= kTcRT) mbar_wait_relaxed(smem_u32(&sm.tempty[t]), ((q / kTcRT) & 1u) ^ 1u);
                tc_fence_after();
#define BLIP_TC_ST16(col, v)                                                                                          \
                asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};" \
                             :: "r"(col), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]), "r"(v[8]),   \
                                "r"(v[9]), "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15]) : "memory")
                BLIP_TC_ST16(tcol, a1);
                BLIP_TC_ST16(tcol + 28, a2);
#undef BLIP_TC_ST16
                unsigned b1[12], b2[12];                     // rows 4..6
#pragma unroll
                for (int i = 0; i < 12; ++i) { b1[i] = word(4 + (i >> 2), i & 3, 0); b2[i] = word(4 + (i >> 2), i & 3, 1); }
#define BLIP_TC_ST8(col, v, o)                                                                                         \
                asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};"              \
                             :: "r"(col), "r"(v[o]), "r"(v[o + 1]), "r"(v[o + 2]), "r"(v[o + 3]), "r"(v[o + 4]), "r"(v[o + 5]), "r"(v[o + 6]), "r"(v[o + 7]) : "memory")
#define BLIP_TC_ST4(col, v, o)                                                                                         \
                asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};" :: "r"(col), "r"(v[o]), "r"(v[o + 1]), "r"(v[o + 2]), "r"(v[o + 3]) : "memory")
                BLIP_TC_ST8(tcol + 16, b1, 0); BLIP_TC_ST4(tcol + 24, b1, 8);
                BLIP_TC_ST8(tcol + 28 + 16, b2, 0); BLIP_TC_ST4(tcol + 28 + 24, b2, 8);
#undef BLIP_TC_ST8
#undef BLIP_TC_ST4
                asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
                tc_fence_before();
                __syncwarp();
                if (lane == 0) { mbar_arrive(smem_u32(&sm.tfull[t])); mbar_arrive(smem_u32(&sm.empty[s])); }
            }
            leave_item(n, false);
        }
    } else if (warp < kTcNC + kTcNE) {
        // ---- epilogue: group eg takes the units with (unit number) % 2 == eg; lane quarter sp
        const int eg = (warp - kTcNC) >> 2, sp = warp & 3;
        const unsigned tl = tbase + ((unsigned)(sp * 32) << 16) + kTcDCol0;
        unsigned ubase = 0;
        for (unsigned n = 0;; ++n) {
            load_item(n);
            if (it_nplanes < 0) break;
            const int col = it_chunk * 128 + sp * 32 + lane;
            float* const vcol = val + col;
            float* const gcol = grad + col;
            float* const lcol = lap + col;
            const bool col_ok = col < 4 * g.pitch4;
            const float oi = col_ok ? __ldg(oinv + col) : 1.0f;      // this lane's orbital: 2^-k_l
            for (unsigned u = (ubase + (unsigned)eg) & 1u; u < it_nunits; u += 2) {      // (ubase + u) % 2 == eg
                const unsigned uc = ubase + u, d = uc % kTcND;
                mbar_wait_relaxed(smem_u32(&sm.dfull[d]), (uc / kTcND) & 1u);
                tc_fence_after();
                const int4 inf = sm.info[uc % kTcNInfo];
                unsigned r[10];
                asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                             : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
                             : "r"(tl + d * 16) : "memory");
                if (MODE != 0)
                    asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0, %1}, [%2];" : "=r"(r[8]), "=r"(r[9]) : "r"(tl + d * 16 + 8) : "memory");
                else r[8] = r[9] = 0u;
                asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(smem_u32(&sm.dempty[d]));
                const int e = inf.z;
                BLIP_ASSERT(e >= 0 && (long long)e < g.M);
                float q[5];
#pragma unroll
                for (int k = 0; k < 5; ++k)
                    q[k] = (MODE != 0 || k == 0) ? __fmul_rn(__fmul_rn(__fadd_rn(__uint_as_float(r[k]), __uint_as_float(r[k + 5])), oi), scl.inv[k]) : 0.f;   // two exact power-of-two multiplies
                if (inf.x < 0)                               // non-finite position (R17): the same for the whole warp, and rare
                    asm volatile("mov.b32 %0, 0x7fc00000; mov.b32 %1, 0x7fc00000; mov.b32 %2, 0x7fc00000; mov.b32 %3, 0x7fc00000; mov.b32 %4, 0x7fc00000;"
                                 : "=f"(q[0]), "=f"(q[1]), "=f"(q[2]), "=f"(q[3]), "=f"(q[4]));
                if (!col_ok) continue;
                float gx = q[1], gy = q[2], gz = q[3];
                if (MODE == 1) {
                    gx = __fmaf_rn(g.J[0], q[1], __fmaf_rn(g.J[3], q[2], __fmul_rn(g.J[6], q[3])));
                    gy = __fmaf_rn(g.J[1], q[1], __fmaf_rn(g.J[4], q[2], __fmul_rn(g.J[7], q[3])));
                    gz = __fmaf_rn(g.J[2], q[1], __fmaf_rn(g.J[5], q[2], __fmul_rn(g.J[8], q[3])));
                }
                BLIP_ASSERT((long long)col < ld);
                if (idx32) {
                    // all element offsets of this call fit in 32 bits (the host checked M x 3 ld): one
                    // multiply-add per array instead of 64-bit pointer arithmetic
                    const unsigned o = (unsigned)e * (unsigned)ld + (unsigned)col;
                    __stcs(val + o, q[0]);
                    if (MODE != 0) {
                        const unsigned og = 3u * (unsigned)e * (unsigned)ld + (unsigned)col;
                        __stcs(grad + og, gx);
                        __stcs(grad + (og + (unsigned)ld), gy);
                        __stcs(grad + (og + 2u * (unsigned)ld), gz);
                        __stcs(lap + o, q[4]);
                    }
                } else {
                    const size_t o = (size_t)(unsigned)e * (size_t)(unsigned)ld;
                    __stcs(vcol + o, q[0]);
                    if (MODE != 0) {
                        float* const gp = gcol + 3 * o;
                        __stcs(gp, gx);
                        __stcs(gp + ld, gy);
                        __stcs(gp + 2 * ld, gz);
                        __stcs(lcol + o, q[4]);
                    }
                }
            }
            ubase += it_nunits;
            leave_item(n, false);
        }
    } else if (warp < kTcNC + kTcNE + kTcNW) {
        // ---- weight warps: warp ww takes the units with (unit number) % kTcNW == ww
        const int ww = warp - (kTcNC + kTcNE);
        float4* const rec4 = sm.wrec[ww];
        const float* const recf = reinterpret_cast<const float*>(rec4);
        unsigned ubase = 0;
        for (unsigned n = 0;; ++n) {
            load_item(n);
            if (it_nplanes < 0) break;
            const float4* rsrc = recs + (size_t)it_u0 * (kRecFloats / 4);
            unsigned u = ((unsigned)ww + kTcNW - (ubase % kTcNW)) % kTcNW;
            float4 pre = make_float4(0.f, 0.f, 0.f, 0.f);
            if (u < it_nunits && lane < kRecFloats / 4) pre = __ldg(rsrc + (size_t)u * (kRecFloats / 4) + lane);
            for (; u < it_nunits; u += kTcNW) {
                const unsigned uc = ubase + u, b = uc % kTcNB;
                __syncwarp();
                if (lane < kRecFloats / 4) rec4[lane] = pre;
                __syncwarp();
                if (u + kTcNW < it_nunits && lane < kRecFloats / 4) pre = __ldg(rsrc + (size_t)(u + kTcNW) * (kRecFloats / 4) + lane);
                const int4 loc = *reinterpret_cast<const int4*>(rec4 + 23);       // {plane in item or -1, byte offset of row (i2, i3), -, electron}
                const int y0 = loc.z >> 8, z0 = loc.z & 255;                      // the cell's offset in its 4 x 4 pencil
                BLIP_ASSERT((long long)it_u0 + u < g.M && loc.w >= 0 && (long long)loc.w < g.M);       // record and electron within the batch
                BLIP_ASSERT(loc.x < it_nplanes - 3 && loc.y >= 0 && y0 < 4 && z0 < 4);                  // block of sites inside the item's planes / pencil
                float wz[3][4];
#pragma unroll
                for (int k = 0; k < 3; ++k)
#pragma unroll
                    for (int m = 0; m < 4; ++m) wz[k][m] = recf[80 + 4 * k + m];
                if (uc >= kTcNB) mbar_wait_relaxed(smem_u32(&sm.bempty[b]), ((uc / kTcNB) & 1u) ^ 1u);
                unsigned char* const bt = sm.bt[b];
                {
                    switch (z0) {                              // the same for the whole warp: placement of the 4 fp16 at compile time
                        case 0: tc_build_tile<0, MODE>(rec4, recf, wz, scl, bt, lane); break;
                        case 1: tc_build_tile<1, MODE>(rec4, recf, wz, scl, bt, lane); break;
                        case 2: tc_build_tile<2, MODE>(rec4, recf, wz, scl, bt, lane); break;
                        default: tc_build_tile<3, MODE>(rec4, recf, wz, scl, bt, lane); break;
                    }
                }
                if (lane == 0) sm.info[uc % kTcNInfo] = make_int4(loc.x >= 0 ? (int)(it_seq0 + (unsigned)loc.x) : -1, y0, loc.w, 0);
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                __syncwarp();
                if (lane == 0) mbar_arrive(smem_u32(&sm.bfull[b]));
            }
            ubase += it_nunits;
            leave_item(n, false);
        }
    } else {
        // ---- issuers: one elected thread of warp ii takes the units with (unit number) % kTcNI == ii
        const int ii = warp - (kTcNC + kTcNE + kTcNW);
        if (tc_elect_one()) {
            unsigned ubase = 0, waited = 0, released = 0;
            const unsigned tfull0 = smem_u32(&sm.tfull[0]), tempty0 = smem_u32(&sm.tempty[0]);
            // planes < end are no longer needed by this issuer: each is handed back to the converters
            // (commit: the arrival waits for the MMAs issued so far) once it has been seen full, so
            // that every arrival belongs to the current phase of its barrier
            auto pass_upto = [&](unsigned end) {
                while (released < end) {
                    if (released >= waited) { mbar_wait(tfull0 + 8u * (released % kTcRT), (released / kTcRT) & 1u); waited = released + 1; }
                    tc_commit(tempty0 + 8u * (released % kTcRT));
                    ++released;
                }
            };
            for (unsigned n = 0;; ++n) {
                load_item(n);
                if (it_nplanes < 0) break;
                for (unsigned u = ((unsigned)ii + kTcNI - (ubase % kTcNI)) % kTcNI; u < it_nunits; u += kTcNI) {
                    const unsigned uc = ubase + u, b = uc % kTcNB, d = uc % kTcND;
                    mbar_wait(smem_u32(&sm.bfull[b]), (uc / kTcNB) & 1u);
                    const int4 inf = sm.info[uc % kTcNInfo];
                    const bool ok = inf.x >= 0;
                    const unsigned sq = (unsigned)inf.x;
                    if (ok) {
                        pass_upto(sq);
                        while (waited < sq + 4) { mbar_wait(tfull0 + 8u * (waited % kTcRT), (waited / kTcRT) & 1u); ++waited; }
                    }
                    if (uc >= kTcND) mbar_wait(smem_u32(&sm.dempty[d]), ((uc / kTcND) & 1u) ^ 1u);
                    tc_fence_after();
                    BLIP_ASSERT(!ok || (sq >= it_seq0 && sq + 4 <= it_seq0 + (unsigned)it_nplanes && sq + 4 <= waited && sq >= released &&
                                        sq + 4 - released <= kTcRT && (unsigned)inf.y < 4u));       // the unit's 4 planes: converted, not handed back, within the ring
                    if (ok) {
                        const unsigned dcol = tbase + kTcDCol0 + d * 16;
                        const uint64_t bd0 = tc_bdesc(smem_u32(&sm.bt[b][0]));
                        const unsigned ay = tbase + 4u * (unsigned)inf.y;
                        unsigned ap[4];
#pragma unroll
                        for (int m1 = 0; m1 < 4; ++m1) ap[m1] = ay + ((sq + m1) % kTcRT) * kTcPlaneCols;
#pragma unroll
                        for (int j = 0; j < 16; ++j) {
                            const int m1 = j >> 2, h = (j >> 1) & 1, part = j & 1;
                            tc_mma(dcol, ap[m1] + part * 28 + h * 8, bd0 + (uint64_t)(((m1 * 2 + h) * 512) >> 4), j > 0);
                        }
                    }
                    tc_commit(smem_u32(&sm.bempty[b]));
                    tc_commit(smem_u32(&sm.dfull[d]));
                }
                if (it_nplanes > 0) pass_upto(it_seq0 + (unsigned)it_nplanes);
                ubase += it_nunits;
                leave_item(n, true);
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" :: "r"(tbase) : "memory");
}

// max |c_l| of every orbital column l of the padded table [nrows][pitch], as the bits of a non-negative float,
// into colmax[pitch] (zero on entry).  Thread = column, CTAs stride over the rows: coalesced.
__global__ void __launch_bounds__(256) tc_colmax_kernel(const float* __restrict__ padded, long long nrows, int pitch, unsigned* __restrict__ colmax)
{
    const int l = blockIdx.y * blockDim.x + threadIdx.x;
    if (l >= pitch) return;
    unsigned m = 0;
    for (long long r = blockIdx.x; r < nrows; r += gridDim.x)
        m = max(m, __float_as_uint(__ldg(padded + (size_t)r * (size_t)pitch + l)) & 0x7fffffffu);
    if (m) atomicMax(colmax + l, m);
}

// Per-orbital power-of-two scale of the fp16 table: oscale[l] = 2^k_l with 2^k_l max|c_l| in [2^8, 2^9)
// (k_l clamped to +-kTcMaxScaleExp; 1 for an all-zero column, which the pad columns l >= L are), and
// oscale[pitch + l] = 2^-k_l for the epilogue.  Both exact.
__global__ void __launch_bounds__(256) tc_colscale_kernel(const unsigned* __restrict__ colmax, int pitch, float* __restrict__ oscale)
{
    const int l = blockIdx.x * blockDim.x + threadIdx.x;
    if (l >= pitch) return;
    const float a = __uint_as_float(colmax[l]);
    int k = 0;
    if (a > 0.f) {
        int ex;
        (void)frexpf(a, &ex);                                // a = m 2^ex, m in [0.5, 1)
        k = min(kTcMaxScaleExp, max(-kTcMaxScaleExp, 9 - ex));
    }
    oscale[l] = ldexpf(1.0f, k);
    oscale[pitch + l] = ldexpf(1.0f, -k);
}

// max |c| of the caller's table (admission to the tensor-core path: finite, below 2^100); non-finite entries set bit 31 of the result
__global__ void __launch_bounds__(256) tc_absmax_kernel(const float* __restrict__ src, long long nfloats, unsigned* __restrict__ out)
{
    unsigned m = 0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < nfloats; i += (long long)gridDim.x * blockDim.x) {
        const unsigned b = __float_as_uint(__ldg(src + i)) & 0x7fffffffu;
        m = max(m, b >= 0x7f800000u ? 0x80000000u : b);
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, d));
    if ((threadIdx.x & 31) == 0 && m) atomicMax(out, m);
}

}  // namespace blip
