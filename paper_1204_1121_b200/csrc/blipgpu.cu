// blipgpu.cu — host side of the C ABI declared in include/blipgpu.h (product path).
// Argument checking, the fp64 inverse lattice, device memory and kernel launches; every
// step of the hot path itself runs in the kernels of blip_kernels.cuh.
#include "blipgpu.h"
#include "blipgpu_dev.h"
#include "blip_host.h"
#include "blip_kernels.cuh"
#include "blip_f64.cuh"
#include "blip_tc.cuh"

#include <cmath>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>

namespace {
// Launch with programmatic stream serialization: the kernel may be set up on the device while
// its predecessor in the stream still runs; it starts with griddepcontrol.wait, which returns
// once the predecessor has completed and its writes are visible — stream order is kept, the
// launch latency between the dependent kernels of one call is hidden.
template <typename... KArgs, typename... Args>
cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t s, Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

// The staged kernel as shipped (blip::eval_staged_kernel template constants): 4 orbitals per
// lane (128 per tile row), pencils of 4 x 4 cells, a ring of 8 table planes in shared memory,
// 16 consumer warps.  The other shapes that were measured (4 x 8 pencils with a 5-plane ring;
// 8 and 12 warps) lost and are not built (round 1; profiles/r1_v3.md, in the git history up to cef06e0).
constexpr int kSVec = 4, kSBY = 4, kSBZ = 4, kSRing = 8, kSWarps = 16;
constexpr int kSC = 32 * kSVec;
using StagedShape = blip::StagedCfg<kSVec, kSBY, kSBZ, kSRing, kSWarps>;

struct StagedArgs {
    const CUtensorMap* tmap; const blip::Geom* g; const blip::StagedGeom* sg; const float4* recs;
    const int4* order; int* meta; int nchunk;
    float* val; float* grad; float* lap; long long ld;
    const float* dvec; long long ldd; float* cout;
    const double* pos; const double* kvec;
};

template <int MODE, int EPI>
cudaError_t staged_prepare1()
{
    return cudaFuncSetAttribute(blip::eval_staged_kernel<MODE, EPI, kSVec, kSBY, kSBZ, kSRing, kSWarps>,
                                cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(StagedShape::Smem));
}
template <int EPI>
cudaError_t staged_prepare_epi()
{
    cudaError_t e = staged_prepare1<0, EPI>();
    if (e == cudaSuccess) e = staged_prepare1<1, EPI>();
    if (e == cudaSuccess) e = staged_prepare1<2, EPI>();
    return e;
}
cudaError_t staged_prepare()
{
    cudaError_t e = staged_prepare_epi<blip::kEpiStore>();
    if (e == cudaSuccess) e = staged_prepare_epi<blip::kEpiContract>();
    if (e == cudaSuccess) e = staged_prepare_epi<blip::kEpiComplex>();
    return e;
}
template <int MODE, int EPI>
cudaError_t staged_launch1(unsigned nctas, cudaStream_t s, const StagedArgs& a)
{
    return launch_pdl(blip::eval_staged_kernel<MODE, EPI, kSVec, kSBY, kSBZ, kSRing, kSWarps>, nctas,
                      StagedShape::THREADS, sizeof(StagedShape::Smem), s, *a.tmap, *a.g, *a.sg, a.recs, a.order, a.meta,
                      a.nchunk, a.val, a.grad, a.lap, a.ld, a.dvec, a.ldd, a.cout, a.pos, a.kvec);
}
template <int EPI>
cudaError_t staged_launch_epi(int mode, unsigned nctas, cudaStream_t s, const StagedArgs& a)
{
    if (mode == 0) return staged_launch1<0, EPI>(nctas, s, a);
    if (mode == 2) return staged_launch1<2, EPI>(nctas, s, a);
    return staged_launch1<1, EPI>(nctas, s, a);
}
cudaError_t staged_launch(int mode, unsigned nctas, cudaStream_t s, const StagedArgs& a)
{
    if (a.dvec) return staged_launch_epi<blip::kEpiContract>(mode, nctas, s, a);
    if (a.kvec) return staged_launch_epi<blip::kEpiComplex>(mode, nctas, s, a);
    return staged_launch_epi<blip::kEpiStore>(mode, nctas, s, a);
}

// Tensor-core form of the staged kernel (blip_tc.cuh): storing epilogue only.
cudaError_t tc_prepare()
{
    cudaError_t e = cudaFuncSetAttribute(blip::eval_tc_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(blip::TcSmem));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(blip::eval_tc_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(blip::TcSmem));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(blip::eval_tc_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(blip::TcSmem));
    return e;
}
cudaError_t tc_launch(int mode, unsigned nctas, cudaStream_t s, const StagedArgs& a, const blip::TcScale& scl, long long M,
                      const float* oinv)
{
    // the epilogue addresses val / grad / lap with 32-bit element offsets when the largest one of this
    // call, (M - 1) * 3 * ld + 3 * ld - 1 (the gradient's), fits; decided here, next to the launch
    const int idx32 = (unsigned long long)M * 3ull * (unsigned long long)a.ld < (1ull << 32) ? 1 : 0;
#define BLIP_TC(MODE) launch_pdl(blip::eval_tc_kernel<MODE>, nctas, blip::kTcThreads, sizeof(blip::TcSmem), s, *a.tmap, *a.g, *a.sg, scl, \
                                 a.recs, a.order, a.meta, a.nchunk, a.val, a.grad, a.lap, a.ld, idx32, oinv)
    if (mode == 0) return BLIP_TC(0);
    if (mode == 2) return BLIP_TC(2);
    return BLIP_TC(1);
#undef BLIP_TC
}
// 2^k with 2^k * bound in (2^(target-1), 2^target]
float pow2_scale(double bound, int target)
{
    if (!(bound > 0.0) || !std::isfinite(bound)) return 1.0f;
    int ex = 0;
    (void)std::frexp(bound, &ex);                    // bound = m 2^ex, m in [0.5, 1)
    return (float)std::ldexp(1.0, target - ex);
}
}

static thread_local int g_create_cuda_error = 0;

// Inverse lattice by cofactors, G = adj(A)/det — the pinned fp64 sequence of DESIGN.md
// "Index map" (each cofactor p*q - r*s, det = (A00 C00 + A01 C01) + A02 C02, true division).
// Compiled with -ffp-contract=off on the host side.
static bool inverse_lattice(const double* A, double* G)
{
    double C[3][3];
    for (int i = 0; i < 3; ++i) {
        const int i1 = (i + 1) % 3, i2 = (i + 2) % 3;
        for (int j = 0; j < 3; ++j) {
            const int j1 = (j + 1) % 3, j2 = (j + 2) % 3;
            // cyclic form of the cofactor: sign is absorbed by the index rotation
            C[i][j] = A[3 * i1 + j1] * A[3 * i2 + j2] - A[3 * i1 + j2] * A[3 * i2 + j1];
        }
    }
    const double det = (A[0] * C[0][0] + A[1] * C[0][1]) + A[2] * C[0][2];
    if (!(det != 0.0) || !std::isfinite(det)) return false;
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) G[3 * i + j] = C[j][i] / det;
    for (int k = 0; k < 9; ++k)
        if (!std::isfinite(G[k])) return false;
    return true;
}

// Quads per lane: a warp covers nq*128 orbitals of one electron.  Larger nq amortises the
// per-column weight reads and address arithmetic over more FMAs at the cost of registers.
int blip_default_nq(int pitch4)
{
    return pitch4 <= 32 ? 1 : (pitch4 < 96 ? 2 : 3);         // measured on the 1,536-orbital table: 3 > 1 > 2
}

static int ensure_workspace(blipgpu_table* t, long long M, cudaStream_t s)
{
    if (M <= t->cap) return BLIPGPU_OK;
    CK(t, cudaStreamSynchronize(s));
    cudaFree(t->bin); cudaFree(t->perm); cudaFree(t->recs);
    t->bin = t->perm = nullptr; t->recs = nullptr; t->cap = 0;
    CK(t, cudaMalloc(&t->bin, sizeof(int) * (size_t)M));
    CK(t, cudaMalloc(&t->perm, sizeof(int) * (size_t)M));
    if (t->staged_ok) CK(t, cudaMalloc(&t->recs, sizeof(float) * blip::kRecFloats * (size_t)M));
    t->cap = M;
    return BLIPGPU_OK;
}

static bool build_tensor_map16(blipgpu_table* t, int nzp);

// The fp16-pair table of the tensor-core kernel (blip_tc.cuh) and its TMA descriptor, built from the
// padded fp32 table the first time the handle takes that path (or by blipgpu_reserve): tables that
// never see a dense batch — the 6.3 GB one of the large config — do not pay for it.  Allocates and
// synchronises, like a workspace growth.  On failure (out of memory, or a stream capture in progress)
// the handle keeps the FP32-pipe staged kernel for good: tc_ok = 0.
static bool ensure_tc_table(blipgpu_table* t, cudaStream_t s)
{
    if (t->table16) return true;
    if (!t->tc_ok) return false;
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(s, &cap) != cudaSuccess || cap != cudaStreamCaptureStatusNone) {
        (void)cudaGetLastError();
        // no allocation inside a capture: this call runs the FP32 kernel — and so do all later dense
        // batches of the handle.  Which arithmetic a handle's dense batches get is decided ONCE (here, by
        // the first of them, or ahead of time by blipgpu_reserve): the same handle and inputs return the
        // same bits whether a call is replayed from the graph or made eagerly afterwards.
        t->tc_ok = 0;
        return false;
    }
    const int nzp = (t->g.np[2] + 1) / 2;
    const long long words = (long long)t->g.np[0] * t->g.np[1] * nzp * 2 * t->pitch;
    bool fine = cudaMalloc(&t->table16, sizeof(unsigned) * (size_t)words) == cudaSuccess;
    unsigned* colmax = nullptr;                              // max |c_l| per orbital, only needed here
    const int pitch = (int)t->pitch;
    fine = fine && cudaMalloc(&t->tc_oscale, sizeof(float) * 2 * (size_t)pitch) == cudaSuccess &&
           cudaMalloc(&colmax, sizeof(unsigned) * (size_t)pitch) == cudaSuccess &&
           cudaMemsetAsync(colmax, 0, sizeof(unsigned) * (size_t)pitch, s) == cudaSuccess;
    if (fine) {
        const float* padded = reinterpret_cast<const float*>(t->table);
        const dim3 cgrid((unsigned)(t->nrows < 8LL * t->nsm ? t->nrows : 8LL * t->nsm), (unsigned)((pitch + 255) / 256));
        blip::tc_colmax_kernel<<<cgrid, 256, 0, s>>>(padded, t->nrows, pitch, colmax);
        blip::tc_colscale_kernel<<<(unsigned)((pitch + 255) / 256), 256, 0, s>>>(colmax, pitch, t->tc_oscale);
        const long long total = words / 2;
        blip::tc_table_kernel<<<(unsigned)((total + 255) / 256), 256, 0, s>>>(t->g, t->tc_oscale, nzp, padded, t->table16, total);
        fine = cudaGetLastError() == cudaSuccess && cudaStreamSynchronize(s) == cudaSuccess && build_tensor_map16(t, nzp);
    }
    cudaFree(colmax);
    if (!fine) {
        cudaFree(t->table16); cudaFree(t->tc_oscale);
        t->table16 = nullptr; t->tc_oscale = nullptr; t->tc_ok = 0;
        (void)cudaGetLastError();
    }
    return fine;
}

// TMA descriptor of the padded table for the staged kernel: 4-D tensor {pitch, n3+3, n2+3,
// n1+3} of fp32, box {C, BZ+3, BY+3, 1} (one plane of a pencil's cross-section), no swizzle,
// out-of-range elements read as zero.  cuTensorMapEncodeTiled is fetched through the runtime
// so that the library does not link against libcuda.
static bool build_tensor_map(blipgpu_table* t)
{
    typedef CUresult (*encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess ||
        qres != cudaDriverEntryPointSuccess || !fn) {
        (void)cudaGetLastError();
        return false;
    }
    const cuuint64_t pitchB = (cuuint64_t)t->pitch * sizeof(float);
    const cuuint64_t dims[4] = {(cuuint64_t)t->pitch, (cuuint64_t)t->g.np[2], (cuuint64_t)t->g.np[1],
                                (cuuint64_t)t->g.np[0]};
    const cuuint64_t strides[3] = {pitchB, pitchB * t->g.np[2], pitchB * t->g.np[2] * t->g.np[1]};
    const cuuint32_t box[4] = {(cuuint32_t)kSC, (cuuint32_t)(kSBZ + 3), (cuuint32_t)(kSBY + 3), 1u};
    const cuuint32_t estr[4] = {1u, 1u, 1u, 1u};
    const CUresult r = ((encode_fn)fn)(&t->tmap, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, t->table, dims, strides, box,
                                       estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                       CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS;
}

static bool build_tensor_map16(blipgpu_table* t, int nzp)
{
    typedef CUresult (*encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess ||
        qres != cudaDriverEntryPointSuccess || !fn) {
        (void)cudaGetLastError();
        return false;
    }
    const cuuint64_t pitchB = (cuuint64_t)t->pitch * 4;
    const cuuint64_t dims[5] = {(cuuint64_t)t->pitch, 2, (cuuint64_t)nzp, (cuuint64_t)t->g.np[1], (cuuint64_t)t->g.np[0]};
    const cuuint64_t strides[4] = {pitchB, 2 * pitchB, 2 * pitchB * nzp, 2 * pitchB * nzp * t->g.np[1]};
    const cuuint32_t box[5] = {128u, 2u, 4u, 7u, 1u};
    const cuuint32_t estr[5] = {1u, 1u, 1u, 1u, 1u};
    const CUresult r = ((encode_fn)fn)(&t->tmap16, CU_TENSOR_MAP_DATA_TYPE_UINT32, 5, t->table16, dims, strides, box,
                                       estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                       CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS;
}

extern "C" int blipgpu_create(const double* lattice, const int* grid, int norb,
                              const float* coeffs, int coeffs_on_device, void* stream,
                              blipgpu_table** out)
{
    g_create_cuda_error = 0;
    if (!lattice || !grid || !coeffs || !out) return BLIPGPU_EINVAL;
    *out = nullptr;
    if (norb < 1 || grid[0] < 4 || grid[1] < 4 || grid[2] < 4) return BLIPGPU_EINVAL;
    for (int k = 0; k < 9; ++k)
        if (!std::isfinite(lattice[k])) return BLIPGPU_EINVAL;
    const long long nsites = (long long)grid[0] * grid[1] * grid[2];
    if (nsites >= (1LL << 31)) return BLIPGPU_EINVAL;
    const long long pitch = ((long long)norb + 3) / 4 * 4;
    const long long nrows = ((long long)grid[0] + 3) * ((long long)grid[1] + 3) * ((long long)grid[2] + 3);
    // the kernels address the padded table with 32-bit float4 indices (tables up to 64 GiB)
    if (nrows >= (1LL << 31) || nrows * (pitch / 4) >= (1LL << 32)) return BLIPGPU_EINVAL;

    int dev = 0;
    cudaError_t ce = cudaGetDevice(&dev);
    cudaDeviceProp prop;
    if (ce == cudaSuccess) ce = cudaGetDeviceProperties(&prop, dev);
    if (ce != cudaSuccess) { g_create_cuda_error = (int)ce; (void)cudaGetLastError(); return BLIPGPU_ECUDA; }
    // The library holds sm_100a code only ('a' targets are not forward compatible, so 10.3 etc.
    // cannot run it); no fallback.  The attribute query fails when the device has no image.
    if (prop.major != 10 || prop.minor != 0) return BLIPGPU_EARCH;
    {
        cudaFuncAttributes fa;
        if (cudaFuncGetAttributes(&fa, blip::bin_kernel) != cudaSuccess) { (void)cudaGetLastError(); return BLIPGPU_EARCH; }
    }

    blipgpu_table* t = new (std::nothrow) blipgpu_table();
    if (!t) return BLIPGPU_ENOMEM;
    if (!inverse_lattice(lattice, t->g.G)) { delete t; return BLIPGPU_EINVAL; }
    double Jd[3][3];
    for (int a = 0; a < 3; ++a) {
        t->g.n[a] = grid[a];
        t->g.np[a] = grid[a] + 3;
        t->g.nb[a] = (grid[a] + blip::kBrick - 1) / blip::kBrick;
        for (int i = 0; i < 3; ++i) {
            Jd[a][i] = (double)grid[a] * t->g.G[3 * i + a];
            t->g.J[3 * a + i] = (float)Jd[a][i];
            t->g64.J[3 * a + i] = Jd[a][i];
        }
    }
    t->diag = 1;
    for (int a = 0; a < 3; ++a)
        for (int i = 0; i < 3; ++i)
            if (a != i && Jd[a][i] != 0.0) t->diag = 0;
    t->g.diag = t->diag;
    const int qa[6] = {0, 1, 2, 0, 0, 1}, qb[6] = {0, 1, 2, 1, 2, 2};
    for (int k = 0; k < 6; ++k) {
        t->g64.Q[k] = Jd[qa[k]][0] * Jd[qb[k]][0] + Jd[qa[k]][1] * Jd[qb[k]][1] + Jd[qa[k]][2] * Jd[qb[k]][2];
        t->g.Q[k] = (float)t->g64.Q[k];
    }
    t->L = norb;
    t->pitch = pitch;
    t->nrows = nrows;
    t->g.L = norb;
    t->g.pitch4 = (int)(pitch / 4);
    t->nsm = prop.multiProcessorCount;
    t->l2_bytes = prop.l2CacheSize;
    t->nchunk = (int)((pitch + kSC - 1) / kSC);
    t->sg.by = kSBY; t->sg.bz = kSBZ;
    t->sg.nby = (grid[1] + t->sg.by - 1) / t->sg.by;
    t->sg.nbz = (grid[2] + t->sg.bz - 1) / t->sg.bz;
    // pencil segments: whole pencils unless that leaves fewer than ~4 work items per SM
    {
        int seg = grid[0];
        const long long pencils = (long long)t->sg.nby * t->sg.nbz * t->nchunk;
        while (seg > 16 && pencils * ((grid[0] + seg - 1) / seg) < 8LL * t->nsm) seg = (seg + 1) / 2;
        t->sg.seg = seg;
    }
    t->sg.nseg = (grid[0] + t->sg.seg - 1) / t->sg.seg;
    {
        const long long nps = (long long)t->sg.nby * t->sg.nbz * t->sg.nseg;
        t->sg.nps = nps < (1LL << 24) ? (int)nps : 0;
    }
    t->nbins_direct = t->g.nb[0] * t->g.nb[1] * t->g.nb[2];
    const long long sbins = (long long)t->sg.nby * t->sg.nbz * grid[0];
    t->nbins_staged = (sbins < (1LL << 30) && t->sg.nps > 0) ? (int)sbins : 0;
    t->nbins = t->nbins_direct > t->nbins_staged ? t->nbins_direct : t->nbins_staged;
    t->nq = blip_default_nq(t->g.pitch4);

    cudaStream_t s = (cudaStream_t)stream;
    int rc = BLIPGPU_OK;
    auto fail = [&](cudaError_t e) {
        g_create_cuda_error = (int)e; (void)cudaGetLastError();
        rc = (e == cudaErrorMemoryAllocation) ? BLIPGPU_ENOMEM : BLIPGPU_ECUDA;
    };
    cudaError_t e;
    const size_t bytes = (size_t)nrows * (size_t)pitch * sizeof(float);
    const size_t src_bytes = (size_t)nsites * (size_t)norb * sizeof(float);
    float* staging = nullptr;                         // device copy of a host table, until padded
    if ((e = cudaMalloc(&t->table, bytes)) != cudaSuccess) fail(e);
    if (rc == BLIPGPU_OK && (e = cudaMalloc(&t->hist, sizeof(unsigned) * (size_t)t->nbins)) != cudaSuccess) fail(e);
    if (rc == BLIPGPU_OK && (e = cudaMalloc(&t->offs, sizeof(unsigned) * (size_t)t->nbins)) != cudaSuccess) fail(e);
    if (rc == BLIPGPU_OK && (e = cudaMemsetAsync(t->hist, 0, sizeof(unsigned) * (size_t)t->nbins, s)) != cudaSuccess) fail(e);
    if (rc == BLIPGPU_OK && (e = cudaMalloc(&t->counters, 4 * sizeof(unsigned) * (size_t)t->nbins)) != cudaSuccess) fail(e);
    if (rc == BLIPGPU_OK && (e = cudaMemsetAsync(t->counters, 0, 4 * sizeof(unsigned) * (size_t)t->nbins, s)) != cudaSuccess) fail(e);
    if (rc == BLIPGPU_OK && (e = cudaMalloc(&t->gstate, 2 * sizeof(unsigned))) != cudaSuccess) fail(e);
    if (rc == BLIPGPU_OK && (e = cudaMemsetAsync(t->gstate, 0, 2 * sizeof(unsigned), s)) != cudaSuccess) fail(e);
    if (rc == BLIPGPU_OK && (e = cudaMalloc(&t->order, sizeof(int4) * (size_t)(t->sg.nps + 1))) != cudaSuccess) fail(e);
    if (rc == BLIPGPU_OK && (e = cudaMalloc(&t->meta, sizeof(int) * 2)) != cudaSuccess) fail(e);
    if (rc == BLIPGPU_OK && !coeffs_on_device) {
        if ((e = cudaMalloc(&staging, src_bytes)) != cudaSuccess) fail(e);
        else if ((e = cudaMemcpyAsync(staging, coeffs, src_bytes, cudaMemcpyHostToDevice, s)) != cudaSuccess) fail(e);
    }
    if (rc == BLIPGPU_OK) {
        const long long total4 = nrows * (pitch / 4);
        const unsigned nblk = (unsigned)((total4 + 255) / 256);
        blip::pad_kernel<<<nblk, 256, 0, s>>>(t->g, coeffs_on_device ? coeffs : staging, t->table, total4);
        if ((e = cudaGetLastError()) == cudaSuccess) e = cudaStreamSynchronize(s);
        if (e != cudaSuccess) fail(e);
    }
    unsigned absmax_bits = 0x80000000u;               // unknown / non-finite: no tensor-core path
    if (rc == BLIPGPU_OK) {
        unsigned* d_max = nullptr;
        if (cudaMalloc(&d_max, sizeof(unsigned)) == cudaSuccess && cudaMemsetAsync(d_max, 0, sizeof(unsigned), s) == cudaSuccess) {
            blip::tc_absmax_kernel<<<(unsigned)(4 * t->nsm), 256, 0, s>>>(reinterpret_cast<const float*>(t->table), nrows * pitch, d_max);
            if (cudaMemcpyAsync(&absmax_bits, d_max, sizeof(unsigned), cudaMemcpyDeviceToHost, s) != cudaSuccess ||
                cudaStreamSynchronize(s) != cudaSuccess)
                absmax_bits = 0x80000000u;
        }
        cudaFree(d_max);
        (void)cudaGetLastError();
    }
    if (rc == BLIPGPU_OK) {
        // staged path: needs a full tile row (pitch >= C), a grid at least as large as one box,
        // the opt-in shared memory size, and the TMA descriptor
        const bool fits = t->pitch >= kSC && t->g.np[1] >= kSBY + 3 && t->g.np[2] >= kSBZ + 3 &&
                          t->nbins_staged > 0 && (size_t)prop.sharedMemPerBlockOptin >= sizeof(StagedShape::Smem);
        if (fits && build_tensor_map(t)) {
            e = staged_prepare();
            if (e == cudaSuccess) t->staged_ok = 1; else (void)cudaGetLastError();
        }
        // tensor-core form: a finite table (a NaN or Inf would reach electrons that do not touch it
        // through the zero-weight rows of an MMA) with max|c| < 2^100, and power-of-two scales that bring
        // the coefficients of every orbital to < 2^9 (per orbital, chosen on the device when the fp16
        // table is built: ensure_tc_table) and the weights of every quantity to <= 2^8 in fp16 (blip_tc.cuh);
        // 2^-kq within 2^+-26 so that 2^-(k_l + kq) is a normal fp32 for every orbital
        if (t->staged_ok && !(absmax_bits & 0x80000000u) && (size_t)prop.sharedMemPerBlockOptin >= sizeof(blip::TcSmem) &&
            tc_prepare() == cudaSuccess) {
            float amax;
            memcpy(&amax, &absmax_bits, sizeof(float));
            const double* Q = t->g64.Q;
            const double jd[3] = {t->diag ? std::fabs(Jd[0][0]) : 1.0, t->diag ? std::fabs(Jd[1][1]) : 1.0, t->diag ? std::fabs(Jd[2][2]) : 1.0};
            const double bound[5] = {1.0, jd[0], jd[1], jd[2],
                                     2.0 * (std::fabs(Q[0]) + std::fabs(Q[1]) + std::fabs(Q[2])) +
                                         4.0 * (std::fabs(Q[3]) + std::fabs(Q[4]) + std::fabs(Q[5]))};
            t->tc_scale[0] = 1.0f;
            bool fine = amax < std::ldexp(1.0f, blip::kTcMaxScaleExp);
            for (int q = 0; q < 5; ++q) {
                t->tc_scale[1 + q] = pow2_scale(bound[q], 8);
                t->tc_scale[6 + q] = 1.0f / t->tc_scale[1 + q];
                fine = fine && std::isfinite(t->tc_scale[1 + q]) && t->tc_scale[6 + q] >= std::ldexp(1.0f, -26) && t->tc_scale[6 + q] <= std::ldexp(1.0f, 26);
            }
            t->tc_ok = fine ? 1 : 0;
        }
        (void)cudaGetLastError();
    }
    if (staging) cudaFree(staging);
    if (rc == BLIPGPU_OK) {
        // one-launch grouping: needs a cooperative launch of one 1,024-thread CTA per SM and the
        // histogram (+ 1 word) in dynamic shared memory next to the kernel's static 33 KB
        int coop = 0;
        const size_t need = sizeof(unsigned) * ((size_t)t->nbins + 8) + 64 * 404;      // histogram + room to stage 64 records
        const size_t room = (size_t)prop.sharedMemPerBlockOptin - 40 * 1024;    // the attribute is per function, not per table: always the maximum
        t->fused_room = (long long)room;
        if (cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev) == cudaSuccess && coop && need <= room &&
            cudaFuncSetAttribute(blip::group_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)room) == cudaSuccess &&
            cudaFuncSetAttribute(blip::group_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)room) == cudaSuccess)
            t->fused_ok = 1;
        (void)cudaGetLastError();
    }
    if (rc != BLIPGPU_OK) { blipgpu_destroy(t); return rc; }
    *out = t;
    return BLIPGPU_OK;
}

extern "C" int blipgpu_destroy(blipgpu_table* t)
{
    if (!t) return BLIPGPU_OK;
    cudaFree(t->table); cudaFree(t->table16); cudaFree(t->tc_oscale); cudaFree(t->bin); cudaFree(t->perm); cudaFree(t->recs); cudaFree(t->hist); cudaFree(t->offs); cudaFree(t->counters); cudaFree(t->gstate);
    cudaFree(t->order); cudaFree(t->meta); cudaFree(t->kvec);
    cudaFree(t->d_pos); cudaFree(t->d_val); cudaFree(t->d_grad); cudaFree(t->d_lap); cudaFree(t->d_cell);
    for (int k = 0; k < 3; ++k) if (t->pe[k]) cudaEventDestroy(t->pe[k]);
    (void)cudaGetLastError();
    delete t;
    return BLIPGPU_OK;
}

static int check_eval_args(const blipgpu_table* t, const double* positions, long long M, int mode,
                           const float* val, const float* grad, const float* lap, long long ld)
{
    if (!t || M < 0) return BLIPGPU_EINVAL;
    if (mode != BLIPGPU_VALUE && mode != BLIPGPU_VGL && mode != BLIPGPU_VGH) return BLIPGPU_EINVAL;
    if (ld < t->L || (ld % 4) != 0) return BLIPGPU_EINVAL;
    if (M == 0) return BLIPGPU_OK;
    if (!positions || !val) return BLIPGPU_EINVAL;
    if (mode != BLIPGPU_VALUE && (!grad || !lap)) return BLIPGPU_EINVAL;
    return BLIPGPU_OK;
}

// Mode VGH (value, gradient, full Cartesian Hessian): blip::eval_full_kernel<T, 2>, T = float or double.
template <typename T>
static int launch_hess(blipgpu_table* t, const double* positions, long long M,
                       T* val, T* grad, T* hess, long long ld, int* cell, cudaStream_t s)
{
    const dim3 grid((unsigned)M, (unsigned)((t->g.pitch4 + 31) / 32));
    blip::eval_full_kernel<T, 2><<<grid, 128, 0, s>>>(t->g, t->g64, t->table, positions, M, val, grad, hess, ld, cell);
    t->launches += 1;
    t->last_path = 4;
    CK(t, cudaGetLastError());
    return BLIPGPU_OK;
}

// Which kernel serves a call (path = 0, automatic):
//   staged   M > 2,048 and every table row is wanted by >= 6 electrons on average: rows are
//            staged once on chip for all electrons of a pencil — in tensor memory, evaluated by
//            tcgen05.mma (blip::eval_tc_kernel), when the results are stored and the table is
//            finite; in shared memory, evaluated by packed FP32 FMAs (blip::eval_staged_kernel),
//            for the contraction and complex-orbital epilogues;
//   grouped  otherwise, if M > 2,048 and the table does not fit in L2: electrons sorted by
//            4x4x4-cell brick so that neighbours run together, then the direct kernel;
//   plain    otherwise (every electron of the batch is in flight at once, or L2 holds the
//            whole table: grouping cannot improve locality and costs 3 launches): caller
//            order, the split kernel up to 16,384 electrons (4 warps per electron and 128
//            orbitals: latency), the direct kernel above.
static const long long kGroupThreshold = 2048;
static const long long kSplitMax = 16384;
// The staged path pays (BY+3)(BZ+3)/(BY BZ) table rows per cell whatever the batch; it wins
// once the rows are shared by enough electrons (average number of electrons touching a row).
static const double kStagedMinReuse = 6.0;
// ... the tensor-core form spends less per electron and wins from 4.5 on (TiO2 table, L2 flushed:
// 12,288 positions = 4.8 electrons per row: 0.235 ms against 0.247 ms for the grouped direct kernel
// and 0.282 ms for the FP32-pipe staged kernel; 9,216 = 3.6: 0.224 against 0.196 ms)
static const double kStagedMinReuseTc = 4.5;

// tc: the call can take the tensor-core form (storing epilogue, finite table)
static bool use_staged(const blipgpu_table* t, long long M, bool tc)
{
    if (!t->staged_ok || t->path == 1) return false;
    if (t->path == 2 || t->path == 5) return true;
    if (M <= kGroupThreshold) return false;
    const double sites = (double)t->g.n[0] * t->g.n[1] * t->g.n[2];
    return 64.0 * (double)M / sites >= (tc ? kStagedMinReuseTc : kStagedMinReuse);
}

// dvec != NULL: contraction mode (blipgpu_eval_contract): the orbitals are not stored but
// contracted with dvec[e][.] into cout[e][0..4] (cleared by the caller of this function).
static int launch_eval(blipgpu_table* t, const double* positions, long long M, int mode,
                       float* val, float* grad, float* lap, long long ld, int* cell,
                       cudaStream_t s, const float* dvec = nullptr, long long ldd = 0, float* cout = nullptr,
                       const double* kvec = nullptr)
{
    t->g.M = M;                                              // bound of the checked build's asserts (nothing else reads it)
    if (mode == BLIPGPU_VGH)                                  // full Hessian: the per-position kernel, fp32
        return launch_hess<float>(t, positions, M, val, grad, lap, ld, cell, s);
    const int* perm = nullptr;
    const bool tc_call = t->tc_ok && !dvec && !kvec && (t->path == 0 || t->path == 5);
    const bool staged = use_staged(t, M, tc_call);
    const int kmode = mode == BLIPGPU_VALUE ? 0 : (t->diag ? 2 : 1);      // kernel template MODE
    if (t->profiling) CK(t, cudaEventRecord(t->pe[0], s));
    const bool grouped = staged || t->path == 1 ||
                         (M > kGroupThreshold && t->nrows * t->pitch * (long long)sizeof(float) > t->l2_bytes * 3 / 4);
    if (grouped && (staged || M > kGroupThreshold)) {
        int rc = ensure_workspace(t, M, s);
        if (rc != BLIPGPU_OK) return rc;
        const int nbins = staged ? t->nbins_staged : t->nbins_direct;
        if (t->fused_ok) {
            // a-4 in one cooperative launch (blip::group_kernel): count, grid barrier, scan + scatter
            cudaLaunchConfig_t cfg = {};
            cfg.gridDim = dim3((unsigned)t->nsm); cfg.blockDim = dim3(blip::kScanThreads);
            // dynamic shared memory: the histogram scan, then (staged form) as many 400-byte records
            // as fit, up to the CTA's share of the batch, + their slots
            const size_t hist_bytes = sizeof(unsigned) * (((size_t)nbins + 1 + 3) & ~(size_t)3);
            const long long share = (M + t->nsm - 2) / (t->nsm > 1 ? t->nsm - 1 : 1);
            long long nstage = ((long long)t->fused_room - (long long)hist_bytes) / (400 + 4);
            if (nstage > share) nstage = share;
            if (nstage < 1) nstage = 1;
            cfg.dynamicSmemBytes = staged ? hist_bytes + (size_t)nstage * (400 + 4) : hist_bytes;
            cfg.stream = s;
            cudaLaunchAttribute attr[1];
            attr[0].id = cudaLaunchAttributeCooperative;
            attr[0].val.cooperative = 1;
            cfg.attrs = attr; cfg.numAttrs = 1;
            if (staged)
                CK(t, cudaLaunchKernelEx(&cfg, blip::group_kernel<true>, t->g, t->sg, (int)kSC, positions, M, t->counters, t->nbins,
                                         nbins, t->gstate, t->order, t->meta, t->recs, t->perm, cell, (int)nstage));
            else
                CK(t, cudaLaunchKernelEx(&cfg, blip::group_kernel<false>, t->g, t->sg, (int)kSC, positions, M, t->counters, t->nbins,
                                         nbins, t->gstate, t->order, t->meta, t->recs, t->perm, cell, 0));
            t->launches += 1;
        } else {
        // three launches (tables whose histogram does not fit in shared memory).
        // t->hist is zero here: blipgpu_create cleared it and the scan kernel of every call puts
        // back to zero what it reads, so the call is self-contained in stream order (no host-side
        // state: a captured call can be replayed).  Only a launch failure half-way leaves it dirty.
        if (t->hist_dirty) {
            CK(t, cudaMemsetAsync(t->hist, 0, sizeof(unsigned) * (size_t)t->nbins, s));
            t->hist_dirty = 0;
        }
        const unsigned nb = (unsigned)((M + 255) / 256);
        CK(t, launch_pdl(blip::bin_kernel, nb, 256, 0, s, t->g, t->sg, staged ? 1 : 0, positions, M, t->bin, t->hist, cell));
        t->hist_dirty = 1;
        CK(t, launch_pdl(blip::scan_kernel, 1, blip::kScanThreads, 0, s, t->hist, t->offs, nbins, M, staged ? 1 : 0,
                         t->g, t->sg, t->order, t->meta));
        t->hist_dirty = 0;
        if (staged)
            CK(t, launch_pdl(blip::scatter_prep_kernel, (unsigned)((M + 127) / 128), 128, 0, s, t->g, t->sg, kSC, positions,
                             (const int*)t->bin, t->offs, M, t->recs));
        else
            CK(t, launch_pdl(blip::scatter_kernel, nb, 256, 0, s, (const int*)t->bin, t->offs, M, t->perm));
        t->launches += 3;
        }
        perm = t->perm;
        cell = nullptr;                                  // already written by bin_kernel
    }
    if (staged) {
        if (t->profiling) CK(t, cudaEventRecord(t->pe[1], s));
        const StagedArgs a = {&t->tmap, &t->g, &t->sg, t->recs, t->order, t->meta, t->nchunk,
                              val, grad, lap, ld, dvec, ldd, cout, positions, kvec};
        if ((t->path == 5 || t->path == 0) && t->tc_ok && !dvec && !kvec && ensure_tc_table(t, s)) {   // storing epilogue: on the tensor cores
            blip::TcScale scl;
            for (int q = 0; q < 5; ++q) { scl.sw[q] = t->tc_scale[1 + q]; scl.inv[q] = t->tc_scale[6 + q]; }
            StagedArgs a16 = a;
            a16.tmap = &t->tmap16;
            CK(t, tc_launch(kmode, (unsigned)t->nsm, s, a16, scl, M, t->tc_oscale + t->pitch));
            t->last_path = 5;
        } else {
            CK(t, staged_launch(kmode, (unsigned)t->nsm, s, a));
            t->last_path = 2;
        }
    } else if (t->path == 0 && !perm && M <= kSplitMax) {
        t->last_path = 3;
        if (t->profiling) CK(t, cudaEventRecord(t->pe[1], s));
        const dim3 grid((unsigned)M, (unsigned)((t->g.pitch4 + 31) / 32));
        if (kmode == 0) blip::eval_split_kernel<0><<<grid, 128, 0, s>>>(t->g, t->table, positions, perm, M, val, grad, lap, ld, dvec, ldd, cout, cell, kvec);
        else if (kmode == 2) blip::eval_split_kernel<2><<<grid, 128, 0, s>>>(t->g, t->table, positions, perm, M, val, grad, lap, ld, dvec, ldd, cout, cell, kvec);
        else blip::eval_split_kernel<1><<<grid, 128, 0, s>>>(t->g, t->table, positions, perm, M, val, grad, lap, ld, dvec, ldd, cout, cell, kvec);
    } else {
        t->last_path = 1;
        const int nq = t->nq;
        const dim3 grid((unsigned)((M + blip::kWarpsPerBlock - 1) / blip::kWarpsPerBlock),
                        (unsigned)((t->g.pitch4 + 32 * nq - 1) / (32 * nq)));
        const dim3 block(blip::kWarpsPerBlock * 32);
        if (t->profiling) CK(t, cudaEventRecord(t->pe[1], s));
#define BLIP_LAUNCH(MODE, NQ)                                                                         \
        blip::eval_direct_kernel<MODE, NQ><<<grid, block, 0, s>>>(t->g, t->table, positions, perm, M, \
                                                                  val, grad, lap, ld, dvec, ldd, cout, cell, kvec)
        if (kmode == 0) {
            if (nq == 1) BLIP_LAUNCH(0, 1); else if (nq == 2) BLIP_LAUNCH(0, 2); else BLIP_LAUNCH(0, 3);
        } else if (kmode == 2) {
            if (nq == 1) BLIP_LAUNCH(2, 1); else if (nq == 2) BLIP_LAUNCH(2, 2); else BLIP_LAUNCH(2, 3);
        } else {
            if (nq == 1) BLIP_LAUNCH(1, 1); else if (nq == 2) BLIP_LAUNCH(1, 2); else BLIP_LAUNCH(1, 3);
        }
#undef BLIP_LAUNCH
    }
    t->launches += 1;
    CK(t, cudaGetLastError());
    if (t->profiling) CK(t, cudaEventRecord(t->pe[2], s));
    return BLIPGPU_OK;
}

extern "C" int blipgpu_eval(blipgpu_table* t, const double* positions, long long M, int mode,
                            float* val, float* grad, float* lap, long long ld, int* cell,
                            void* stream)
{
    int rc = check_eval_args(t, positions, M, mode, val, grad, lap, ld);
    if (rc != BLIPGPU_OK || M == 0) return rc;
    if (((uintptr_t)val & 15) || (mode != BLIPGPU_VALUE && (((uintptr_t)grad & 15) || ((uintptr_t)lap & 15))))
        return BLIPGPU_EINVAL;
    if (M >= (1LL << 31)) return BLIPGPU_EINVAL;
    return launch_eval(t, positions, M, mode, val, grad, lap, ld, cell, (cudaStream_t)stream);
}

extern "C" int blipgpu_set_kpoints(blipgpu_table* t, const double* kpoints)
{
    if (!t) return BLIPGPU_EINVAL;
    if (!kpoints) {                                           // back to real orbitals only
        cudaFree(t->kvec);
        t->kvec = nullptr;
        return BLIPGPU_OK;
    }
    if (t->L % 2) return BLIPGPU_EINVAL;                      // a complex orbital is two adjacent real channels
    const size_t n = 3 * (size_t)(t->L / 2);
    for (size_t i = 0; i < n; ++i)
        if (!std::isfinite(kpoints[i])) return BLIPGPU_EINVAL;
    if (!t->kvec) CK(t, cudaMalloc(&t->kvec, sizeof(double) * n));
    CK(t, cudaMemcpy(t->kvec, kpoints, sizeof(double) * n, cudaMemcpyHostToDevice));
    return BLIPGPU_OK;
}

extern "C" int blipgpu_eval_complex(blipgpu_table* t, const double* positions, long long M, int mode,
                                    float* val, float* grad, float* lap, long long ld, int* cell, void* stream)
{
    if (!t || !t->kvec) return BLIPGPU_EINVAL;
    if (mode != BLIPGPU_VALUE && mode != BLIPGPU_VGL) return BLIPGPU_EINVAL;
    int rc = check_eval_args(t, positions, M, mode, val, grad, lap, ld);
    if (rc != BLIPGPU_OK || M == 0) return rc;
    if (((uintptr_t)val & 15) || (mode == BLIPGPU_VGL && (((uintptr_t)grad & 15) || ((uintptr_t)lap & 15))))
        return BLIPGPU_EINVAL;
    if (M >= (1LL << 31)) return BLIPGPU_EINVAL;
    return launch_eval(t, positions, M, mode, val, grad, lap, ld, cell, (cudaStream_t)stream, nullptr, 0, nullptr, t->kvec);
}

extern "C" int blipgpu_eval_contract(blipgpu_table* t, const double* positions, long long M, int mode,
                                     const float* d, long long ldd, float* out, int* cell, void* stream)
{
    if (!t || M < 0) return BLIPGPU_EINVAL;
    if (mode != BLIPGPU_VALUE && mode != BLIPGPU_VGL) return BLIPGPU_EINVAL;
    if (ldd < t->L || (ldd % 4) != 0) return BLIPGPU_EINVAL;
    if (M == 0) return BLIPGPU_OK;
    if (!positions || !d || !out) return BLIPGPU_EINVAL;
    if (((uintptr_t)d & 15) || ((uintptr_t)out & 15) || M >= (1LL << 31)) return BLIPGPU_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    CK(t, cudaMemsetAsync(out, 0, sizeof(float) * 8 * (size_t)M, s));
    return launch_eval(t, positions, M, mode, nullptr, nullptr, nullptr, t->pitch, cell, s, d, ldd, out);
}

extern "C" int blipgpu_eval_f64(blipgpu_table* t, const double* positions, long long M, int mode,
                                double* val, double* grad, double* lap, long long ld, int* cell, void* stream)
{
    if (!t || M < 0) return BLIPGPU_EINVAL;
    if (mode != BLIPGPU_VALUE && mode != BLIPGPU_VGL && mode != BLIPGPU_VGH) return BLIPGPU_EINVAL;
    if (ld < t->L || (ld % 4) != 0) return BLIPGPU_EINVAL;
    if (M == 0) return BLIPGPU_OK;
    if (!positions || !val || (mode != BLIPGPU_VALUE && (!grad || !lap))) return BLIPGPU_EINVAL;
    if (((uintptr_t)val & 15) || (mode != BLIPGPU_VALUE && (((uintptr_t)grad & 15) || ((uintptr_t)lap & 15))))
        return BLIPGPU_EINVAL;
    if (M >= (1LL << 31)) return BLIPGPU_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    t->g.M = M;                                              // bound of the checked build's asserts
    if (mode == BLIPGPU_VGH) return launch_hess<double>(t, positions, M, val, grad, lap, ld, cell, s);
    const dim3 grid((unsigned)M, (unsigned)((t->g.pitch4 + 31) / 32));
    if (mode == BLIPGPU_VALUE)
        blip::eval_f64_kernel<0><<<grid, 128, 0, s>>>(t->g, t->g64, t->table, positions, M, val, grad, lap, ld, cell);
    else
        blip::eval_f64_kernel<1><<<grid, 128, 0, s>>>(t->g, t->g64, t->table, positions, M, val, grad, lap, ld, cell);
    t->launches += 1;
    t->last_path = 4;
    CK(t, cudaGetLastError());
    return BLIPGPU_OK;
}

extern "C" int blipgpu_reserve(blipgpu_table* t, long long M_max)
{
    if (!t || M_max < 0 || M_max >= (1LL << 31)) return BLIPGPU_EINVAL;
    if (M_max == 0) return BLIPGPU_OK;
    if (t->tc_ok && (t->path == 0 || t->path == 5) && use_staged(t, M_max, true)) (void)ensure_tc_table(t, nullptr);
    return ensure_workspace(t, M_max, nullptr);
}

// Staging buffers of blipgpu_eval_host: full-batch device copies of positions and outputs.
static int ensure_host_staging(blipgpu_table* t, long long M, int mode, long long ld, bool want_cell,
                               cudaStream_t s)
{
    const bool fits = M <= t->hcap && ld == t->hld && (mode <= t->hmode) && (!want_cell || t->d_cell);
    if (fits) return BLIPGPU_OK;
    CK(t, cudaStreamSynchronize(s));
    cudaFree(t->d_pos); cudaFree(t->d_val); cudaFree(t->d_grad); cudaFree(t->d_lap); cudaFree(t->d_cell);
    t->d_pos = nullptr; t->d_val = t->d_grad = t->d_lap = nullptr; t->d_cell = nullptr;
    t->hcap = 0; t->hmode = -1;
    const long long cap = M;
    CK(t, cudaMalloc(&t->d_pos, sizeof(double) * 3 * (size_t)cap));
    CK(t, cudaMalloc(&t->d_val, sizeof(float) * (size_t)cap * (size_t)ld));
    if (mode != BLIPGPU_VALUE) {
        CK(t, cudaMalloc(&t->d_grad, sizeof(float) * 3 * (size_t)cap * (size_t)ld));
        CK(t, cudaMalloc(&t->d_lap, sizeof(float) * (mode == BLIPGPU_VGH ? 6 : 1) * (size_t)cap * (size_t)ld));
    }
    CK(t, cudaMalloc(&t->d_cell, sizeof(int) * 3 * (size_t)cap));
    t->hcap = cap; t->hld = ld; t->hmode = mode;
    return BLIPGPU_OK;
}

extern "C" int blipgpu_eval_host(blipgpu_table* t, const double* positions, long long M, int mode,
                                 float* val, float* grad, float* lap, long long ld, int* cell,
                                 void* stream)
{
    int rc = check_eval_args(t, positions, M, mode, val, grad, lap, ld);
    if (rc != BLIPGPU_OK || M == 0) return rc;
    if (M >= (1LL << 31)) return BLIPGPU_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    rc = ensure_host_staging(t, M, mode, ld, cell != nullptr, s);
    if (rc != BLIPGPU_OK) return rc;
    // positions in, ONE evaluation of the whole batch (the same kernels, hence the same bits, as
    // blipgpu_eval on device buffers; the staged kernel streams the table once), results out.
    // The device->host copy of psi dominates (the largest transfer in the paper's Table XI too,
    // PAPER.md:343): 20 B per evaluation over PCIe against < 1 ms of kernel time, so there is
    // nothing to gain from cutting the batch into pieces to overlap the two.
    CK(t, cudaMemcpyAsync(t->d_pos, positions, sizeof(double) * 3 * (size_t)M, cudaMemcpyHostToDevice, s));
    rc = launch_eval(t, t->d_pos, M, mode, t->d_val, mode != BLIPGPU_VALUE ? t->d_grad : nullptr,
                     mode != BLIPGPU_VALUE ? t->d_lap : nullptr, ld, cell ? t->d_cell : nullptr, s);
    if (rc != BLIPGPU_OK) return rc;
    const size_t rowb = sizeof(float) * (size_t)ld;
    CK(t, cudaMemcpyAsync(val, t->d_val, rowb * (size_t)M, cudaMemcpyDeviceToHost, s));
    if (mode != BLIPGPU_VALUE) {
        CK(t, cudaMemcpyAsync(grad, t->d_grad, 3 * rowb * (size_t)M, cudaMemcpyDeviceToHost, s));
        CK(t, cudaMemcpyAsync(lap, t->d_lap, (mode == BLIPGPU_VGH ? 6 : 1) * rowb * (size_t)M, cudaMemcpyDeviceToHost, s));
    }
    if (cell) CK(t, cudaMemcpyAsync(cell, t->d_cell, sizeof(int) * 3 * (size_t)M, cudaMemcpyDeviceToHost, s));
    CK(t, cudaStreamSynchronize(s));
    return BLIPGPU_OK;
}

extern "C" int blipgpu_info(const blipgpu_table* t, int* grid, int* norb, long long* pitch,
                            long long* table_bytes)
{
    if (!t) return BLIPGPU_EINVAL;
    if (grid) { grid[0] = t->g.n[0]; grid[1] = t->g.n[1]; grid[2] = t->g.n[2]; }
    if (norb) *norb = t->L;
    if (pitch) *pitch = t->pitch;
    if (table_bytes) *table_bytes = t->nrows * t->pitch * (long long)sizeof(float);   // ghost-padded
    return BLIPGPU_OK;
}

extern "C" const char* blipgpu_strerror(int code)
{
    switch (code) {
        case BLIPGPU_OK: return "ok";
        case BLIPGPU_EINVAL: return "invalid argument";
        case BLIPGPU_ENOMEM: return "out of memory";
        case BLIPGPU_ECUDA: return "CUDA runtime error (see blipgpu_last_cuda_error)";
        case BLIPGPU_EARCH: return "device is not compute capability 10.x (sm_100a code only, no fallback)";
        case BLIPGPU_ELIMIT: return "batch or table too large for blipgpu_eval_static's fixed workspace (BLIPGPU_STATIC_MAX_POSITIONS / _BRICKS)";
        default: return "unknown blipgpu error code";
    }
}

extern "C" int blipgpu_last_cuda_error(const blipgpu_table* t)
{
    return t ? t->last_cuda : g_create_cuda_error;
}

// ------------------------------------------------------------------------------------------------
// blipgpu_eval_static — the grouped direct-gather path of blipgpu_eval for callers that must not
// allocate device memory once they are sampling (a host code that has given the rest of the GPU
// to its own arena, or that cannot take the device-wide stall of cudaMalloc / cudaFree while its
// other streams run walkers; include/blipgpu.h has the full contract).  The same four kernels as
// launch_eval's three-launch grouping + eval_direct_kernel; what differs is where their workspace
// lives: not in the handle (cudaMalloc, grown on demand) but in the array below, which is part of
// the library image, so this entry point calls no cudaMalloc, cudaFree or allocating routine.
//
//   g_static_scratch   [hist: MAX_BRICKS u32][offs: MAX_BRICKS u32][bin: MAX_POSITIONS i32][perm: MAX_POSITIONS i32]
//                      = BLIPGPU_STATIC_BYTES (768 KiB) on every GPU that loads the library, until exit.
//
// In host code the NAME g_static_scratch is only the host-side stand-in the runtime registers the
// array under, not a device address — a kernel handed `g_static_scratch` itself would fault, or on
// a system where the GPU can reach host memory quietly use the wrong bytes.  The device address
// comes from cudaGetSymbolAddress, asked once per device with that device current and kept in
// g_static_ptr[device ordinal]; that look-up is the set-up step the header tells callers to get
// done (first call) before any stream capture.  All calls on a device share the array: the brick
// counts are cleared at the start of each call (the rest is fully rewritten before it is read),
// and calls that overlap on the GPU race — documented, not detected.
// ------------------------------------------------------------------------------------------------
static __device__ __align__(256) unsigned char g_static_scratch[BLIPGPU_STATIC_BYTES];

namespace {
constexpr int kStaticMaxDevices = 64;
constexpr size_t kStaticOffs = sizeof(unsigned) * BLIPGPU_STATIC_MAX_BRICKS;           // byte offsets into the array,
constexpr size_t kStaticBin = 2 * sizeof(unsigned) * BLIPGPU_STATIC_MAX_BRICKS;       // each a multiple of 256
constexpr size_t kStaticPerm = kStaticBin + sizeof(int) * BLIPGPU_STATIC_MAX_POSITIONS;
static_assert(kStaticPerm + sizeof(int) * BLIPGPU_STATIC_MAX_POSITIONS == BLIPGPU_STATIC_BYTES, "layout fills the array");
static_assert(kStaticOffs % 256 == 0 && kStaticBin % 256 == 0 && kStaticPerm % 256 == 0, "sub-arrays stay 256-byte aligned");

std::mutex g_static_mu;
unsigned char* g_static_ptr[kStaticMaxDevices];          // device address of g_static_scratch on device d; NULL: not asked yet

// Device address of the array on the CURRENT device (asked from the runtime the first time).
cudaError_t static_scratch_address(unsigned char** out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kStaticMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_ptr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_static_ptr[dev] = static_cast<unsigned char*>(p);
    }
    *out = g_static_ptr[dev];
    return cudaSuccess;
}
}  // namespace

extern "C" int blipgpu_eval_static(blipgpu_table* t, const double* positions, long long M, int mode,
                                   float* val, float* grad, float* lap, long long ld, int* cell, void* stream)
{
    if (mode != BLIPGPU_VALUE && mode != BLIPGPU_VGL) return BLIPGPU_EINVAL;
    int rc = check_eval_args(t, positions, M, mode, val, grad, lap, ld);
    if (rc != BLIPGPU_OK || M == 0) return rc;
    if (((uintptr_t)val & 15) || (mode == BLIPGPU_VGL && (((uintptr_t)grad & 15) || ((uintptr_t)lap & 15))))
        return BLIPGPU_EINVAL;
    const int nbins = t->nbins_direct;
    if (M > BLIPGPU_STATIC_MAX_POSITIONS || nbins > BLIPGPU_STATIC_MAX_BRICKS) return BLIPGPU_ELIMIT;

    cudaStream_t s = (cudaStream_t)stream;
    unsigned char* base = nullptr;
    CK(t, static_scratch_address(&base));
    unsigned* hist = reinterpret_cast<unsigned*>(base);
    unsigned* offs = reinterpret_cast<unsigned*>(base + kStaticOffs);
    int* bin = reinterpret_cast<int*>(base + kStaticBin);
    int* perm = reinterpret_cast<int*>(base + kStaticPerm);

    blip::Geom g = t->g;                                     // the handle's copy is left alone
    g.M = M;
    // a-4: the counts must start at zero and the array holds whatever the last call (any handle, any
    // stream) left: clear the bins of THIS table.  bin / offs / perm are written before they are read.
    CK(t, cudaMemsetAsync(hist, 0, sizeof(unsigned) * (size_t)nbins, s));
    const unsigned nb = (unsigned)((M + 255) / 256);
    blip::bin_kernel<<<nb, 256, 0, s>>>(g, t->sg, 0, positions, M, bin, hist, cell);
    blip::scan_kernel<<<1, blip::kScanThreads, 0, s>>>(hist, offs, nbins, M, 0, g, t->sg, nullptr, nullptr);
    blip::scatter_kernel<<<nb, 256, 0, s>>>(bin, offs, M, perm);
    CK(t, cudaGetLastError());
    // a-1..a-3, a-5: one warp per position in brick order, results to the caller's order (cell: done above)
    const int kmode = mode == BLIPGPU_VALUE ? 0 : (t->diag ? 2 : 1);
    const int nq = t->nq;
    const dim3 grid((unsigned)((M + blip::kWarpsPerBlock - 1) / blip::kWarpsPerBlock),
                    (unsigned)((t->g.pitch4 + 32 * nq - 1) / (32 * nq)));
    const dim3 block(blip::kWarpsPerBlock * 32);
#define BLIP_LAUNCH(MODE, NQ)                                                                         \
    blip::eval_direct_kernel<MODE, NQ><<<grid, block, 0, s>>>(g, t->table, positions, perm, M, val, grad, lap, ld, \
                                                              nullptr, 0, nullptr, nullptr, nullptr)
    if (kmode == 0) {
        if (nq == 1) BLIP_LAUNCH(0, 1); else if (nq == 2) BLIP_LAUNCH(0, 2); else BLIP_LAUNCH(0, 3);
    } else if (kmode == 2) {
        if (nq == 1) BLIP_LAUNCH(2, 1); else if (nq == 2) BLIP_LAUNCH(2, 2); else BLIP_LAUNCH(2, 3);
    } else {
        if (nq == 1) BLIP_LAUNCH(1, 1); else if (nq == 2) BLIP_LAUNCH(1, 2); else BLIP_LAUNCH(1, 3);
    }
#undef BLIP_LAUNCH
    CK(t, cudaGetLastError());
    t->launches += 4;
    t->last_path = 1;
    return BLIPGPU_OK;
}
