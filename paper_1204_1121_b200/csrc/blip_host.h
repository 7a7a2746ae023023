// blip_host.h — the handle behind `blipgpu_table` and the error-check macro, shared by the two
// host translation units of the library: blipgpu.cu (the C ABI of include/blipgpu.h) and
// blipgpu_dev.cu (the developer / benchmark instrumentation of include/blipgpu_dev.h).
#pragma once
#include "blip_types.h"

struct blipgpu_table {
    blip::Geom g;
    blip::Geom64 g64;                // J and Q in fp64, for the fp64 kernels
    blip::StagedGeom sg;
    int L = 0;
    long long pitch = 0;             // floats per table row (multiple of 4)
    long long nrows = 0;             // rows of the padded table, (n1+3)(n2+3)(n3+3)
    float4* table = nullptr;         // device, ghost-padded [n1+3][n2+3][n3+3][pitch/4]
    int nbins = 0;                   // max(bricks, staged bins)
    int nbins_direct = 0, nbins_staged = 0;
    int nq = 1;                      // direct kernel: quads of 4 orbitals per lane (1..3)
    int diag = 0;                    // lattice vectors along the Cartesian axes: J diagonal (kernel MODE 2)
    int path = 0;                    // 0 auto, 1 direct, 2 staged (FP32 pipe), 5 staged on the tensor cores (blipgpu_set_tuning)
    int staged_ok = 0;               // TMA descriptor built and the grid is large enough
    int tc_ok = 0;                   // tensor-core form of the staged kernel usable (finite table, shared memory fits)
    unsigned* table16 = nullptr;     // device, the table of the tensor-core path: scaled fp16 halves, z pairs (blip_tc.cuh)
    CUtensorMap tmap16;              // its 5-D TMA descriptor
    float tc_scale[11] = {0};        // blip::TcScale: [1..5] 2^kq of the weights of quantity q, [6..10] 2^-kq ([0] unused)
    float* tc_oscale = nullptr;      // device [2][pitch]: 2^k_l per orbital applied to the fp16 table, and 2^-k_l (built with table16)
    int nchunk = 0;                  // staged path: orbital chunks of 128
    int nsm = 0;                     // SMs of the device (CTAs of the persistent staged kernel)
    long long l2_bytes = 0;          // L2 capacity of the device
    CUtensorMap tmap;
    int4* order = nullptr;           // [sg.nps] work items {segment, first unit, units, 0}, heaviest first
    int* meta = nullptr;             // [2] {non-empty pencil segments, work counter}
    // grouping workspace (device)
    long long cap = 0;               // electrons the workspace holds
    int* bin = nullptr;              // [cap]
    int* perm = nullptr;             // [cap]
    float4* recs = nullptr;          // [cap][24] per-electron records (staged path)
    unsigned* hist = nullptr;        // [nbins] electrons per bin; zero between calls (scan_kernel clears what it reads)
    unsigned* offs = nullptr;        // [nbins] exclusive scan of hist: where each bin starts in the sorted order
    int hist_dirty = 0;              // a grouping launch failed half-way: clear hist before the next call
    // one-launch grouping (blip::group_kernel, cooperative): two groups of {count, cursor} arrays that
    // alternate by the parity of the grid barrier's generation word, all device-side state
    unsigned* counters = nullptr;    // [4][nbins], zero at creation
    unsigned* gstate = nullptr;      // [2] {barrier arrivals, barrier generation}
    int fused_ok = 0;                // cooperative launch available and the histogram fits in shared memory
    long long fused_room = 0;        // dynamic shared memory the grouping kernel may use
    // complex orbitals (blipgpu_set_kpoints): Cartesian k of complex orbital m, device [L/2][3] fp64
    double* kvec = nullptr;
    // staging for blipgpu_eval_host (device)
    long long hcap = 0, hld = 0; int hmode = -1;
    double* d_pos = nullptr; float* d_val = nullptr; float* d_grad = nullptr; float* d_lap = nullptr;
    int* d_cell = nullptr;
    // optional timing of the kernels of the last blipgpu_eval (blipgpu_set_profiling)
    int profiling = 0;
    cudaEvent_t pe[3] = {nullptr, nullptr, nullptr};   // call start, eval kernel start, end
    int last_cuda = 0;
    int last_path = 0;               // gather+FMA kernel of the last eval: 1 direct, 2 staged, 3 split, 4 fp64/Hessian, 5 staged on the tensor cores
    long long launches = 0;
};

#define CK(t, call)                                                        \
    do {                                                                   \
        cudaError_t e_ = (call);                                           \
        if (e_ != cudaSuccess) {                                           \
            (t)->last_cuda = (int)e_;                                      \
            (void)cudaGetLastError();                                      \
            return e_ == cudaErrorMemoryAllocation ? BLIPGPU_ENOMEM : BLIPGPU_ECUDA; \
        }                                                                  \
    } while (0)
