// blip_types.h — plain structs and constants shared by the device code (blip_kernels.cuh,
// blip_f64.cuh) and the two host translation units (blipgpu.cu, blipgpu_dev.cu).  No kernels here.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

// Checked build (-DBLIP_CHECKED; tests/harness builds it as libblipgpu_checked.so): every table
// row index, sorted-slot, unit, plane and output index the kernels compute is compared with its
// bound, a violation prints the expression and traps.  It stands in for compute-sanitizer's
// memcheck on a pool where that tool is closed (profiles/r2_checks.md); the shipped build has none.
#ifdef BLIP_CHECKED
#include <cstdio>
#define BLIP_ASSERT(cond)                                                                      \
    do {                                                                                       \
        if (!(cond)) {                                                                         \
            printf("BLIP_ASSERT failed: %s  (%s:%d, block %d thread %d)\n", #cond, __FILE__, __LINE__, \
                   (int)blockIdx.x, (int)threadIdx.x);                                         \
            __trap();                                                                          \
        }                                                                                      \
    } while (0)
#else
#define BLIP_ASSERT(cond) do { } while (0)
#endif

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
    int diag;           // J diagonal (lattice vectors along the Cartesian axes): the kernels' MODE 2
    long long M;        // positions of the current call: set per launch, read only by the asserts of the BLIP_CHECKED build
};

// Geometry of the staged path: pencils of BY x BZ cells running along axis 1, cut into
// segments of `seg` cell planes.  Sort key of an electron = (pencil, i1).
struct StagedGeom {
    int by, bz;         // cross-section of a pencil in cells (template constants of the kernel)
    int nby, nbz;       // pencils per axis
    int seg;            // cell planes per segment
    int nseg;           // segments per pencil = ceil(n1 / seg)
    int nps;            // pencil segments = nby * nbz * nseg (the work items, per orbital chunk)
};
constexpr int kMaxSortedItems = 8192;      // pencil segments the scan kernel can order by load

struct Geom64 {
    double J[9];        // J[a][i] = n_a G[i][a]
    double Q[6];        // J J^T: Q00 Q11 Q22 Q01 Q02 Q12
};

}  // namespace blip
