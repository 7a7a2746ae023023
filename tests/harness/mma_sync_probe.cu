// mma_sync_probe.cu — harness program around mma_sync_probe.cuh: the measurement behind "tensor
// cores only if the dense recast is shown to win" (BASELINE.json north_star; PAPER.md:401-419
// §VI.E) for the mma.sync form.  Runs `units_per_sm` units (one electron x 128 orbitals:
// D[128][5] = C^T[128][64] W[64][5] from a shared-memory tile) on every SM, three ways, and prints
// their times: packed FP32 FMAs, mma.sync.m16n8k8 tf32 with the 3-term split, one tf32 term.
// Not part of libblipgpu.so (it was, as blipgpu_probe_tensor, until round 3).
//
//   usage: mma_sync_probe [units_per_sm = 1993]        (the TiO2-sized step has 1,993 units per SM)
#include "mma_sync_probe.cuh"

#include <cstdio>
#include <cstdlib>

template <int FORM>
static cudaError_t run_form(int nsm, float* out, int units_per_warp, float* ms)
{
    using namespace blip_probe;
    cudaError_t e = cudaFuncSetAttribute(mma_sync_probe_kernel<FORM>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)sizeof(ProbeSmem));
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (e == cudaSuccess) e = cudaEventCreate(&e0);
    if (e == cudaSuccess) e = cudaEventCreate(&e1);
    for (int rep = 0; rep < 3 && e == cudaSuccess; ++rep) {          // the last of three runs is timed
        e = cudaEventRecord(e0, 0);
        mma_sync_probe_kernel<FORM><<<nsm, kProbeWarps * 32, sizeof(ProbeSmem)>>>(out, units_per_warp, 1e-3f);
        if (e == cudaSuccess) e = cudaGetLastError();
        if (e == cudaSuccess) e = cudaEventRecord(e1, 0);
        if (e == cudaSuccess) e = cudaEventSynchronize(e1);
        if (e == cudaSuccess) e = cudaEventElapsedTime(ms, e0, e1);
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    return e;
}

int main(int argc, char** argv)
{
    const int units_per_sm = argc > 1 ? atoi(argv[1]) : 1993;
    if (units_per_sm < blip_probe::kProbeWarps) { fprintf(stderr, "units_per_sm must be >= %d\n", blip_probe::kProbeWarps); return 2; }
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, 0) != cudaSuccess || prop.major != 10) { fprintf(stderr, "needs an sm_100 device\n"); return 3; }
    const int nsm = prop.multiProcessorCount, upw = units_per_sm / blip_probe::kProbeWarps;
    float* out = nullptr;
    if (cudaMalloc(&out, sizeof(float) * (size_t)nsm * blip_probe::kProbeWarps * 5 * 128) != cudaSuccess) return 4;
    float ms[3] = {0.f, 0.f, 0.f};
    cudaError_t e = run_form<0>(nsm, out, upw, &ms[0]);
    if (e == cudaSuccess) e = run_form<1>(nsm, out, upw, &ms[1]);
    if (e == cudaSuccess) e = run_form<2>(nsm, out, upw, &ms[2]);
    cudaFree(out);
    if (e != cudaSuccess) { fprintf(stderr, "CUDA error: %s\n", cudaGetErrorString(e)); return 1; }
    printf("mma_sync_probe: units_per_sm %d  fp32_ffma2 %.4f ms  tf32x3_mma_sync %.4f ms  tf32x1_mma_sync %.4f ms\n",
           upw * blip_probe::kProbeWarps, ms[0], ms[1], ms[2]);
    return 0;
}
