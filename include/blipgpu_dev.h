/*
 * blipgpu_dev.h — developer / benchmark instrumentation of libblipgpu.so.
 *
 * NOT part of the boundary of SURVEY.md §8(b) (that is blipgpu.h): nothing here is needed to
 * evaluate orbitals.  These calls exist so that the tests can force each kernel, and so that
 * bench.py can report `gpu_launches`, the device time of the dominant kernel and an FP32 peak
 * measured in the same run (SURVEY.md §8d "Timing protocol").
 */
#ifndef BLIPGPU_DEV_H
#define BLIPGPU_DEV_H

#include "blipgpu.h"

#ifdef __cplusplus
extern "C" {
#endif

/* blipgpu_set_tuning — force a kernel; the defaults are chosen from the table and batch shape.
 *   path  0: automatic (staged for dense batches; else the split kernel up to 16,384 positions
 *            or the direct kernel, after grouping by cell brick when the table exceeds L2);
 *         1: always the direct-gather kernel (grouped above 2,048 positions);
 *         2: always the shared-memory staged kernel on the FP32 pipe (EINVAL if this table cannot
 *            use it: fewer than 128 orbitals, a grid smaller than one staging box, or no TMA
 *            descriptor);
 *         5: always the tensor-core staged kernel (EINVAL if the table cannot use it: as for 2, or
 *            a table with a non-finite coefficient); the contraction and complex-orbital entry
 *            points run the kernel of path 2 instead
 *   nq    direct kernel: quads of 4 orbitals per lane, 1..3; 0 restores the default.
 * The direct and the FP32 staged kernel run the same arithmetic sequence and return the same bits;
 * the tensor-core kernel multiplies exact two-term fp16 splits of coefficients and weights and
 * accumulates in fp32 in the tensor core, so its results differ from theirs in the last bits;
 * the split kernel adds the four plane partial sums last, so its results differ from theirs
 * in the last bits (all are within the stated tolerances of the fp64 definition). */
int blipgpu_set_tuning(blipgpu_table* t, int path, int nq);

/* blipgpu_probe_fp32 — measures the device's packed-FP32 FMA rate with a register-only kernel
 * (3 launches on `stream`, the last one timed; synchronises) and returns it in TFLOP/s in
 * *tflops (HOST).  For the benchmark's FP32 roofline, measured in the same run at the clocks
 * the run sees.  Errors: EINVAL, ENOMEM, ECUDA. */
int blipgpu_probe_fp32(blipgpu_table* t, double* tflops, void* stream);

/* blipgpu_last_path — which gather+FMA kernel the last blipgpu_eval / blipgpu_eval_host of this
 * handle launched: 1 direct (one warp per electron, rows from L2/HBM), 2 staged (table planes
 * through shared memory, FP32 pipe), 5 staged on the tensor cores (table planes through tensor memory), 3 split (four warps per electron, small batches), 4 the fp64 kernel of blipgpu_eval_f64; 0 before
 * any call. */
int blipgpu_last_path(const blipgpu_table* t);

/* blipgpu_launch_count — number of kernels this handle has launched since creation (the
 * benchmark's "gpu_launches" evidence).  */
long long blipgpu_launch_count(const blipgpu_table* t);

/* blipgpu_set_profiling — on != 0: every following blipgpu_eval also records CUDA events on
 * its stream at the start of the call, before and after the gather+FMA kernel (no
 * synchronisation is added).  Off by default. */
int blipgpu_set_profiling(blipgpu_table* t, int on);

/* blipgpu_last_kernel_ms — waits for the last profiled blipgpu_eval and returns the device
 * time (ms) of its grouping kernels (step a-4) and of its gather+FMA kernel (steps a-1..a-3,
 * a-5).  HOST out pointers, either may be NULL.  EINVAL if profiling is off or nothing ran. */
int blipgpu_last_kernel_ms(blipgpu_table* t, float* group_ms, float* eval_ms);

#ifdef __cplusplus
}
#endif
#endif /* BLIPGPU_DEV_H */
