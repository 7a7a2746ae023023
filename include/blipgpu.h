/*
 * blipgpu.h — C ABI of the B200 (sm_100a) blip orbital evaluator.
 *
 * The one operation behind this boundary is the bottleneck of arxiv/paper_1204_1121
 * (Uejima & Maezono, "GPGPU for orbital function evaluation with a new updating scheme"):
 *
 *     psi_l(r_j) = sum_{s=1..64} a_{l,s(r_j)} * Theta_s(r_j)                     (Eq. 6)
 *     Theta_s(r) = phi((x-X_s)/b_x) phi((y-Y_s)/b_y) phi((z-Z_s)/b_z)            (Eq. 7)
 *
 * for every orbital l and every electron position r_j of a batch, the 64 sites s(r_j) being
 * the 4x4x4 block of the periodic coefficient grid around r_j (Eq. 8), plus
 * the Cartesian gradient and Laplacian of psi_l (needed by the local-energy call,
 * PAPER.md:124; BASELINE.json north_star).  The coefficient table is loaded once and stays
 * resident on the device; one call evaluates a batch of M positions,
 * which stands in for the paper's quasi-simultaneous update of all N electrons
 * (Eq. 11-12).
 *
 * Conventions: phi is the cardinal cubic B-spline (weights sum to 1);
 * lattice A is 3x3 row-major with row a = lattice vector a (bohr); fractional u = r.A^-1;
 * grid coordinate t_a = n_a u_a; the 4 sites along axis a are floor(t_a)-1 .. floor(t_a)+2,
 * periodic; coefficient c[k1][k2][k3][l] sits at grid point (k1,k2,k3), orbital index l
 * innermost ("l ... sequential memory access").
 *
 * Every pointer argument says HOST or DEVICE.  Nothing throws; every call returns a code.
 * There is no CPU fallback: without a CUDA device of compute capability 10.0 (B200; the
 * library holds sm_100a code only) it fails with BLIPGPU_EARCH / BLIPGPU_ECUDA.
 *
 * This header is the whole boundary.  Test and benchmark instrumentation
 * (forcing a kernel, launch counts, kernel timers, the FP32 probe) is in blipgpu_dev.h.
 */
#ifndef BLIPGPU_H
#define BLIPGPU_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct blipgpu_table blipgpu_table;       /* opaque handle: table + workspace */

/* mode */
#define BLIPGPU_VALUE 0                           /* psi only                              */
#define BLIPGPU_VGL   1                           /* psi, Cartesian gradient, Laplacian    */
#define BLIPGPU_VGH   2                           /* psi, Cartesian gradient, Cartesian Hessian (6 components) */

/* return codes */
#define BLIPGPU_OK       0
#define BLIPGPU_EINVAL  (-1)                      /* bad argument (see each call)          */
#define BLIPGPU_ENOMEM  (-2)                      /* host or device allocation failed      */
#define BLIPGPU_ECUDA   (-3)                      /* CUDA runtime error: blipgpu_last_cuda_error */
#define BLIPGPU_EARCH   (-4)                      /* current device is not compute capability 10.0 */

/*
 * blipgpu_create — load a coefficient table onto the current CUDA device.
 * ("precomputed ... stored in memory at the beginning of the simulation".)
 *
 *   lattice   HOST  [9]   row-major, row a = lattice vector a (bohr); |det| must be finite, non-zero
 *   grid      HOST  [3]   n1,n2,n3 grid points per axis, each >= 4 (fewer would alias the 4 sites)
 *   norb            L >= 1 real orbitals; a complex orbital is two adjacent real channels
 *   coeffs    HOST or DEVICE  [n1][n2][n3][L] fp32, C order, l innermost; n1*n2*n3 < 2^31
 *   coeffs_on_device      0: `coeffs` is a host pointer; 1: a device pointer
 *   stream    cudaStream_t (as void*), may be NULL; the copy is ordered on it and the call
 *             returns only after the copy has completed (the caller's buffer is not retained)
 *   out       HOST  receives the handle
 *
 * Ownership: the library keeps its own device copy, re-laid-out: row pitch padded to a
 * multiple of 4 floats and 3 periodic ghost planes per axis ((n1+3)(n2+3)(n3+3) rows), so the
 * 4x4x4 block of any cell is a box without wrap-around; the caller may free `coeffs` on
 * return.  A host table is staged through a temporary device buffer of its own size.
 * Errors: EINVAL (NULL pointer, n_a < 4, L < 1, singular / non-finite lattice, too many grid
 * points, padded table of 64 GiB or more), EARCH, ENOMEM, ECUDA.
 */
int blipgpu_create(const double* lattice, const int* grid, int norb, const float* coeffs,
                   int coeffs_on_device, void* stream, blipgpu_table** out);

/*
 * blipgpu_eval — evaluate all L orbitals at M positions (steps a-1..a-5 of SURVEY.md §8a:
 * cell map, per-axis weights, 64-row gather + FMA, grouping, output), asynchronously on
 * `stream`.  No host synchronisation, no host<->device copy inside.
 *
 *   positions DEVICE [M][3] fp64 Cartesian (bohr); any finite value (wrapped into the cell)
 *   M               >= 0; M == 0 returns OK without launching anything
 *   mode            BLIPGPU_VALUE, BLIPGPU_VGL or BLIPGPU_VGH
 *   val       DEVICE [M][ld]      fp32 out, required               val[j][l]     = psi_l(r_j)
 *   grad      DEVICE [M][3][ld]   fp32 out, required iff VGL / VGH grad[j][i][l] = d psi_l / d r_i
 *   lap       DEVICE [M][ld]      fp32 out, required iff VGL       lap[j][l]     = nabla^2 psi_l
 *             DEVICE [M][6][ld]   fp32 out, required iff VGH       lap[j][q][l]  = d2 psi_l / d r_a d r_b,
 *                                 q = 0..5 <-> (a,b) = xx, yy, zz, xy, xz, yz (the local-energy call's
 *                                 second derivatives; its trace is the Laplacian)
 *   ld              row pitch in floats: ld >= L and ld % 4 == 0.  Columns L..ld-1 are
 *                   padding; up to the next multiple of 4 they may be overwritten
 *   cell      DEVICE [M][3] int32 out, optional (NULL ok): floor(t_a) in [0,n_a) of step a-1
 *   stream    cudaStream_t (as void*), may be NULL
 *
 * Results are in the caller's position order whatever internal grouping is used.  A
 * non-finite position gives NaN outputs and cell = -1 for that position (no error code:
 * detecting it would need a synchronisation).  Output pointers must be 16-byte aligned.
 * One handle serves one stream at a time (it owns the grouping workspace); if the
 * workspace must grow the call synchronises `stream` once — blipgpu_reserve avoids that (the first
 * dense batch of a handle also builds the library's second copy of the table, the fp16 form its
 * tensor-core kernel reads; blipgpu_reserve with that batch size does it ahead of time).
 * Which kernel a handle's dense batches run is decided once, by the first of them or by
 * blipgpu_reserve: if the fp16 copy cannot be built at that moment (no memory, or the call is being
 * captured in a CUDA graph, where nothing can be allocated) the handle keeps the FP32-pipe kernel
 * for all later dense batches too, so that the same handle and inputs always return the same bits
 * (the two kernels differ in the last bits; both meet the tolerances).
 * The call keeps no state on the host between calls and leaves its device workspace as it
 * found it, so once the workspace is reserved it may be captured in a CUDA graph and
 * replayed.
 * VGH runs the per-position kernel of blipgpu_eval_f64 in fp32 (no grouping): it is meant for
 * the occasional local-energy call, not for the per-move batch.
 * Errors: EINVAL (NULL required pointer, M < 0, unknown mode, bad ld, misaligned output),
 * ENOMEM, ECUDA.
 */
int blipgpu_eval(blipgpu_table* t, const double* positions, long long M, int mode,
                 float* val, float* grad, float* lap, long long ld, int* cell, void* stream);

/*
 * blipgpu_eval_host — the same evaluation with HOST buffers: the paper's per-step data flow
 * (trial positions host->device, orbital values device->host; Fig. 4,
 * 336-343 Table XI).  Copies positions in, evaluates the whole batch with the kernels
 * blipgpu_eval would use (same bits) and copies the results out; returns after everything has
 * landed (synchronises `stream`).  The device->host copy dominates (20 B per evaluation over
 * PCIe); pinned host buffers run it at the link rate, pageable ones work but are slower.
 *
 *   positions HOST [M][3] fp64;  val/grad/lap HOST, shapes and `ld` as in blipgpu_eval
 *   (no alignment requirement);  cell HOST [M][3] int32, optional.
 */
int blipgpu_eval_host(blipgpu_table* t, const double* positions, long long M, int mode,
                      float* val, float* grad, float* lap, long long ld, int* cell, void* stream);

/*
 * blipgpu_eval_contract — evaluate and contract the orbital axis in the same pass (the step the
 * paper names as next after the orbital evaluation: the determinant update needs
 * sum_l psi_l(r'_j) (D^-1)_lj for the acceptance ratio of electron j, Eq. 11,
 * 395-399 §VI.D).  For every position j and the caller's vector d_j:
 *
 *     out[j][0]    = sum_l psi_l(r_j) d[j][l]
 *     out[j][1..3] = sum_l d psi_l / d r_i (r_j) d[j][l]   (i = x, y, z)        VGL only
 *     out[j][4]    = sum_l nabla^2 psi_l (r_j) d[j][l]                          VGL only
 *
 * The [M][L] orbitals are never written: the 20 B per evaluation of output traffic of
 * blipgpu_eval become 4 B of input.  Asynchronous on `stream` like blipgpu_eval.
 *
 *   positions DEVICE [M][3] fp64, as in blipgpu_eval;  mode BLIPGPU_VALUE (out[j][0] only) or VGL
 *   d         DEVICE [M][ldd] fp32, 16-byte aligned; ldd >= L, ldd % 4 == 0; columns >= L are ignored
 *   out       DEVICE [M][8] fp32, 16-byte aligned; entries 5..7 (1..7 for VALUE) are set to zero
 *   cell      DEVICE [M][3] int32, optional
 *
 * Sums run in fp32: over the orbitals of a lane, the lanes of a warp, then one atomic add per
 * 128-orbital tile, so the last bits depend on the order the tiles finish in.  A non-finite
 * position gives NaN in out[j][0..4].  Errors: EINVAL (NULL pointer, M < 0, bad mode / ldd,
 * misaligned d or out), ENOMEM, ECUDA.
 */
int blipgpu_eval_contract(blipgpu_table* t, const double* positions, long long M, int mode,
                          const float* d, long long ldd, float* out, int* cell, void* stream);

/*
 * blipgpu_eval_f64 — the same evaluation with fp64 weights, fp64 accumulation and fp64 outputs
 * from the resident fp32 table.  The paper keeps the local-energy evaluation in double
 * precision on the CPU because the bias of single-precision orbitals in the energy is
 * untested, and uses the fp32 values only for accept/reject; this entry
 * point lets that occasional call stay on the device.  Results agree with the fp64 definition
 * to rounding (~1e-14 relative to max|c| x weights).  It is the accuracy path, not the fast
 * one: one CTA per (position, 128 orbitals), no grouping, about 1/2 the FMA rate.
 *
 *   positions DEVICE [M][3] fp64;  mode BLIPGPU_VALUE, BLIPGPU_VGL or BLIPGPU_VGH
 *   val  DEVICE [M][ld] fp64;  grad DEVICE [M][3][ld] fp64 (VGL, VGH);
 *   lap  DEVICE [M][ld] fp64 (VGL) or [M][6][ld] fp64 (VGH: Hessian xx, yy, zz, xy, xz, yz)
 *   ld   row pitch in doubles, >= L, multiple of 4; outputs 16-byte aligned
 *   cell DEVICE [M][3] int32, optional
 *
 * Non-finite positions give NaN outputs and cell = -1.  Asynchronous on `stream`.
 * Errors: EINVAL (as blipgpu_eval), ECUDA.
 */
int blipgpu_eval_f64(blipgpu_table* t, const double* positions, long long M, int mode,
                     double* val, double* grad, double* lap, long long ld, int* cell, void* stream);

/*
 * blipgpu_set_kpoints / blipgpu_eval_complex — complex orbitals with a per-orbital Bloch phase.
 * The paper's coefficients are complex ("2 components in complex numbers"); the
 * table holds complex orbital m as the two adjacent real channels (2m, 2m+1), so that
 * u_m(r) = S_2m(r) + i S_2m+1(r) is periodic in the cell, and the orbital itself is
 *
 *     psi_m(r) = exp(i k_m . r) u_m(r),      m = 0 .. L/2 - 1
 *
 * with k_m the k-point (twist) of orbital m [the paper does not write the phase out; DESIGN.md
 * reading R8a].  blipgpu_eval_complex returns psi_m, its Cartesian gradient and Laplacian
 *     grad psi_m = e^{i k.r} (grad u_m + i k_m u_m),
 *     lap  psi_m = e^{i k.r} (lap u_m + 2 i k_m . grad u_m - |k_m|^2 u_m)
 * as interleaved (re, im) fp32 in the places of the two real channels: val[j][2m] = Re psi_m(r_j),
 * val[j][2m+1] = Im psi_m(r_j), likewise grad and lap — i.e. `val` viewed as complex64 is
 * [M][ld/2].  It is the same pass as blipgpu_eval (same kernels, same grouping); the phase is an
 * epilogue on the accumulators, k.r taken in fp64 and reduced mod 2 pi before it is rounded.
 *
 *   blipgpu_set_kpoints   kpoints HOST [L/2][3] fp64, Cartesian, rad / bohr; copied (synchronous);
 *                         NULL drops them.  EINVAL if L is odd or a component is not finite.
 *   blipgpu_eval_complex  arguments as blipgpu_eval; mode BLIPGPU_VALUE or BLIPGPU_VGL;
 *                         EINVAL also if no k-points are set.
 */
int blipgpu_set_kpoints(blipgpu_table* t, const double* kpoints);
int blipgpu_eval_complex(blipgpu_table* t, const double* positions, long long M, int mode,
                         float* val, float* grad, float* lap, long long ld, int* cell, void* stream);

/* blipgpu_reserve — pre-size the grouping workspace (bins, permutation, per-electron records)
 * for batches of up to M_max positions, so that blipgpu_eval never has to grow it (growing
 * synchronises the stream once), and, if batches of M_max positions are dense enough for the
 * staged kernels, build the fp16 copy of the table the tensor-core kernel reads (as much device
 * memory again as the table).  Optional; needed before a call is captured in a CUDA graph (a
 * capture cannot allocate: a dense call captured without it runs the FP32-pipe kernel, and the handle
 * then stays on that kernel).  The device staging buffers of blipgpu_eval_host
 * are sized by that call itself.  Errors: EINVAL, ENOMEM, ECUDA. */
int blipgpu_reserve(blipgpu_table* t, long long M_max);

/*
 * blipgpu_eval_static — blipgpu_eval for callers that must not allocate device memory while they
 * sample.  Two kinds of caller are meant.  A QMC code that, once its walkers are set up, hands
 * all remaining device memory to an arena of its own: a cudaMalloc issued by a library after that
 * point fails.  And a code that runs other walkers on other streams of the same GPU: cudaMalloc
 * and cudaFree stall the whole device until those streams drain, which such a code cannot afford
 * inside its sampling loop.  blipgpu_eval grows its grouping workspace with cudaMalloc when a
 * batch is larger than any before it (and builds the tensor-core copy of the table on the first
 * dense batch); this call never does.  It calls no cudaMalloc, cudaFree or other allocating
 * routine, whatever the batch.
 *
 * What it runs: steps a-1..a-5 as the grouped direct-gather path of blipgpu_eval — positions are
 * counted into bricks of 4x4x4 cells, a prefix sum turns the counts into slots, the positions are
 * scattered into brick order, and one warp per position gathers the 64 coefficient rows
 * (blip::bin_kernel, scan_kernel, scatter_kernel, eval_direct_kernel).  The four arrays those
 * kernels need between them (brick of each position, count and slot per brick, sorted order) do
 * not come from the handle's workspace but from ONE fixed array that is part of the library
 * image: BLIPGPU_STATIC_BYTES (768 KiB) of device memory on every GPU that loads the library,
 * held until the process exits, used or not.  The table is still the handle's: create the handle
 * with blipgpu_create during set-up, while allocating is still allowed.
 *
 *   arguments, output layout, alignment rules and non-finite positions: as blipgpu_eval;
 *   mode            BLIPGPU_VALUE or BLIPGPU_VGL (VGH uses no workspace: call blipgpu_eval)
 *   M               <= BLIPGPU_STATIC_MAX_POSITIONS, else BLIPGPU_ELIMIT
 *   the table       at most BLIPGPU_STATIC_MAX_BRICKS bricks, ceil(n1/4) ceil(n2/4) ceil(n3/4)
 *                   (every config of BASELINE.json fits; a 128^3 grid is the limit), else ELIMIT
 *
 * Results: the bits blipgpu_eval returns when it runs the direct-gather kernel (fp32 FMAs); a
 * dense batch, which blipgpu_eval gives to its tensor-core kernel, differs from that in the last
 * bits, both within the tolerances of the fp64 definition.
 *
 * Rules that come with the fixed array.
 *  - Every call on a device uses the same array, whatever the handle and the stream.  Calls that
 *    may overlap on the GPU (two streams, two host threads) race on it and return garbage: order
 *    them yourself (one stream, or events).  Calls on different GPUs are independent.
 *  - The array keeps what the previous call left in it.  The call clears the brick counts it is
 *    about to use (a memset on `stream`) before it counts; nothing else needs a clean start.
 *  - The first call on each device looks up the device address of the array (the handle's device
 *    must be current, as for every call).  That look-up is a set-up step: make the first call on
 *    a device before you begin any stream capture.  Later calls on that device only launch.
 * Errors: EINVAL (as blipgpu_eval; mode VGH), ELIMIT, ECUDA.
 */
#define BLIPGPU_ELIMIT  (-5)                      /* larger than blipgpu_eval_static's fixed array allows */
#define BLIPGPU_STATIC_MAX_POSITIONS 65536
#define BLIPGPU_STATIC_MAX_BRICKS    32768
#define BLIPGPU_STATIC_BYTES (8 * BLIPGPU_STATIC_MAX_POSITIONS + 8 * BLIPGPU_STATIC_MAX_BRICKS)
int blipgpu_eval_static(blipgpu_table* t, const double* positions, long long M, int mode,
                        float* val, float* grad, float* lap, long long ld, int* cell, void* stream);

/* blipgpu_destroy — free the table and workspace.  destroy(NULL) is a no-op returning OK. */
int blipgpu_destroy(blipgpu_table* t);

/* blipgpu_info — HOST out: grid[3], norb, internal row pitch (floats), table bytes on device.
 * Any out pointer may be NULL. */
int blipgpu_info(const blipgpu_table* t, int* grid, int* norb, long long* pitch,
                 long long* table_bytes);

/* blipgpu_strerror — static string for a return code. */
const char* blipgpu_strerror(int code);

/* blipgpu_last_cuda_error — the cudaError_t (as int) behind the last BLIPGPU_ECUDA of this
 * handle; with t == NULL, of the last failed blipgpu_create on this thread. */
int blipgpu_last_cuda_error(const blipgpu_table* t);

#ifdef __cplusplus
}
#endif
#endif /* BLIPGPU_H */
