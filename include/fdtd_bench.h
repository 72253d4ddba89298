/* fdtd_bench.h — measurement aids of libfdtd_b200, kept out of the product ABI (include/fdtd.h).
 *
 * Same shared library, separate header: these two entry points exist for bench.py's roofline block and its
 * gpu_launches count; nothing on the method's path needs them.
 */
#ifndef FDTD_B200_BENCH_H
#define FDTD_B200_BENCH_H

#include "fdtd.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Measurement aid for bench.py's roofline: launch stencil kernel `kernel_id` reps times back to back on the current
 * buffers between two CUDA events (after `warm` untimed launches) and return the mean milliseconds per launch.
 * ids: 0 fwd_e, 1 fwd_h, 2 inv_h, 3 adj_h, 4 grad_inv_e, 5 adj_e, 6 record, 7 inject_h, 8 inject_e, 9 fused forward
 * marching kernel, 10 slab kernels of the fused forward path (FDTD_ERR_UNSUPPORTED where the grid cannot fuse); 11-14 the
 * lean / row kernel of split half-step id - 11 alone, 15-18 its general (slab-box) kernel alone; 19 the fused reverse marching
 * kernel (inverse-H + inverse-E), 20 the gradient kernel alone, 21 the adjoint marching kernel, 22 the slab kernels beside it.  Ids 7 / 8 time inject as the active reverse path launches it.  Needs a reverse workspace for
 * ids >= 2 and a completed forward run for ids 6-8 (its store stays readable through any sequence of these calls).  The field
 * contents are garbage afterwards: call fdtd_reset.
 * Synchronises.  algo_bytes (may be NULL) receives the algorithmic bytes one launch moves. */
fdtd_status fdtd_profile_kernel(fdtd_sim*, int kernel_id, int warm, int reps, double* ms_per_launch, double* algo_bytes);

/* Number of kernels this library has launched on behalf of the handle since create (bench.py's gpu_launches). */
unsigned long long fdtd_launch_count(const fdtd_sim*);

/* Debugging aid standing in for compute-sanitizer (closed on the GPU pool this library is developed on).  With FDTD_WS_GUARD in
 * the flags of fdtd_workspace_bytes / fdtd_set_workspace every sub-array of the workspace is followed by a 4 KiB guard band and
 * the whole workspace starts as 0xFF bytes: a kernel that WRITES out of bounds dirties a guard band (counted here), a kernel that
 * READS a guard band or a sub-array nobody initialised picks up a NaN that reaches the fields or the gradient (caught by the
 * parity tests).  Returns the number of guard bytes that lost the pattern, -1 without a guarded workspace.  Synchronises. */
#define FDTD_WS_GUARD 4u
long long fdtd_debug_guard_check(fdtd_sim*);

#ifdef __cplusplus
}
#endif
#endif /* FDTD_B200_BENCH_H */
