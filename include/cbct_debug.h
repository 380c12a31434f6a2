/* cbct_debug.h -- probes of libcbct_b200 that are NOT part of the product ABI (include/cbct.h): the launch counter and the
 * kernel timer bench.py uses for its claims, and the micro-benchmarks that measure the roofline denominators
 * MEASURED_PEAKS.json lacks.  Same conventions as cbct.h. */
#ifndef CBCT_DEBUG_H
#define CBCT_DEBUG_H

#include "cbct.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Number of kernels of this library launched by this process so far (all threads). */
long long cbct_launch_count(void);

/* Optional kernel timer.  Between _begin and _end every cbct_forward / cbct_backproject launch (also
 * those inside CGLS and the driver) is bracketed by CUDA events on its own stream.  _end waits for
 * those events and returns the summed device time in ms and the launch count, index 0 = P, 1 = P^T. */
int cbct_profile_begin(void);
int cbct_profile_end(double ms[2], int count[2]);

/* Micro-benchmarks of the per-SM rates that bound the projector kernels on the device in use (the
 * denominators MEASURED_PEAKS.json does not have).  Synchronises `stream`.  kind:
 *   0 FFMA, 1 FFMA2 (packed pair), 2 LDS.32 conflict-free, 3 ATOMS.ADD.S32 conflict-free, 4 LDG.32 hitting L1
 *     -> out[0] = warp instructions per clock per SM (clock64 inside the kernel, slowest warp of 32 per SM);
 *   7 ATOMS.ADD.64 conflict-free (256 contiguous bytes per instruction) -> warp instructions per clock per SM;
 *   5 L2 read bandwidth on a 64 MB set -> out[0] = GB/s;   6 coalesced RED.ADD.S32 into a 64 MB set -> out[0] = 1e9 reductions/s.
 * out[1] = seconds of the measured launch (CUDA events), out[2] = its work items.
 * iters: length of the timed loop (<= 0: the default, 2000; tests use a few). */
int cbct_microbench(int kind, int iters, double out[3], void *stream);

/* The direct 27 x 27-tap form of tf_reconstruct (every coefficient read 27 times): the cross-check of the separable
 * kernel behind tf_reconstruct.  Same arguments and result. */
int tf_reconstruct_direct(const float *d_alpha, float *d_f, int nx, int ny, int nz, void *stream);

/* The two kernels behind tf_apply_fused (include/cbct.h), each on its own: _tile is the 3-D shared-memory tile with
 * 27-tap sums, _march the z-marching separable kernel that reads every voxel once.  tf_apply_fused uses _march once it
 * has reproduced _tile on the device in use (one built-in problem, first call of the process; CBCT_TF_FUSED_IMPL =
 * tile | march forces a choice); _describe names the kernel in use (static storage).  Same arguments and result. */
int tf_apply_fused_tile(const float *d_in, float *d_out, float mu, int clamp_nonneg, int nx, int ny, int nz, void *stream);
int tf_apply_fused_march(const float *d_in, float *d_out, float mu, int clamp_nonneg, int nx, int ny, int nz, void *stream);
const char *tf_apply_fused_describe(void);

#ifdef __cplusplus
}
#endif
#endif /* CBCT_DEBUG_H */
