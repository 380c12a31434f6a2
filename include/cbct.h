/* cbct.h -- C ABI of the B200-native (sm_100a) hot path of tight-frame-regularised cone-beam CT
 * reconstruction (arxiv/paper_1008_2042: Jia, Dong, Lou, Jiang).
 *
 * Citations are "/root/reference/PAPER.md:<line> (section / equation)" plus the reading of
 * SURVEY.md §8(c) where the paper is silent.  All kernels are hand-written CUDA for sm_100a;
 * there is NO CPU fallback and no other backend: on a device that is not compute capability 10.x
 * every entry point that would launch a kernel returns CBCT_E_UNSUPPORTED.
 *
 * Conventions (all entry points)
 *   - Lengths in mm, angles in rad.  Volumes are f[z][y][x] (x fastest), projections g[view][v][u]
 *     (u fastest), tight-frame coefficients alpha[27][z][y][x] with band i = l + 3m + 9n (l on x).
 *     Everything is contiguous fp32.
 *   - Pointers named d_* are DEVICE pointers, 16-byte aligned, owned by the caller (e.g. a PyTorch
 *     tensor's data_ptr()).  Pointers named h_* are HOST pointers.  `stream` is a cudaStream_t passed
 *     as void* (NULL = the legacy default stream).
 *   - in and out must not alias unless a function says "in place".  Outputs are overwritten.
 *   - Hot calls are asynchronous on `stream`, allocate nothing and never synchronise the host; they
 *     return launch errors only.  Handles own their device workspace (allocated at *_create / *_prepare).
 *   - A handle's workspace is used by every call on it: ONE call in flight per handle (calls on the same
 *     stream are ordered and therefore fine; two streams or threads sharing a handle are not).
 *   - Return value: 0 = CBCT_OK, < 0 = error, CBCT_BREAKDOWN (+1) = CGLS breakdown (not a failure;
 *     SURVEY.md §8(b) calls it CBCT_E_BREAKDOWN, the E_ is dropped here because it is not an error).
 *     Nothing throws or aborts.
 *   - No kernel of this library waits without a bound or indexes shared memory unchecked: a TMA copy that never
 *     arrives, or a sampling box that does not cover its samples, raises the handle's device error word
 *     (cbct_geometry_status) and the kernel leaves through its normal exit path; every later call on the handle
 *     returns CBCT_E_DEVICE until the word is cleared.
 *   - Which kernel variant serves a handle is decided once, in cbct_geometry_create (cbct_geometry_describe reports
 *     it).  The selection variables below are read THERE and nowhere else; they exist for tests and A/B timing:
 *       CBCT_FORWARD_IMPL = tma | tiled | global      CBCT_BACKPROJECT_IMPL = scatter | cell | gather
 *       CBCT_FW_PACKED = 0|1   CBCT_BT_PACKED = 0|1   (packed fp32-pair or scalar instruction stream)
 *       CBCT_BT_LANES = 0|1    (lane layout of the scatter kernel)
 *     (tf_apply_fused has a process-wide selection of the same kind, CBCT_TF_FUSED_IMPL: see there.)
 *     A forced implementation that the geometry cannot use makes cbct_geometry_create fail (CBCT_E_UNSUPPORTED);
 *     nothing falls back silently at launch time.
 */
#ifndef CBCT_H
#define CBCT_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
    CBCT_OK = 0,
    CBCT_E_INVALID = -1,      /* bad argument (null pointer, non-positive size, geometry rejected) */
    CBCT_E_UNSUPPORTED = -2,  /* no sm_100-class device / feature not available */
    CBCT_E_CUDA = -3,         /* a CUDA runtime call failed; see cbct_last_cuda_error() */
    CBCT_E_DEVICE = -4,       /* a kernel raised the handle's device error word; see cbct_geometry_status() */
    CBCT_BREAKDOWN = 1        /* CGLS: gamma == 0 or ||q||^2 == 0 (PAPER.md:446, :461 would divide by 0) */
};
/* bits of the device error word (cbct_geometry_status) */
enum {
    CBCT_STATUS_WAIT_TIMEOUT = 1,       /* a bounded mbarrier wait expired (TMA copy never completed) */
    CBCT_STATUS_FORWARD_RANGE = 2,      /* cbct_forward: a thread's samples left the staged box (skipped, not read) */
    CBCT_STATUS_BACKPROJECT_RANGE = 4,  /* cbct_backproject: a thread's samples left the accumulator box (skipped) */
    CBCT_STATUS_FIXED_POINT_RANGE = 8   /* cbct_backproject: an int32 accumulator reached 2^30, half its range: the head-room
                                           plan (cbct_backproject_fixed_point_plan) does not hold for this geometry / input */
};

/* Static string for a status code. */
const char *cbct_status_string(int status);
/* Raw cudaError_t of the last CBCT_E_CUDA seen on the calling thread (0 if none). */
int cbct_last_cuda_error(void);
/* Library version, e.g. 100 = 1.0.0. */
int cbct_version(void);
/* (Probes -- launch counter, kernel timer, micro-benchmarks -- are declared in cbct_debug.h.) */

/* ------------------------------------------------------------------------------------------------
 * Geometry: circular orbit, flat panel (Eq. 1, Fig. 1 caption).
 * Frame (the figure itself is missing from the paper text): origin = isocentre,
 * z = rotation axis, source x_S = (SAD cos th, SAD sin th, 0), detector centre
 * c_D = -(SDD-SAD)(cos th, sin th, 0), e_u = (-sin th, cos th, 0), e_v = (0,0,1).
 * Voxel centre x = ox + (ix-(nx-1)/2) dx; pixel centre u = u0 + (iu-(nu-1)/2) du.  One ray per pixel
 * centre.
 * ---------------------------------------------------------------------------------------------- */
typedef struct {
    int32_t nx, ny, nz;       /* volume size in voxels */
    double dx, dy, dz;        /* voxel pitch */
    double ox, oy, oz;        /* volume centre offset from the isocentre */
    int32_t nu, nv;           /* detector size in pixels */
    double du, dv;            /* pixel pitch */
    double u0, v0;            /* detector centre offset */
    double sad, sdd;          /* source-axis and source-detector distance */
    int32_t n_views;
    const double *angles;     /* HOST array[n_views]; copied at create */
    double step_mm;           /* sampling step; <= 0 selects 0.5*min(dx,dy,dz) */
} cbct_geometry_desc;

typedef struct cbct_geometry cbct_geometry; /* opaque; owns device-side per-view tables + workspace */

/* Validates and builds a geometry handle on the current CUDA device.
 * CBCT_E_INVALID: null pointers, non-positive sizes/pitches, sad <= 0, sdd <= sad, or the padded
 * volume's bounding radius R >= SAD (source inside the volume).  Synchronous; allocates. */
int cbct_geometry_create(const cbct_geometry_desc *desc, cbct_geometry **out);
int cbct_geometry_destroy(cbct_geometry *geom);

/* Derived quantities (any out pointer may be NULL):
 *   n_vox, n_rays; K, t_min, step_mm of the global sample grid t_k = t_min + (k+1/2) step,
 *   t_min = SAD - R, K = ceil(2R/step), R = half-diagonal of the zero-padded box;
 *   n_samples_algorithmic = sum over rays of chord(padded box)/step (the unit of "Gsamples/s");
 *   workspace_bytes = device memory owned by the handle. */
int cbct_geometry_info(const cbct_geometry *geom, int64_t *n_vox, int64_t *n_rays, int32_t *K,
                       double *t_min, double *step_mm, int64_t *n_samples_algorithmic,
                       size_t *workspace_bytes);

/* The kernels that serve this handle, as text, e.g.
 *   "forward: forward_tma_kernel<40,30,scalar> box 40x30x7; backproject: backproject_scatter_kernel<40,30,LM1,scalar> ..."
 * written to buf (NUL-terminated, truncated to cap).  Host only. */
int cbct_geometry_describe(const cbct_geometry *geom, char *buf, size_t cap);

/* Device error word of the handle.  Synchronises `stream`, stores the CBCT_STATUS_* bits raised by kernels of this
 * handle since the last clear in *flags (may be NULL), clears the word if `clear` != 0.
 * Returns CBCT_OK if no bit was set, CBCT_E_DEVICE otherwise. */
int cbct_geometry_status(cbct_geometry *geom, void *stream, int *flags, int clear);

/* g = P f.  PAPER.md:73 Eq. 1 discretised as step * sum_k T[f](x_S + n t_k), T = zero-padded
 * trilinear interpolation (north_star).  d_vol: nx*ny*nz, d_proj: n_views*nv*nu. */
int cbct_forward(const cbct_geometry *geom, const float *d_vol, float *d_proj, void *stream);

/* f = P^T g, the exact matrix transpose of cbct_forward ("f = P^T g"; north_star),
 * deterministic (bit-identical from call to call).  d_proj: n_views*nv*nu, d_vol: nx*ny*nz, finite values.
 * Where nx and ny are multiples of 4 and the sampling box fits shared memory the transpose is evaluated
 * ray-driven with fixed-point shared-memory accumulators (error per contribution <= max|g| / 2^(qb+1), see
 * cbct_backproject_fixed_point_plan); otherwise voxel-driven in fp32 without atomics. */
int cbct_backproject(const cbct_geometry *geom, const float *d_proj, float *d_vol, void *stream);

/* The paper's own backprojector, Eq. 3: f(x) = (dx dy dz)/(du dv) sum_theta L^3(u*)/(L0 l^2(x)) g(u*),
 * g(u*) bilinear, zero outside the imager.  An APPROXIMATE adjoint of cbct_forward ("numerical error
 * less than 1%"); provided for matched/unmatched comparisons, never used by cbct_cgls_*.
 * Same buffers and conventions as cbct_backproject. */
int cbct_backproject_eq3(const cbct_geometry *geom, const float *d_proj, float *d_vol, void *stream);

/* The paper's OWN forward projector, PAPER.md:191 ("the line integral of Eq. (1) along an x-ray line using Siddon's
 * ray-tracing algorithm"; also PAPER.md:211, :256), and its exact transpose:
 *   g[ray] = sum over voxels |ray INTERSECT voxel| * f[voxel]   (lengths in mm),
 * the volume being piecewise constant on the boxes [xb + ix dx, xb + (ix+1) dx] x ..., xb = ox - nx dx / 2, the ray the
 * segment from the source to the pixel centre.  No sampling step: geom's step_mm is not used.  A second matched pair
 * next to cbct_forward / cbct_backproject (which are the fixed-step trilinear pair north_star prescribes); CGLS in this
 * library uses the trilinear pair.  Buffers and conventions as cbct_forward / cbct_backproject; outputs overwritten.
 * cbct_siddon_prepare allocates the pair's workspace (a y-fastest volume copy, two int32 accumulator volumes; synchronous)
 * and must be called once per handle before the two hot calls, which return CBCT_E_INVALID otherwise and, like every hot
 * call, allocate nothing.  cbct_siddon_backproject accumulates in fixed point relative to max|g| (deterministic,
 * error per contribution <= max|g| / 2^(qb+1) mm with qb >= 9 chosen from a bound on the path length one voxel can
 * collect); CBCT_E_UNSUPPORTED if no qb satisfies the bound. */
int cbct_siddon_prepare(cbct_geometry *geom);
int cbct_siddon_forward(const cbct_geometry *geom, const float *d_vol, float *d_proj, void *stream);
int cbct_siddon_backproject(const cbct_geometry *geom, const float *d_proj, float *d_vol, void *stream);

/* Host arithmetic only: the fixed-point plan of cbct_siddon_backproject.  max_path_sum_per_view bounds the path length
 * (mm) one voxel can collect from one view: (pixels its shadow can touch at the nearest depth) x (voxel diagonal);
 * views_per_group * max_path_sum_per_view * 2^qb < 2^31.  CBCT_E_UNSUPPORTED if no qb >= 9 fits one view. */
int cbct_siddon_fixed_point_plan(const cbct_geometry_desc *desc, int32_t *qb, int32_t *views_per_group, double *max_path_sum_per_view);

/* Host arithmetic only (no device needed): the fixed-point plan cbct_backproject uses for this geometry.
 *   max_weight_sum_per_view: planned bound on the sum of trilinear weights one voxel receives from one view
 *                    (1.25 x the largest continuum sample density x the under-sampling excess per axis; pinned
 *                    against the oracle's exact sums in tests/test_abi.py);
 *   qb: contributions are rounded to multiples of max|g| / 2^qb;
 *   views_per_group: views accumulated in int32 before conversion to fp32:
 *                    views_per_group * max_weight_sum_per_view * 2^qb <= 2^30, HALF the int32 range.  The conversion
 *                    pass raises CBCT_STATUS_FIXED_POINT_RANGE if any accumulator reaches 2^30, so a geometry that
 *                    exceeds the planned bound by up to 3x is reported (cbct_geometry_status), never wrapped silently.
 * Any out pointer may be NULL.  CBCT_E_INVALID as cbct_geometry_create; CBCT_E_UNSUPPORTED if no plan exists. */
int cbct_backproject_fixed_point_plan(const cbct_geometry_desc *desc, int32_t *qb, int32_t *views_per_group,
                                      double *max_weight_sum_per_view);

/* Host-buffer variants (used for end-to-end timing): copy h_in -> device workspace, run, copy the
 * result to h_out, all on `stream`; the caller synchronises the stream.  Pinned host memory makes
 * the copies asynchronous. */
int cbct_forward_host(cbct_geometry *geom, const float *h_vol, float *h_proj, void *stream);
int cbct_backproject_host(cbct_geometry *geom, const float *h_proj, float *h_vol, void *stream);

/* ------------------------------------------------------------------------------------------------
 * CGLS (Appendix 1).  State vectors x, p (volume size) and r (projection size) are
 * the caller's; the handle owns q (projection size), s (volume size) and the fp64 device scalars.
 * ---------------------------------------------------------------------------------------------- */
typedef struct cbct_cgls cbct_cgls;
int cbct_cgls_create(const cbct_geometry *geom, cbct_cgls **out);
int cbct_cgls_destroy(cbct_cgls *cg);

/* Initialize: r = g - P x0; p = s = P^T r; gamma = ||s||^2.  d_x holds x0. */
int cbct_cgls_init(cbct_cgls *cg, const float *d_g, const float *d_x, float *d_r, float *d_p, void *stream);

/* One pass through steps 1-7: q = P p; alpha = gamma/||q||^2; x += alpha p;
 * r -= alpha q; s = P^T r; gamma' = ||s||^2; beta = gamma'/gamma; p = s + beta p.
 * All scalars stay on the device (fp64).  On breakdown (gamma == 0 or ||q||^2 == 0) the step leaves
 * x, r, p unchanged and sets the device flag; still returns CBCT_OK because
 * the host is never synchronised here -- read the flag with cbct_cgls_scalars. */
int cbct_cgls_step(cbct_cgls *cg, float *d_x, float *d_r, float *d_p, void *stream);

/* Synchronises `stream` and copies out {gamma, ||q||^2, alpha, beta, ||r||^2}.  ||r||^2 is computed
 * here from d_r if d_r != NULL, else reported as -1 (the residual belongs to the caller, so it is an
 * argument here; SURVEY.md §8(b) sketched the call without it).  Returns CBCT_BREAKDOWN if the flag is set. */
int cbct_cgls_scalars(cbct_cgls *cg, const float *d_r, double out[5], void *stream);

/* ------------------------------------------------------------------------------------------------
 * Piecewise-linear tight frame: h0 = 1/4[1,2,1], h1 = sqrt(2)/4[1,0,-1],
 * h2 = 1/4[-1,2,-1]; psi_i = h_l(x) h_m(y) h_n(z); alpha_i = psi_i (*) f (true convolution),
 * edge-replicate extension of f; D^T is the exact transpose.
 * ---------------------------------------------------------------------------------------------- */
int tf_decompose(const float *d_f, float *d_alpha, int nx, int ny, int nz, void *stream);
/* Vector shrinkage T_mu, Eq. 2, in place on bands 1..26 (band 0 untouched);
 * factor max(1 - mu/||alpha_h||, 0), := 0 where ||alpha_h|| = 0. */
int tf_shrink(float *d_alpha, float mu, int nx, int ny, int nz, void *stream);
/* f = D^T alpha = sum_i psi_i(-x) (*) alpha_i. */
int tf_reconstruct(const float *d_alpha, float *d_f, int nx, int ny, int nz, void *stream);
/* f_out = [H] D^T T_mu D f_in without materialising alpha (H = max(.,0), PAPER.md:131,
 * applied when clamp_nonneg != 0).  d_in != d_out.
 * Two kernels compute it (cbct_debug.h exposes each): a 3-D shared-memory tile and a z-marching separable one that
 * reads every voxel once.  The marching kernel serves this call once it has reproduced the tile kernel on the device in
 * use; that one-off check (a 45x37x11 built-in volume) runs inside the first call of the process -- or earlier, inside
 * cbct_recon_create -- and synchronises the device then; no later call does.  CBCT_TF_FUSED_IMPL = tile | march (read
 * once, at that point) forces a choice. */
int tf_apply_fused(const float *d_in, float *d_out, float mu, int clamp_nonneg, int nx, int ny, int nz,
                   void *stream);

/* ------------------------------------------------------------------------------------------------
 * The paper's COMPARISON regulariser: total variation through the Rudin-Osher-Fatemi
 * sub-problem:  f = argmin ||f - u||^2 + mu_tv ||f||_TV  "by a simple gradient descent method ...
 * with an adaptively adjusted step length", stopped when the energy decreases by less than rel_tol (the paper: 0.1 %).
 * Discretisation (the paper gives none; DESIGN.md §1b T1-T6): forward differences, zero across the last faces;
 * isotropic TV smoothed as sqrt(|Df|^2 + eps^2), eps > 0 in the units of f; a trial step f - tau grad E is accepted
 * iff it lowers E (tau *= 1.2, else tau /= 2; tau starts at 0.25, f at u); stop at the first accepted step with
 * (E_k - E_k+1)/E_k < rel_tol, after max_iter trials, or at once if E(u) = 0.  The control state lives in device
 * memory: asynchronous on `stream`, nothing is read back.  clamp_nonneg != 0 applies H = max(.,0) to the result.
 * d_work: caller-owned device scratch of tv_rof_workspace_bytes(nx,ny,nz) bytes (256-byte aligned).  d_u != d_f.
 * tv_rof_result synchronises `stream` and reports the trials used, the accepted steps and the final energy.
 * ---------------------------------------------------------------------------------------------- */
size_t tv_rof_workspace_bytes(int nx, int ny, int nz);
int tv_rof(const float *d_u, float *d_f, void *d_work, float mu_tv, float eps, int max_iter, float rel_tol,
           int clamp_nonneg, int nx, int ny, int nz, void *stream);
int tv_rof_result(const void *d_work, int nx, int ny, int nz, int *trials, int *accepted, double *energy, void *stream);

/* ------------------------------------------------------------------------------------------------
 * Multigrid transfers (§2.2.3).  Per-axis factors fx,fy,fz in {1,2}; fine sizes must be
 * divisible.  restrict = mean of the children; prolong = cell-centred linear interpolation (weights
 * 3/4, 1/4, neighbour clamped at the faces).
 * ---------------------------------------------------------------------------------------------- */
int mg_restrict(const float *d_fine, float *d_coarse, int nx_f, int ny_f, int nz_f, int fx, int fy, int fz,
                void *stream);
int mg_prolong(const float *d_coarse, float *d_fine, int nx_f, int ny_f, int nz_f, int fx, int fy, int fz,
               void *stream);

/* Algorithm A2 step 1 (garbled; reading of SURVEY.md §8(c) item 11):
 * v = f_cur + coef (f_cur - f_prev), coef = (t^(k-1) - 1)/t^(k).  n = element count. */
int cbct_a2_extrapolate(const float *d_f_cur, const float *d_f_prev, float *d_v, float coef, int64_t n,
                        void *stream);

/* ------------------------------------------------------------------------------------------------
 * Driver: Algorithm A2 inside the coarse-to-fine multigrid cascade
 * (PAPER.md:232): levels coarsen x,y by 2 each, z kept, g at full resolution; n_outer[] is
 * coarse -> fine (PAPER.md:288 uses 5/10/15); n_cgls passes of CGLS steps 1-7 per outer iteration
 * ("M = 2~3"); one mu for all levels; momentum = 0 gives Algorithm A1.
 * d_f receives the finest-level volume.
 * ---------------------------------------------------------------------------------------------- */
typedef struct cbct_recon cbct_recon; /* opaque; owns per-level geometry, CGLS state and volumes */
/* Allocates everything the cascade needs (finest nx, ny must be divisible by 2^(n_levels-1)). */
int cbct_recon_create(const cbct_geometry_desc *finest, int n_levels, cbct_recon **out);
/* Same with options.  CBCT_RECON_BIN_DETECTOR: the level whose voxels are coarsened by a
 * factor c in x,y works on projections binned by c (every c x c block of pixels replaced by its mean, pixel pitch
 * x c, same detector centre; nu, nv must be divisible by 2^(n_levels-1)) -- the paper coarsens only the volume
 * (PAPER.md:232 is silent on the data; reading of SURVEY.md §8(c) item 21), binning divides the rays of a coarse
 * level by c^2.  The finest level always uses the full-resolution data. */
enum { CBCT_RECON_BIN_DETECTOR = 1, CBCT_RECON_TV = 2 /* also allocate the workspace cbct_recon_run_tv needs */ };
int cbct_recon_create_ex(const cbct_geometry_desc *finest, int n_levels, unsigned flags, cbct_recon **out);
int cbct_recon_destroy(cbct_recon *recon);
/* Runs the cascade asynchronously on `stream` (no allocation, no host synchronisation). */
int cbct_recon_run(cbct_recon *recon, const float *d_g, float *d_f, const int *n_outer, int n_cgls, float mu,
                   int momentum, void *stream);
/* The TV comparison algorithm of PAPER.md:236 on the same cascade: as cbct_recon_run, with the tight-frame shrinkage of
 * every outer iteration replaced by tv_rof(mu_tv, eps, max_rof_iter, rel_tol) followed by H.  The handle must have been
 * created with CBCT_RECON_TV (CBCT_E_INVALID otherwise). */
int cbct_recon_run_tv(cbct_recon *recon, const float *d_g, float *d_f, const int *n_outer, int n_cgls, float mu_tv,
                      float eps, int max_rof_iter, float rel_tol, int momentum, void *stream);
/* HOST buffers: h_g -> device, run, volume -> h_f; synchronises `stream` before returning. */
int cbct_recon_run_host(cbct_recon *recon, const float *h_g, float *h_f, const int *n_outer, int n_cgls,
                        float mu, int momentum, void *stream);

/* Device error words of the per-level geometry handles, ORed (cbct_geometry_status); synchronises `stream`. */
int cbct_recon_status(cbct_recon *recon, void *stream, int *flags, int clear);
/* The kernels serving the finest level (cbct_geometry_describe). */
int cbct_recon_describe(const cbct_recon *recon, char *buf, size_t cap);

/* One-shot convenience wrappers: create + run + synchronise + destroy.  A raised device error word is returned as
 * CBCT_E_DEVICE. */
int cbct_tf_reconstruct(const cbct_geometry_desc *finest, const float *d_g, float *d_f, int n_levels,
                        const int *n_outer, int n_cgls, float mu, int momentum, void *stream);
/* Same with HOST buffers: copies h_g to the device, reconstructs, copies the volume back to h_f. */
int cbct_tf_reconstruct_host(const cbct_geometry_desc *finest, const float *h_g, float *h_f, int n_levels,
                             const int *n_outer, int n_cgls, float mu, int momentum, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* CBCT_H */
