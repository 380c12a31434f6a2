// common.cuh -- internal declarations shared by the CUDA translation units of libcbct_b200.
// Nothing in this directory is shared with oracle/ (the fp64 checker) and vice versa.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <vector>

#include "../../include/cbct.h"

namespace cbct {

// ---- error plumbing -------------------------------------------------------------------------
int set_cuda_error(cudaError_t e);          // records e for cbct_last_cuda_error(), returns CBCT_E_CUDA
int device_supported();                     // CBCT_OK on a compute-capability-10.x device
#define CBCT_CUDA_TRY(expr)                                        \
    do {                                                           \
        cudaError_t _e = (expr);                                   \
        if (_e != cudaSuccess) return ::cbct::set_cuda_error(_e);  \
    } while (0)
#define CBCT_TRY(expr)                 \
    do {                               \
        int _s = (expr);               \
        if (_s != CBCT_OK) return _s;  \
    } while (0)
void count_launch();                        // one of OUR kernels was launched (cbct_launch_count)
#define CBCT_LAUNCH_CHECK()                   \
    do {                                      \
        ::cbct::count_launch();               \
        CBCT_CUDA_TRY(cudaGetLastError());    \
    } while (0)

// optional in-library kernel timer: CUDA events recorded on the launching stream around P / P^T
enum { PROF_FORWARD = 0, PROF_BACK = 1, PROF_KINDS = 2 };
struct ProfScope {
    int slot;
    cudaStream_t st;
    ProfScope(int kind, cudaStream_t s);
    ~ProfScope();
};

static inline cudaStream_t as_stream(void *s) { return reinterpret_cast<cudaStream_t>(s); }
static inline int cdiv(long long a, long long b) { return (int)((a + b - 1) / b); }

// ---- device-side geometry (POD, passed by value to kernels) ------------------------------------
// Index coordinates: X = x * inv_dx + cx  with cx = -ox/dx + (nx-1)/2.
// Sample grid: tau_k = t_k - SAD = tau0 + k*step, tau0 = t_min + step/2 - SAD; rays are re-anchored at
// t = SAD (near the isocentre) so that fp32 positions stay accurate.
struct DevGeom {
    int nx, ny, nz, nu, nv, n_views, K;
    double sad, sdd, du, dv, u_first, v_first;   // u = u_first + iu*du
    double inv_dx, inv_dy, inv_dz, cx, cy, cz;
    double tau0, step;
    const double2 *view_cs;                      // device: (cos th, sin th) per view
    // device: a permutation of the views, those whose fast shared-memory axis is x first, then the y-fast ones (stable).
    // The TMA kernels take their view from it (blockIdx.z is a POSITION in this order), so that each of the two
    // orientation-specific copies of the volume / accumulator volumes is used in one contiguous phase of the launch and
    // stays L2-resident during it (two 73 / 113 MB copies do not fit the 126 MB L2 together, one does).
    const int *view_order;
};

// device error word of a geometry handle (see cbct_geometry_status in include/cbct.h): `dev` lives in device memory
// (kernels OR their code into it and poll it at CTA start), `host` is the device alias of a mapped pinned host int that
// the entry points read without synchronising.
struct DevErr { int *dev; int *host; };
enum { DEV_ERR_WAIT_TIMEOUT = CBCT_STATUS_WAIT_TIMEOUT, DEV_ERR_FW_RANGE = CBCT_STATUS_FORWARD_RANGE,
       DEV_ERR_BT_RANGE = CBCT_STATUS_BACKPROJECT_RANGE, DEV_ERR_FIXED_POINT = CBCT_STATUS_FIXED_POINT_RANGE };

struct RayF {                                    // one ray in index space, fp32: P(tau) = c + b*tau
    float cx, cy, cz, bx, by, bz;
};

// fp64 ray set-up, identical for P and P^T so both sample the same points.
__device__ __forceinline__ void ray_setup(const DevGeom &g, int view, int iv, int iu, RayF &r,
                                          double &bxd, double &byd, double &bzd, double &cxd, double &cyd,
                                          double &czd) {
    const double2 cs = g.view_cs[view];
    const double u = g.u_first + iu * g.du, v = g.v_first + iv * g.dv;
    const double ex = -g.sdd * cs.x - u * cs.y, ey = -g.sdd * cs.y + u * cs.x, ez = v;
    const double invL = rsqrt(ex * ex + ey * ey + ez * ez);
    const double nx_ = ex * invL, ny_ = ey * invL, nz_ = ez * invL;
    // point at t = SAD
    const double px = g.sad * cs.x + nx_ * g.sad, py = g.sad * cs.y + ny_ * g.sad, pz = nz_ * g.sad;
    cxd = px * g.inv_dx + g.cx; cyd = py * g.inv_dy + g.cy; czd = pz * g.inv_dz + g.cz;
    bxd = nx_ * g.inv_dx; byd = ny_ * g.inv_dy; bzd = nz_ * g.inv_dz;
    r.cx = (float)cxd; r.cy = (float)cyd; r.cz = (float)czd;
    r.bx = (float)bxd; r.by = (float)byd; r.bz = (float)bzd;
}

// ---- deterministic two-level fp64 reduction (256-thread blocks) ---------------------------------------------------------
// Every thread brings its partial sum `acc`; the block's total goes to partials[blockIdx.x]; the block that finishes last
// adds up all block totals and thread 0 of that block gets the result (return value true, `total` set, counter reset).
// The order of every addition is fixed by (gridDim, blockDim) alone, so the result is reproducible; the last step is
// done by the whole block (thread t takes partials t, t + 256, ..., then the same warp / block tree), not by one thread
// walking gridDim.x dependent loads from L2 -- with 1184 blocks that walk was most of the kernel's time in round 1.
// `sh` = 8 doubles and `last` = one bool of shared memory, both declared by the calling kernel.
__device__ __forceinline__ bool ordered_total_at(double acc, double *partials, unsigned int *counter, double *sh, bool *last, double &total,
                                                 unsigned tid, unsigned n_threads, unsigned bid, unsigned n_blocks) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((tid & 31) == 0) sh[tid >> 5] = acc;
    __syncthreads();
    if (tid == 0) {
        double s = 0.0;
        for (int w = 0; w < 8; ++w) s += sh[w];
        partials[bid] = s;
        __threadfence();
        *last = (atomicAdd(counter, 1u) == n_blocks - 1);
    }
    __syncthreads();
    if (!*last) return false;                                    // block-uniform
    __threadfence();
    double s = 0.0;
    for (unsigned b = tid; b < n_blocks; b += n_threads) s += ((volatile double *)partials)[b];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((tid & 31) == 0) sh[tid >> 5] = s;                        // thread 0 read sh before the barrier above: no hazard
    __syncthreads();
    if (tid != 0) return false;
    total = 0.0;
    for (int w = 0; w < 8; ++w) total += sh[w];
    *counter = 0u;
    return true;
}
__device__ __forceinline__ bool ordered_total(double acc, double *partials, unsigned int *counter, double *sh, bool *last, double &total) {
    return ordered_total_at(acc, partials, counter, sh, last, total, threadIdx.x, blockDim.x, blockIdx.x, gridDim.x);
}
// where a kernel leaves the squared norm of its OUTPUT (SURVEY.md §8(d) "fused minimum": ||q||^2 in the epilogue of P, ||s||^2
// in the conversion pass of P^T); out == nullptr: not wanted
struct NormOut { double *out; double *partials; unsigned int *counter; };

// ---- P^T (cell-driven) tables, built in fp64 at geometry create, stored fp32 ------------------------
// With r = t / L(u,v) (t = distance from the source) a ray is  X = Kx + Ax r,  Y = Ky + Ay r,  Z = Kz + vz r,
// so clipping against a cell is done in r and only then scaled by L.  Sample positions use the
// re-anchored form  X = cX + bX * tau  (tau = t - SAD) with cX built from cancellation-free terms.
struct BpView {                 // per view
    float Kx, Ky;               // source position in index coordinates
    float Fx, Fy;               // SAD cos/dx, SAD sin/dy
    float D0, Dx, Dy;           // depth  D   = SAD - (x cos + y sin) as an affine function of cell indices (mm)
    float T0, Tx, Ty;           // lateral tau = -x sin + y cos, same (mm)
    float hl, hd;               // half lateral / half depth extent of one cell (mm)
};
struct BpViewU {                // per (view, iu)
    float Ax, Ay;               // (-SDD cos - u sin)/dx, (-SDD sin + u cos)/dy
    float Wx, Wy;               // 1/Ax, 1/Ay (denominators nudged away from 0; used for clipping only)
    float Gx, Gy;               // -SAD u sin/dx, SAD u cos/dy
    float pad0, pad1;
};
struct BpTables {
    const BpView *views;        // [n_views]
    const BpViewU *viewu;       // [n_views][nu]
    const float4 *pixT;         // [nu][nv] (v fastest): {1/L, q = 1 - SDD/L, L, 0},  L = sqrt(SDD^2 + u^2 + v^2)
    const float2 *rows;         // [nv]: {vz = v/dz, 1/vz (nudged)}
    float Kz, cx0, cy0, cz0;    // Kz = cz0: index coordinate of the plane z = 0
    float sdd, sad, u_first, inv_du, dz_dv, vfirst_dv, t0, inv_step, stepf, tau0f, k_eps;
};

}  // namespace cbct

// ---- opaque handles --------------------------------------------------------------------------------
struct cbct_geometry {
    cbct_geometry_desc desc;            // desc.angles points into `angles`
    std::vector<double> angles;
    double R, t_min, step;
    int32_t K;
    int64_t n_vox, n_rays, n_samples;
    cbct::DevGeom dg;
    double2 *d_view_cs;
    int *d_view_order;
    float *d_ws_vol, *d_ws_proj;        // staging for the *_host entry points (allocated at create)
    float *d_bp_partial;                // P^T workspace: 8 per-corner partial volumes over the (n+1)^3 cells
    float *d_bp_projT;                  // P^T workspace: projections transposed to [view][iu][iv]
    cbct::BpTables bp;                  // P^T lookup tables (device pointers + constants)
    // Which kernels run for this handle: decided ONCE, in cbct_geometry_create (plan + the CBCT_* selection variables read
    // there, include/cbct.h), reported by cbct_geometry_describe; launches never re-route and never read the environment.
    int fw_impl;                            // FW_TMA / FW_TILED / FW_GLOBAL
    int fw_packed;                          // forward_tma_kernel: packed-pair (1) or scalar (0) instruction stream
    int bp_impl;                            // BP_SCATTER / BP_CELL / BP_GATHER
    int bt_packed;                          // backproject_scatter_kernel: packed-pair (1) or scalar (0) stream
    // device error word (cbct_geometry_status): device int + mapped pinned host int
    cbct::DevErr err;
    int *h_err;                             // host address of the mapped word
    // forward TMA path (forward_tma.cu): box plan, y-fastest volume copy and its tensor map
    int fw_tma_ok, fw_b, fw_bs, fw_bz;      // box: fw_b columns (= row pitch) x fw_bs rows x fw_bz planes
    float fw_margin;
    float *d_fw_volT;
    double *d_fw_norm_partials;             // ||q||^2 block partials of forward_tma_kernel (one per CTA) + its counter
    unsigned int *d_fw_norm_counter;
    alignas(64) unsigned char fw_map_y[128];
    // P^T scatter path (backproject_tma.cu): int32 accumulator volumes (x-fastest, then y-fastest), max|g|, fixed-point plan
    int bt_b, bt_bs, bt_bz;                 // accumulator box (row pitch bt_b, bt_bs rows, bt_bz planes)
    int bt_lm;                              // lane layout of the scatter kernel (template parameter LM)
    int bt_ok, bt_qb, bt_group;             // 2^bt_qb = fixed-point unit per max|g|; views per accumulation group
    int *d_bt_acc;
    size_t bt_acc_y_off, bt_acc_elems;      // element offset of the y-fastest accumulator, total elements
    unsigned *d_bt_absmax;                  // [0] bits of max|g|, [1] bits of the fixed-point reference T = min(max|g|, 8 rms(g))
    double *d_bt_sumsq, *d_bt_partials;     // ||g||^2 (deterministic two-level reduction) and its scratch
    unsigned *d_bt_counter;
    double *d_bt_norm_partials;             // ||s||^2 block partials of the conversion pass (one per block) + its counter
    unsigned int *d_bt_norm_counter;
    alignas(64) unsigned char bt_map_x[128];
    alignas(64) unsigned char bt_map_y[128];
    // Siddon pair (siddon.cu), allocated by cbct_siddon_prepare: y-fastest volume copy, two int32 accumulator volumes, max|g|
    float *d_sd_volT;
    int *d_sd_acc;
    unsigned *d_sd_absmax;
    int sd_qb, sd_group;
    size_t workspace_bytes;
};

struct cbct_cgls {
    const cbct_geometry *geom;
    float *d_q, *d_s;
    double *d_scal;                     // {gamma, qq, alpha, beta, rr, gamma_new}
    int *d_flag;                        // breakdown flag
    double *d_partials;                 // reduction scratch
    unsigned int *d_counter;
};

namespace cbct {
enum { FW_TMA = 0, FW_TILED = 1, FW_GLOBAL = 2 };
enum { BP_SCATTER = 0, BP_CELL = 1, BP_GATHER = 2 };
bool forward_tiled_fits(const cbct_geometry *G, float *margin_out);
void describe_forward_tma(const cbct_geometry *G, char *buf, size_t cap);
void describe_backproject_tma(const cbct_geometry *G, char *buf, size_t cap);
// CBCT_E_DEVICE if a kernel of this handle has raised the device error word (read from the mapped host word: no sync)
static inline int device_error_pending(const cbct_geometry *G) {
    return (G->h_err && *reinterpret_cast<volatile int *>(G->h_err)) ? CBCT_E_DEVICE : CBCT_OK;
}
// kernels' host launchers used across translation units
// d_norm != nullptr: the caller wants ||output||^2 (fp64, device) from the same launch; *fused says whether the kernel that
// served the handle delivered it (the TMA kernels do: SURVEY.md §8(d) "fused minimum"), else the caller reduces the output itself
int launch_forward(const cbct_geometry *g, const float *d_vol, float *d_proj, cudaStream_t st, double *d_norm = nullptr, bool *fused = nullptr);
int launch_backproject(const cbct_geometry *g, const float *d_proj, float *d_vol, cudaStream_t st, double *d_norm = nullptr, bool *fused = nullptr);
void plan_forward_tma(cbct_geometry *g);     // decides whether/how the TMA forward kernel runs for this geometry
int launch_forward_tma(const cbct_geometry *g, const float *d_vol, float *d_proj, cudaStream_t st, double *d_norm = nullptr);
void plan_backproject_tma(cbct_geometry *g); // after plan_forward_tma: same boxes, int32 accumulators
void free_backproject_tma(cbct_geometry *g);
bool bt_fixed_point_plan(const cbct_geometry_desc &d, double R, double step, int *qb, int *views_per_group, double *w_view);
int launch_backproject_tma(const cbct_geometry *g, const float *d_proj, float *d_vol, cudaStream_t st, double *d_norm = nullptr);
void free_siddon(cbct_geometry *g);
bool siddon_fixed_point_plan(const cbct_geometry_desc &d, double R, int *qb, int *views_per_group, double *w_view);
// kernels launched from more than one translation unit
__global__ void transpose_vol_kernel(const float *__restrict__ v, float *__restrict__ vT, int nx, int ny);      // forward_tma.cu
__global__ void absmax_kernel(const float *__restrict__ g, long long n, unsigned *out);                        // backproject_tma.cu
__global__ void backproject_finalize_kernel(const int *__restrict__ acc_x, const int *__restrict__ acc_y, float *__restrict__ vol,
                                            int nx, int ny, int pf, int ps, int pz, const unsigned *__restrict__ absmax_bits,
                                            float step_over_two_qb, int accumulate, long long sat_limit, DevErr err, NormOut norm);  // backproject_tma.cu
int build_bp_tables(cbct_geometry *g);      // allocates + fills g->bp and g->d_bp_partial
void free_bp_tables(cbct_geometry *g);
int launch_sumsq(const float *d_v, int64_t n, double *d_out, double *d_partials, unsigned int *d_counter,
                 cudaStream_t st);
constexpr int kReduceBlocks = 1184;     // 148 SMs x 8
void tf_fused_prepare();                // decides (once per process) which kernel serves tf_apply_fused; may synchronise the device
}  // namespace cbct
