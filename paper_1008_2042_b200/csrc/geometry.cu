// geometry.cu -- status plumbing, geometry handle, host-buffer entry points.
// cbct_geometry_create / _info: include/cbct.h; conventions of SURVEY.md §8(c) c.1-c.2.
#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>

#include "../../include/cbct_debug.h"
#include "common.cuh"

#ifdef CBCT_TEST_FAULTS
extern "C" int cbct_test_fault = 0;       // host-side test build only (tma_common.cuh)
#endif

namespace cbct {

static thread_local int g_last_cuda_error = 0;

int set_cuda_error(cudaError_t e) {
    g_last_cuda_error = (int)e;
    (void)cudaGetLastError();  // clear the sticky-free error state
    return CBCT_E_CUDA;
}

static std::atomic<long long> g_launches{0};
void count_launch() { g_launches.fetch_add(1, std::memory_order_relaxed); }

// ---- kernel timer ----------------------------------------------------------------------------
static std::mutex g_prof_mu;
static bool g_prof_on = false;
struct ProfRec { cudaEvent_t a, b; int kind; };
static std::vector<ProfRec> g_prof;

ProfScope::ProfScope(int kind, cudaStream_t s) : slot(-1), st(s) {
    if (!g_prof_on) return;
    std::lock_guard<std::mutex> lk(g_prof_mu);
    ProfRec r{};
    r.kind = kind;
    if (cudaEventCreate(&r.a) != cudaSuccess || cudaEventCreate(&r.b) != cudaSuccess) { (void)cudaGetLastError(); return; }
    cudaEventRecord(r.a, st);
    g_prof.push_back(r);
    slot = (int)g_prof.size() - 1;
}
ProfScope::~ProfScope() {
    if (slot < 0) return;
    std::lock_guard<std::mutex> lk(g_prof_mu);
    cudaEventRecord(g_prof[slot].b, st);
}

int device_supported() {
    int dev = 0, major = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { (void)cudaGetLastError(); return CBCT_E_UNSUPPORTED; }
    if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) {
        (void)cudaGetLastError();
        return CBCT_E_UNSUPPORTED;
    }
    return major == 10 ? CBCT_OK : CBCT_E_UNSUPPORTED;  // sm_100a code only: no other backend, no CPU path
}

// chord of every ray through the zero-padded box [-1, n]^3 (index space), in samples; block partials
__global__ void sample_count_kernel(DevGeom g, double *partials) {
    const long long n_rays = (long long)g.n_views * g.nv * g.nu;
    double acc = 0.0;
    for (long long r = blockIdx.x * (long long)blockDim.x + threadIdx.x; r < n_rays;
         r += (long long)gridDim.x * blockDim.x) {
        const int iu = (int)(r % g.nu), iv = (int)((r / g.nu) % g.nv), view = (int)(r / ((long long)g.nu * g.nv));
        RayF rf;
        double b[3], c[3];
        ray_setup(g, view, iv, iu, rf, b[0], b[1], b[2], c[0], c[1], c[2]);
        const double hi[3] = {(double)g.nx, (double)g.ny, (double)g.nz};
        double tin = -1e300, tout = 1e300;
        bool miss = false;
        for (int a = 0; a < 3; ++a) {
            if (b[a] == 0.0) { miss |= (c[a] < -1.0 || c[a] > hi[a]); continue; }
            double t1 = (-1.0 - c[a]) / b[a], t2 = (hi[a] - c[a]) / b[a];
            if (t1 > t2) { double t = t1; t1 = t2; t2 = t; }
            tin = fmax(tin, t1); tout = fmin(tout, t2);
        }
        if (!miss && tout > tin) acc += (tout - tin) / g.step;
    }
    __shared__ double sh[256];
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int s = blockDim.x / 2; s > 0; s >>= 1) {
        if ((int)threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x == 0) partials[blockIdx.x] = sh[0];
}

}  // namespace cbct

using namespace cbct;

extern "C" const char *cbct_status_string(int status) {
    switch (status) {
        case CBCT_OK: return "ok";
        case CBCT_E_INVALID: return "invalid argument";
        case CBCT_E_UNSUPPORTED: return "unsupported device (needs compute capability 10.x, sm_100a)";
        case CBCT_E_CUDA: return "CUDA runtime error (see cbct_last_cuda_error)";
        case CBCT_E_DEVICE: return "a kernel raised the device error word (see cbct_geometry_status)";
        case CBCT_BREAKDOWN: return "CGLS breakdown (gamma == 0 or ||q||^2 == 0)";
        default: return "unknown status";
    }
}

extern "C" int cbct_last_cuda_error(void) { return g_last_cuda_error; }
extern "C" int cbct_version(void) { return 100; }
extern "C" long long cbct_launch_count(void) { return g_launches.load(); }

extern "C" int cbct_profile_begin(void) {
    std::lock_guard<std::mutex> lk(g_prof_mu);
    for (auto &r : g_prof) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
    g_prof.clear();
    g_prof_on = true;
    return CBCT_OK;
}

extern "C" int cbct_profile_end(double ms[2], int count[2]) {
    std::lock_guard<std::mutex> lk(g_prof_mu);
    g_prof_on = false;
    int status = CBCT_OK;
    for (int k = 0; k < PROF_KINDS; ++k) { if (ms) ms[k] = 0.0; if (count) count[k] = 0; }
    for (auto &r : g_prof) {
        float t = 0.f;
        cudaError_t e = cudaEventSynchronize(r.b);
        if (e == cudaSuccess) e = cudaEventElapsedTime(&t, r.a, r.b);
        if (e != cudaSuccess) status = set_cuda_error(e);
        else { if (ms) ms[r.kind] += t; if (count) count[r.kind] += 1; }
        cudaEventDestroy(r.a); cudaEventDestroy(r.b);
    }
    g_prof.clear();
    return status;
}

// The selection variables of include/cbct.h, read once per cbct_geometry_create.  -1 = not forced.
// The instruction stream / lane layout of the TMA kernels, when not forced, is decided by fast_variants_ok() below.
struct Options { int fw_impl, bp_impl, fw_packed, bt_packed, bt_lanes; };
static Options read_options() {
    Options o{-1, -1, -1, -1, -1};
    if (const char *e = getenv("CBCT_FORWARD_IMPL")) {
        if (!strcmp(e, "tma")) o.fw_impl = FW_TMA; else if (!strcmp(e, "tiled")) o.fw_impl = FW_TILED; else if (!strcmp(e, "global")) o.fw_impl = FW_GLOBAL;
    }
    if (const char *e = getenv("CBCT_BACKPROJECT_IMPL")) {
        if (!strcmp(e, "scatter")) o.bp_impl = BP_SCATTER; else if (!strcmp(e, "cell")) o.bp_impl = BP_CELL; else if (!strcmp(e, "gather")) o.bp_impl = BP_GATHER;
    }
    if (const char *e = getenv("CBCT_FW_PACKED")) o.fw_packed = atoi(e) != 0;
    if (const char *e = getenv("CBCT_BT_PACKED")) o.bt_packed = atoi(e) != 0;
    if (const char *e = getenv("CBCT_BT_LANES")) o.bt_lanes = atoi(e) == 1 ? 1 : 0;
    return o;
}

static int validate(const cbct_geometry_desc *d, double *R_out, double *step_out) {
    if (!d || !d->angles) return CBCT_E_INVALID;
    if (d->nx <= 0 || d->ny <= 0 || d->nz <= 0 || d->nu <= 0 || d->nv <= 0 || d->n_views <= 0) return CBCT_E_INVALID;
    if (!(d->dx > 0) || !(d->dy > 0) || !(d->dz > 0) || !(d->du > 0) || !(d->dv > 0)) return CBCT_E_INVALID;
    if (!(d->sad > 0) || !(d->sdd > d->sad)) return CBCT_E_INVALID;
    if ((long long)d->nx * d->ny * d->nz > (1LL << 31) - 1) return CBCT_E_INVALID;
    if ((long long)d->nu * d->nv * d->n_views > (1LL << 31) - 1) return CBCT_E_INVALID;
    const double hx = 0.5 * (d->nx + 1) * d->dx, hy = 0.5 * (d->ny + 1) * d->dy, hz = 0.5 * (d->nz + 1) * d->dz;
    const double R = std::sqrt(hx * hx + hy * hy + hz * hz) + std::sqrt(d->ox * d->ox + d->oy * d->oy + d->oz * d->oz);
    if (!(R < d->sad)) return CBCT_E_INVALID;   // source would sit inside the padded volume
    double step = d->step_mm > 0 ? d->step_mm : 0.5 * std::fmin(d->dx, std::fmin(d->dy, d->dz));
    if (!(step > 0) || !std::isfinite(step)) return CBCT_E_INVALID;
    if (2.0 * R / step > 1e7) return CBCT_E_INVALID;   // K must stay exactly representable in fp32
    for (int i = 0; i < d->n_views; ++i)
        if (!std::isfinite(d->angles[i])) return CBCT_E_INVALID;
    *R_out = R;
    *step_out = step;
    return CBCT_OK;
}

static int create_with_options(const cbct_geometry_desc *desc, Options opt, cbct_geometry **out);

// ---- self-check of the fast TMA kernel variants (once per process, on the device in use) ------------------------------
// The packed-pair instruction streams (FFMA2 / FADD2 with per-instruction rounding modes) and the skewed 8x4 lane layout
// with same-cell merging are the fast variants of P and P^T; the scalar streams and the 16x2 layout are the plain ones.
// Both are the same arithmetic (P: bit-identical by construction; P^T: the same integer sums up to the rounding of the
// weight products).  Before a handle defaults to the fast variants, they are run once against the plain ones on a
// small built-in problem (64x64x16 volume, 8 views in all four quadrants, 96x32 detector): P must agree bit for bit,
// P^T to 2e-6 relative L2, and no device error word may be raised.  If not, every handle of this process uses the plain
// variants and cbct_geometry_describe says so.  (Forcing a variant with CBCT_FW_PACKED / CBCT_BT_PACKED / CBCT_BT_LANES
// bypasses the check: that is what the parity tests do to test each variant on its own.)
static int g_fast_state = -1;                          // -1 not run, 0 rejected, 1 accepted
static std::mutex g_fast_mu;
static bool run_fast_selfcheck() {
    const int nx = 64, ny = 64, nz = 16, nu = 96, nv = 32, nvw = 8;
    const double ang[nvw] = {0.1, 0.9, 1.7, 2.5, 3.3, 4.1, 4.9, 5.7};
    cbct_geometry_desc d{};
    d.nx = nx; d.ny = ny; d.nz = nz; d.dx = d.dy = d.dz = 4.0; d.ox = 3.0; d.oy = -2.0; d.oz = 1.0;
    d.nu = nu; d.nv = nv; d.du = d.dv = 3.2; d.u0 = 1.1; d.v0 = -0.7; d.sad = 1000.0; d.sdd = 1500.0;
    d.n_views = nvw; d.angles = ang; d.step_mm = 0.0;
    const size_t n_vox = (size_t)nx * ny * nz, n_rays = (size_t)nu * nv * nvw;
    std::vector<float> hv(n_vox), hp(n_rays), out[4];
    unsigned lcg = 12345u;
    auto rnd = [&]() { lcg = lcg * 1664525u + 1013904223u; return (float)(lcg >> 8) * (1.0f / 16777216.0f); };
    for (auto &v : hv) v = rnd();
    for (auto &v : hp) v = rnd() - 0.4f;
    float *d_v = nullptr, *d_p = nullptr, *d_o = nullptr;
    bool ok = cudaMalloc(&d_v, sizeof(float) * n_vox) == cudaSuccess && cudaMalloc(&d_p, sizeof(float) * n_rays) == cudaSuccess &&
              cudaMalloc(&d_o, sizeof(float) * std::max(n_vox, n_rays)) == cudaSuccess;
    ok = ok && cudaMemcpy(d_v, hv.data(), sizeof(float) * n_vox, cudaMemcpyHostToDevice) == cudaSuccess &&
         cudaMemcpy(d_p, hp.data(), sizeof(float) * n_rays, cudaMemcpyHostToDevice) == cudaSuccess;
    for (int fast = 0; fast < 2 && ok; ++fast) {
        cbct_geometry *G = nullptr;
        ok = create_with_options(&d, Options{FW_TMA, BP_SCATTER, fast, fast, fast ? 0 : 1}, &G) == CBCT_OK;
        if (!ok) break;
        out[2 * fast].resize(n_rays); out[2 * fast + 1].resize(n_vox);
        ok = launch_forward(G, d_v, d_o, nullptr) == CBCT_OK &&
             cudaMemcpy(out[2 * fast].data(), d_o, sizeof(float) * n_rays, cudaMemcpyDeviceToHost) == cudaSuccess &&
             launch_backproject(G, d_p, d_o, nullptr) == CBCT_OK &&
             cudaMemcpy(out[2 * fast + 1].data(), d_o, sizeof(float) * n_vox, cudaMemcpyDeviceToHost) == cudaSuccess;
        int bits = 0;
        ok = ok && cbct_geometry_status(G, nullptr, &bits, 0) == CBCT_OK;
        cbct_geometry_destroy(G);
    }
    cudaFree(d_v); cudaFree(d_p); cudaFree(d_o);
    (void)cudaGetLastError();
    if (!ok) return false;
    if (std::memcmp(out[0].data(), out[2].data(), sizeof(float) * n_rays) != 0) return false;     // P: bit for bit
    double num = 0, den = 0;
    for (size_t i = 0; i < n_vox; ++i) {
        const double a = out[1][i], b = out[3][i];
        num += (a - b) * (a - b); den += a * a;
    }
    return den > 0 && num <= 4e-12 * den;                                                       // P^T: 2e-6 relative L2
}
#ifdef CBCT_TEST_FAULTS
extern "C" void cbct_test_reset_selfcheck(void) { std::lock_guard<std::mutex> lk(g_fast_mu); g_fast_state = -1; }   // test build only
#endif
static bool fast_variants_ok() {
    std::lock_guard<std::mutex> lk(g_fast_mu);
    if (g_fast_state < 0) {
        g_fast_state = 0;                              // a nested create (the check's own handles) never re-enters
        g_fast_state = run_fast_selfcheck() ? 1 : 0;
    }
    return g_fast_state == 1;
}

extern "C" int cbct_geometry_create(const cbct_geometry_desc *desc, cbct_geometry **out) {
    if (!out) return CBCT_E_INVALID;
    *out = nullptr;
    double R = 0, step = 0;
    CBCT_TRY(validate(desc, &R, &step));
    CBCT_TRY(device_supported());
    Options opt = read_options();
    if (opt.fw_packed < 0 || opt.bt_packed < 0 || opt.bt_lanes < 0) {
        const bool fast = fast_variants_ok();
        if (opt.fw_packed < 0) opt.fw_packed = fast ? 1 : 0;
        if (opt.bt_packed < 0) opt.bt_packed = fast ? 1 : 0;
        if (opt.bt_lanes < 0) opt.bt_lanes = fast ? 0 : 1;
    }
    return create_with_options(desc, opt, out);
}

static int create_with_options(const cbct_geometry_desc *desc, Options opt, cbct_geometry **out) {
    *out = nullptr;
    double R = 0, step = 0;
    CBCT_TRY(validate(desc, &R, &step));
    cbct_geometry *G = new (std::nothrow) cbct_geometry();
    if (!G) return CBCT_E_INVALID;
    G->desc = *desc;
    G->angles.assign(desc->angles, desc->angles + desc->n_views);
    G->desc.angles = G->angles.data();
    G->desc.step_mm = step;
    G->R = R; G->step = step; G->t_min = desc->sad - R;
    G->K = (int32_t)std::ceil(2.0 * R / step);
    G->n_vox = (int64_t)desc->nx * desc->ny * desc->nz;
    G->n_rays = (int64_t)desc->nu * desc->nv * desc->n_views;
    G->d_view_order = nullptr;
    G->d_view_cs = nullptr; G->d_ws_vol = nullptr; G->d_ws_proj = nullptr; G->d_bp_partial = nullptr; G->d_bp_projT = nullptr; G->d_fw_volT = nullptr; G->d_fw_norm_partials = nullptr; G->d_fw_norm_counter = nullptr; G->fw_tma_ok = 0;
    G->err = DevErr{nullptr, nullptr}; G->h_err = nullptr;
    G->bt_ok = 0; G->d_bt_acc = nullptr; G->d_bt_absmax = nullptr;
    G->d_sd_volT = nullptr; G->d_sd_acc = nullptr; G->d_sd_absmax = nullptr; G->sd_qb = 0; G->sd_group = 0;
    G->bp = BpTables{};
    G->workspace_bytes = 0;

    std::vector<double2> cs(desc->n_views);
    for (int i = 0; i < desc->n_views; ++i) cs[i] = make_double2(std::cos(desc->angles[i]), std::sin(desc->angles[i]));
    std::vector<int> order;                                    // x-fast views, then y-fast views (same rule as the kernels)
    for (int pass = 0; pass < 2; ++pass)
        for (int i = 0; i < desc->n_views; ++i)
            if ((std::fabs(cs[i].x) > std::fabs(cs[i].y)) == (pass == 1)) order.push_back(i);
    cudaError_t e = cudaMalloc(&G->d_view_cs, sizeof(double2) * cs.size());
    if (e == cudaSuccess) e = cudaMemcpy(G->d_view_cs, cs.data(), sizeof(double2) * cs.size(), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMalloc(&G->d_view_order, sizeof(int) * order.size());
    if (e == cudaSuccess) e = cudaMemcpy(G->d_view_order, order.data(), sizeof(int) * order.size(), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMalloc(&G->d_ws_vol, sizeof(float) * G->n_vox);
    if (e == cudaSuccess) e = cudaMalloc(&G->d_ws_proj, sizeof(float) * G->n_rays);
    // device error word: a device int the kernels OR into, and a mapped pinned host int the entry points poll
    if (e == cudaSuccess) e = cudaMalloc(&G->err.dev, sizeof(int));
    if (e == cudaSuccess) e = cudaMemset(G->err.dev, 0, sizeof(int));
    if (e == cudaSuccess) e = cudaHostAlloc(reinterpret_cast<void **>(&G->h_err), sizeof(int), cudaHostAllocMapped);
    if (e == cudaSuccess) { *G->h_err = 0; e = cudaHostGetDevicePointer(reinterpret_cast<void **>(&G->err.host), G->h_err, 0); }
    if (e != cudaSuccess) { cbct_geometry_destroy(G); return set_cuda_error(e); }
    G->workspace_bytes = sizeof(double2) * cs.size() + sizeof(float) * (G->n_vox + G->n_rays);

    DevGeom &g = G->dg;
    g.nx = desc->nx; g.ny = desc->ny; g.nz = desc->nz; g.nu = desc->nu; g.nv = desc->nv;
    g.n_views = desc->n_views; g.K = G->K;
    g.sad = desc->sad; g.sdd = desc->sdd; g.du = desc->du; g.dv = desc->dv;
    g.u_first = desc->u0 - 0.5 * (desc->nu - 1) * desc->du;
    g.v_first = desc->v0 - 0.5 * (desc->nv - 1) * desc->dv;
    g.inv_dx = 1.0 / desc->dx; g.inv_dy = 1.0 / desc->dy; g.inv_dz = 1.0 / desc->dz;
    g.cx = -desc->ox / desc->dx + 0.5 * (desc->nx - 1);
    g.cy = -desc->oy / desc->dy + 0.5 * (desc->ny - 1);
    g.cz = -desc->oz / desc->dz + 0.5 * (desc->nz - 1);
    g.step = step;
    g.tau0 = G->t_min + 0.5 * step - desc->sad;
    g.view_cs = G->d_view_cs;
    g.view_order = G->d_view_order;

    // ---- which kernels serve this handle: plan + the selection variables, read HERE and nowhere else (cbct.h) ----
    G->fw_packed = opt.fw_packed; G->bt_packed = opt.bt_packed; G->bt_lm = opt.bt_lanes;
    plan_forward_tma(G);
    plan_backproject_tma(G);
    {
        float margin = 0.f;
        const bool tiled_ok = forward_tiled_fits(G, &margin);
        int want = opt.fw_impl;
        if (want < 0) want = G->fw_tma_ok ? FW_TMA : (tiled_ok ? FW_TILED : FW_GLOBAL);
        if ((want == FW_TMA && !G->fw_tma_ok) || (want == FW_TILED && !tiled_ok)) { cbct_geometry_destroy(G); return CBCT_E_UNSUPPORTED; }
        G->fw_impl = want;
        want = opt.bp_impl;
        if (want < 0) want = G->bt_ok ? BP_SCATTER : BP_CELL;
        if (want == BP_SCATTER && !G->bt_ok) { cbct_geometry_destroy(G); return CBCT_E_UNSUPPORTED; }
        if (want == BP_CELL && desc->nz + 1 > 512) {
            if (opt.bp_impl == BP_CELL) { cbct_geometry_destroy(G); return CBCT_E_UNSUPPORTED; }
            want = BP_GATHER;                             // volumes too tall for the cell kernel's z-lanes
        }
        G->bp_impl = want;
        if (G->bp_impl != BP_SCATTER) free_backproject_tma(G);       // accumulators of a path that will not run
        const int st_bp = build_bp_tables(G);
        if (st_bp != CBCT_OK) { cbct_geometry_destroy(G); return st_bp; }
    }

    // algorithmic sample count (unit of Gsamples/s), once, on the device
    const int blocks = 592;
    double *d_part = nullptr;
    e = cudaMalloc(&d_part, sizeof(double) * blocks);
    if (e != cudaSuccess) { cbct_geometry_destroy(G); return set_cuda_error(e); }
    sample_count_kernel<<<blocks, 256>>>(g, d_part);
    std::vector<double> part(blocks);
    e = cudaMemcpy(part.data(), d_part, sizeof(double) * blocks, cudaMemcpyDeviceToHost);
    cudaFree(d_part);
    if (e != cudaSuccess) { cbct_geometry_destroy(G); return set_cuda_error(e); }
    double total = 0;
    for (double p : part) total += p;
    G->n_samples = (int64_t)std::llround(total);
    *out = G;
    return CBCT_OK;
}

extern "C" int cbct_backproject_fixed_point_plan(const cbct_geometry_desc *desc, int32_t *qb, int32_t *views_per_group,
                                                double *max_weight_sum_per_view) {
    double R = 0, step = 0;
    CBCT_TRY(validate(desc, &R, &step));
    int q = 0, grp = 0;
    double w = 0;
    if (!bt_fixed_point_plan(*desc, R, step, &q, &grp, &w)) return CBCT_E_UNSUPPORTED;
    if (qb) *qb = q;
    if (views_per_group) *views_per_group = grp;
    if (max_weight_sum_per_view) *max_weight_sum_per_view = w;
    return CBCT_OK;
}

extern "C" int cbct_siddon_fixed_point_plan(const cbct_geometry_desc *desc, int32_t *qb, int32_t *views_per_group,
                                           double *max_path_sum_per_view) {
    double R = 0, step = 0;
    CBCT_TRY(validate(desc, &R, &step));
    int q = 0, grp = 0;
    double w = 0;
    if (!siddon_fixed_point_plan(*desc, R, &q, &grp, &w)) return CBCT_E_UNSUPPORTED;
    if (qb) *qb = q;
    if (views_per_group) *views_per_group = grp;
    if (max_path_sum_per_view) *max_path_sum_per_view = w;
    return CBCT_OK;
}

extern "C" int cbct_geometry_describe(const cbct_geometry *G, char *buf, size_t cap) {
    if (!G || !buf || !cap) return CBCT_E_INVALID;
    char fw[160], bp[200];
    if (G->fw_impl == FW_TMA) describe_forward_tma(G, fw, sizeof fw);
    else snprintf(fw, sizeof fw, "%s", G->fw_impl == FW_TILED ? "forward_tiled_kernel" : "forward_global_kernel");
    if (G->bp_impl == BP_SCATTER) describe_backproject_tma(G, bp, sizeof bp);
    else snprintf(bp, sizeof bp, "%s", G->bp_impl == BP_CELL ? "backproject_cell_kernel + backproject_combine_kernel" : "backproject_gather_kernel");
    snprintf(buf, cap, "forward: %s; backproject: %s%s", fw, bp,
             g_fast_state == 0 ? " (fast variants rejected by the create-time self-check)" : "");
    return CBCT_OK;
}

extern "C" int cbct_geometry_status(cbct_geometry *G, void *stream, int *flags, int clear) {
    if (!G) return CBCT_E_INVALID;
    CBCT_CUDA_TRY(cudaStreamSynchronize(as_stream(stream)));
    int bits = 0;
    CBCT_CUDA_TRY(cudaMemcpy(&bits, G->err.dev, sizeof(int), cudaMemcpyDeviceToHost));
    bits |= *reinterpret_cast<volatile int *>(G->h_err);
    if (flags) *flags = bits;
    if (clear && bits) {
        CBCT_CUDA_TRY(cudaMemset(G->err.dev, 0, sizeof(int)));
        *reinterpret_cast<volatile int *>(G->h_err) = 0;
    }
    return bits ? CBCT_E_DEVICE : CBCT_OK;
}

extern "C" int cbct_geometry_destroy(cbct_geometry *G) {
    if (!G) return CBCT_OK;
    cudaFree(G->err.dev);
    if (G->h_err) cudaFreeHost(G->h_err);
    cudaFree(G->d_view_cs);
    cudaFree(G->d_view_order);
    cudaFree(G->d_ws_vol);
    cudaFree(G->d_ws_proj);
    free_bp_tables(G);
    free_backproject_tma(G);
    cudaFree(G->d_fw_volT);
    cudaFree(G->d_fw_norm_partials);
    cudaFree(G->d_fw_norm_counter);
    free_siddon(G);
    (void)cudaGetLastError();
    delete G;
    return CBCT_OK;
}

extern "C" int cbct_geometry_info(const cbct_geometry *G, int64_t *n_vox, int64_t *n_rays, int32_t *K, double *t_min,
                                  double *step_mm, int64_t *n_samples_algorithmic, size_t *workspace_bytes) {
    if (!G) return CBCT_E_INVALID;
    if (n_vox) *n_vox = G->n_vox;
    if (n_rays) *n_rays = G->n_rays;
    if (K) *K = G->K;
    if (t_min) *t_min = G->t_min;
    if (step_mm) *step_mm = G->step;
    if (n_samples_algorithmic) *n_samples_algorithmic = G->n_samples;
    if (workspace_bytes) *workspace_bytes = G->workspace_bytes;
    return CBCT_OK;
}

extern "C" int cbct_forward(const cbct_geometry *G, const float *d_vol, float *d_proj, void *stream) {
    if (!G || !d_vol || !d_proj) return CBCT_E_INVALID;
    return launch_forward(G, d_vol, d_proj, as_stream(stream));
}

extern "C" int cbct_backproject(const cbct_geometry *G, const float *d_proj, float *d_vol, void *stream) {
    if (!G || !d_vol || !d_proj) return CBCT_E_INVALID;
    return launch_backproject(G, d_proj, d_vol, as_stream(stream));
}

extern "C" int cbct_forward_host(cbct_geometry *G, const float *h_vol, float *h_proj, void *stream) {
    if (!G || !h_vol || !h_proj) return CBCT_E_INVALID;
    cudaStream_t st = as_stream(stream);
    CBCT_CUDA_TRY(cudaMemcpyAsync(G->d_ws_vol, h_vol, sizeof(float) * G->n_vox, cudaMemcpyHostToDevice, st));
    CBCT_TRY(launch_forward(G, G->d_ws_vol, G->d_ws_proj, st));
    CBCT_CUDA_TRY(cudaMemcpyAsync(h_proj, G->d_ws_proj, sizeof(float) * G->n_rays, cudaMemcpyDeviceToHost, st));
    return CBCT_OK;
}

extern "C" int cbct_backproject_host(cbct_geometry *G, const float *h_proj, float *h_vol, void *stream) {
    if (!G || !h_vol || !h_proj) return CBCT_E_INVALID;
    cudaStream_t st = as_stream(stream);
    CBCT_CUDA_TRY(cudaMemcpyAsync(G->d_ws_proj, h_proj, sizeof(float) * G->n_rays, cudaMemcpyHostToDevice, st));
    CBCT_TRY(launch_backproject(G, G->d_ws_proj, G->d_ws_vol, st));
    CBCT_CUDA_TRY(cudaMemcpyAsync(h_vol, G->d_ws_vol, sizeof(float) * G->n_vox, cudaMemcpyDeviceToHost, st));
    return CBCT_OK;
}
