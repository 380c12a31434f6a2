// driver.cu -- Algorithm A2 inside the coarse-to-fine multigrid cascade
// (PAPER.md:232): cbct_recon_* and the one-shot cbct_tf_reconstruct*.  The host only sequences
// launches: the t-sequence of A2 step 5 is data independent, so nothing is read back and the whole
// reconstruction is one asynchronous stream of kernels.
#include <cmath>
#include <new>

#include "common.cuh"

struct cbct_recon_level {
    cbct_geometry *geom;
    cbct_cgls *cg;
    float *d_x, *d_p, *d_fa, *d_fb, *d_fc;   // volume-sized: CGLS x, p; A2 f^(k), f^(k-1), scratch
    float *d_gbin;                            // this level's binned projections (CBCT_RECON_BIN_DETECTOR, coarse levels), else null
    void *d_tv_work;                          // scratch of tv_rof (CBCT_RECON_TV), else null
    int nx, ny, nz, nu, nv;
};

struct cbct_recon {
    int n_levels;
    std::vector<cbct_recon_level> lev;       // coarse -> fine
    float *d_r;                               // projection-sized CGLS residual (g is full size on every level)
    float *d_g, *d_f;                         // staging for the host entry point
    int64_t n_rays, n_vox_finest;
};

using namespace cbct;

extern "C" int cbct_recon_destroy(cbct_recon *R) {
    if (!R) return CBCT_OK;
    for (auto &L : R->lev) {
        cbct_cgls_destroy(L.cg);
        cbct_geometry_destroy(L.geom);
        cudaFree(L.d_x); cudaFree(L.d_p); cudaFree(L.d_fa); cudaFree(L.d_fb); cudaFree(L.d_fc); cudaFree(L.d_gbin); cudaFree(L.d_tv_work);
    }
    cudaFree(R->d_r); cudaFree(R->d_g); cudaFree(R->d_f);
    (void)cudaGetLastError();
    delete R;
    return CBCT_OK;
}

extern "C" int cbct_recon_create(const cbct_geometry_desc *finest, int n_levels, cbct_recon **out) {
    return cbct_recon_create_ex(finest, n_levels, 0u, out);
}

extern "C" int cbct_recon_create_ex(const cbct_geometry_desc *finest, int n_levels, unsigned flags, cbct_recon **out) {
    if (!finest || !out || n_levels < 1 || n_levels > 8 || (flags & ~(unsigned)(CBCT_RECON_BIN_DETECTOR | CBCT_RECON_TV))) return CBCT_E_INVALID;
    *out = nullptr;
    const int fac0 = 1 << (n_levels - 1);
    if (finest->nx % fac0 || finest->ny % fac0) return CBCT_E_INVALID;   // x,y coarsened by 2 per level, z kept
    const bool bin = (flags & CBCT_RECON_BIN_DETECTOR) != 0;
    if (bin && (finest->nu % fac0 || finest->nv % fac0)) return CBCT_E_INVALID;
    cbct_recon *R = new (std::nothrow) cbct_recon();
    if (!R) return CBCT_E_INVALID;
    R->n_levels = n_levels;
    R->d_r = R->d_g = R->d_f = nullptr;
    R->n_rays = (int64_t)finest->nu * finest->nv * finest->n_views;
    R->n_vox_finest = (int64_t)finest->nx * finest->ny * finest->nz;
    int status = CBCT_OK;
    for (int l = 0; l < n_levels && status == CBCT_OK; ++l) {
        const int fac = 1 << (n_levels - 1 - l);
        cbct_geometry_desc d = *finest;
        d.nx = finest->nx / fac; d.ny = finest->ny / fac;
        d.dx = finest->dx * fac; d.dy = finest->dy * fac;             // same extent, coarser pitch
        if (bin) {                                                    // NEXT-4: same detector extent and centre, coarser pixels
            d.nu = finest->nu / fac; d.nv = finest->nv / fac;
            d.du = finest->du * fac; d.dv = finest->dv * fac;
        }
        cbct_recon_level L{};
        L.nx = d.nx; L.ny = d.ny; L.nz = d.nz; L.nu = d.nu; L.nv = d.nv;
        if (bin && fac > 1) {
            cudaError_t e = cudaMalloc(&L.d_gbin, sizeof(float) * (size_t)d.nu * d.nv * d.n_views);
            if (e != cudaSuccess) status = set_cuda_error(e);
        }
        if ((flags & CBCT_RECON_TV) && status == CBCT_OK) {
            cudaError_t e = cudaMalloc(&L.d_tv_work, tv_rof_workspace_bytes(d.nx, d.ny, d.nz));
            if (e != cudaSuccess) status = set_cuda_error(e);
        }
        status = cbct_geometry_create(&d, &L.geom);
        if (status == CBCT_OK) status = cbct_cgls_create(L.geom, &L.cg);
        const size_t bytes = sizeof(float) * (size_t)d.nx * d.ny * d.nz;
        float **bufs[5] = {&L.d_x, &L.d_p, &L.d_fa, &L.d_fb, &L.d_fc};
        for (auto b : bufs)
            if (status == CBCT_OK) {
                cudaError_t e = cudaMalloc(b, bytes);
                if (e != cudaSuccess) status = set_cuda_error(e);
            }
        R->lev.push_back(L);
    }
    float **pb[3] = {&R->d_r, &R->d_g, &R->d_f};
    const size_t pbytes[3] = {sizeof(float) * (size_t)R->n_rays, sizeof(float) * (size_t)R->n_rays,
                              sizeof(float) * (size_t)R->n_vox_finest};
    for (int i = 0; i < 3 && status == CBCT_OK; ++i) {
        cudaError_t e = cudaMalloc(pb[i], pbytes[i]);
        if (e != cudaSuccess) status = set_cuda_error(e);
    }
    if (status != CBCT_OK) { cbct_recon_destroy(R); return status; }
    tf_fused_prepare();                                  // the one-off self-check of the fused tight-frame kernel happens here, not in a hot call
    *out = R;
    return CBCT_OK;
}

// the regulariser of A2 steps 3-4: the tight frame or the TV comparison
struct Regulariser { bool tv; float mu, eps, rel_tol; int max_iter; };
static int run_cascade(cbct_recon *R, const float *d_g, float *d_f, const int *n_outer, int n_cgls, const Regulariser &reg,
                       int momentum, void *stream);

extern "C" int cbct_recon_run(cbct_recon *R, const float *d_g, float *d_f, const int *n_outer, int n_cgls, float mu,
                              int momentum, void *stream) {
    if (!R || !d_g || !d_f || !n_outer || n_cgls < 0 || !(mu >= 0.f)) return CBCT_E_INVALID;
    return run_cascade(R, d_g, d_f, n_outer, n_cgls, Regulariser{false, mu, 0.f, 0.f, 0}, momentum, stream);
}

extern "C" int cbct_recon_run_tv(cbct_recon *R, const float *d_g, float *d_f, const int *n_outer, int n_cgls, float mu_tv, float eps,
                                 int max_rof_iter, float rel_tol, int momentum, void *stream) {
    if (!R || !d_g || !d_f || !n_outer || n_cgls < 0 || !(mu_tv >= 0.f) || !(eps > 0.f) || max_rof_iter < 0 || !(rel_tol >= 0.f))
        return CBCT_E_INVALID;
    for (auto &L : R->lev)
        if (!L.d_tv_work) return CBCT_E_INVALID;          // created without CBCT_RECON_TV
    return run_cascade(R, d_g, d_f, n_outer, n_cgls, Regulariser{true, mu_tv, eps, rel_tol, max_rof_iter}, momentum, stream);
}

static int run_cascade(cbct_recon *R, const float *d_g, float *d_f, const int *n_outer, int n_cgls, const Regulariser &reg,
                       int momentum, void *stream) {
    cudaStream_t st = as_stream(stream);
    // detector binning: level l's data = block means of level l+1's (finest = d_g), i.e. mg_restrict on [view][v][u]
    for (int l = R->n_levels - 2; l >= 0; --l) {
        cbct_recon_level &L = R->lev[l], &F = R->lev[l + 1];
        if (!L.d_gbin) continue;
        const int n_views = (int)(R->n_rays / ((int64_t)R->lev.back().nu * R->lev.back().nv));
        CBCT_TRY(mg_restrict(F.d_gbin ? F.d_gbin : d_g, L.d_gbin, F.nu, F.nv, n_views, 2, 2, 1, stream));
    }
    for (int l = 0; l < R->n_levels; ++l) {
        cbct_recon_level &L = R->lev[l];
        const float *g_l = L.d_gbin ? L.d_gbin : d_g;
        const int64_t n = (int64_t)L.nx * L.ny * L.nz;
        float *f_cur = L.d_fa, *f_prev = L.d_fb, *f_new = L.d_fc;
        if (l == 0) {
            CBCT_CUDA_TRY(cudaMemsetAsync(f_cur, 0, sizeof(float) * n, st));          // f^(0) = 0
        } else {
            cbct_recon_level &C = R->lev[l - 1];                                         // "smoothly extend"
            CBCT_TRY(mg_prolong(C.d_fa, f_cur, L.nx, L.ny, L.nz, 2, 2, 1, stream));
        }
        CBCT_CUDA_TRY(cudaMemcpyAsync(f_prev, f_cur, sizeof(float) * n, cudaMemcpyDeviceToDevice, st));  // f^(-1) = f^(0)
        double t_prev = 1.0, t_cur = 1.0;                                                // t^(-1) = t^(0) = 1
        for (int k = 0; k < n_outer[l]; ++k) {
            const float coef = momentum ? (float)((t_prev - 1.0) / t_cur) : 0.f;
            CBCT_TRY(cbct_a2_extrapolate(f_cur, f_prev, L.d_x, coef, n, stream));        // 1. v
            CBCT_TRY(cbct_cgls_init(L.cg, g_l, L.d_x, R->d_r, L.d_p, stream));           // 2. f = CGLS[v]
            for (int m = 0; m < n_cgls; ++m) CBCT_TRY(cbct_cgls_step(L.cg, L.d_x, R->d_r, L.d_p, stream));
            if (!reg.tv) CBCT_TRY(tf_apply_fused(L.d_x, f_new, reg.mu, 1, L.nx, L.ny, L.nz, stream));   // 3.+4. shrink, clamp
            else CBCT_TRY(tv_rof(L.d_x, f_new, L.d_tv_work, reg.mu, reg.eps, reg.max_iter, reg.rel_tol, 1, L.nx, L.ny, L.nz, stream));
            float *tmp = f_prev; f_prev = f_cur; f_cur = f_new; f_new = tmp;
            const double t_next = 0.5 * (1.0 + std::sqrt(1.0 + 4.0 * t_cur * t_cur));    // 5.
            t_prev = t_cur; t_cur = t_next;
        }
        if (f_cur != L.d_fa)   // keep the level's result in d_fa for the prolongation / output
            CBCT_CUDA_TRY(cudaMemcpyAsync(L.d_fa, f_cur, sizeof(float) * n, cudaMemcpyDeviceToDevice, st));
    }
    CBCT_CUDA_TRY(cudaMemcpyAsync(d_f, R->lev.back().d_fa, sizeof(float) * R->n_vox_finest, cudaMemcpyDeviceToDevice, st));
    return CBCT_OK;
}

extern "C" int cbct_recon_run_host(cbct_recon *R, const float *h_g, float *h_f, const int *n_outer, int n_cgls, float mu,
                                   int momentum, void *stream) {
    if (!R || !h_g || !h_f) return CBCT_E_INVALID;
    cudaStream_t st = as_stream(stream);
    CBCT_CUDA_TRY(cudaMemcpyAsync(R->d_g, h_g, sizeof(float) * R->n_rays, cudaMemcpyHostToDevice, st));
    CBCT_TRY(cbct_recon_run(R, R->d_g, R->d_f, n_outer, n_cgls, mu, momentum, stream));
    CBCT_CUDA_TRY(cudaMemcpyAsync(h_f, R->d_f, sizeof(float) * R->n_vox_finest, cudaMemcpyDeviceToHost, st));
    CBCT_CUDA_TRY(cudaStreamSynchronize(st));
    return CBCT_OK;
}

extern "C" int cbct_recon_status(cbct_recon *R, void *stream, int *flags, int clear) {
    if (!R) return CBCT_E_INVALID;
    int all = 0, status = CBCT_OK;
    for (auto &L : R->lev) {
        int bits = 0;
        const int s = cbct_geometry_status(L.geom, stream, &bits, clear);
        if (s != CBCT_OK && s != CBCT_E_DEVICE) return s;
        if (s == CBCT_E_DEVICE) status = CBCT_E_DEVICE;
        all |= bits;
    }
    if (flags) *flags = all;
    return status;
}

extern "C" int cbct_recon_describe(const cbct_recon *R, char *buf, size_t cap) {
    if (!R || R->lev.empty()) return CBCT_E_INVALID;
    return cbct_geometry_describe(R->lev.back().geom, buf, cap);
}

extern "C" int cbct_tf_reconstruct(const cbct_geometry_desc *finest, const float *d_g, float *d_f, int n_levels,
                                   const int *n_outer, int n_cgls, float mu, int momentum, void *stream) {
    cbct_recon *R = nullptr;
    CBCT_TRY(cbct_recon_create(finest, n_levels, &R));
    int s = cbct_recon_run(R, d_g, d_f, n_outer, n_cgls, mu, momentum, stream);
    if (s == CBCT_OK) s = cbct_recon_status(R, stream, nullptr, 0);      // synchronises; CBCT_E_DEVICE if a kernel gave up
    cbct_recon_destroy(R);
    return s;
}

extern "C" int cbct_tf_reconstruct_host(const cbct_geometry_desc *finest, const float *h_g, float *h_f, int n_levels,
                                        const int *n_outer, int n_cgls, float mu, int momentum, void *stream) {
    cbct_recon *R = nullptr;
    CBCT_TRY(cbct_recon_create(finest, n_levels, &R));
    int s = cbct_recon_run_host(R, h_g, h_f, n_outer, n_cgls, mu, momentum, stream);
    if (s == CBCT_OK) s = cbct_recon_status(R, stream, nullptr, 0);
    cbct_recon_destroy(R);
    return s;
}
