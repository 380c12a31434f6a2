// cgls.cu -- CGLS (Appendix 1) around cbct_forward / cbct_backproject.
// The paper uses CUBLAS for the vector-vector operations; here they are fused
// kernels whose scalars (gamma, ||q||^2, alpha, beta) never leave the device, so a step is a fixed
// launch sequence with no host synchronisation.  Reductions accumulate in fp64 and are summed in a
// fixed order (deterministic).  ||q||^2 and ||s||^2 are delivered by the projector launches themselves where the
// TMA kernels serve the handle (epilogue of P, conversion pass of P^T: SURVEY.md §8(d) "fused minimum").
#include <new>

#include "common.cuh"

namespace cbct {

// float4 accesses only where every base pointer is 16-byte aligned (cbct.h asks for it; a misaligned vector access is
// an SM exception, so the kernels check and fall back to scalar accesses instead of trusting the caller)
__device__ __forceinline__ bool aligned16(const void *a, const void *b = nullptr) {
    return ((reinterpret_cast<uintptr_t>(a) | reinterpret_cast<uintptr_t>(b)) & 15) == 0;
}

enum { S_GAMMA = 0, S_QQ = 1, S_ALPHA = 2, S_BETA = 3, S_RR = 4, S_GAMMA_NEW = 5, S_COUNT = 8 };

// ||v||^2 -> *out.  Block partials in fp64, summed by the last block to finish in a fixed order (common.cuh: ordered_total).
__global__ void __launch_bounds__(256) sumsq_kernel(const float *__restrict__ v, long long n, double *out,
                                                    double *partials, unsigned int *counter) {
    double acc = 0.0;
    const long long n4 = aligned16(v) ? n >> 2 : 0;
    const float4 *v4 = reinterpret_cast<const float4 *>(v);
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n4; i += (long long)gridDim.x * blockDim.x) {
        const float4 a = __ldg(v4 + i);
        acc += (double)a.x * a.x + (double)a.y * a.y + (double)a.z * a.z + (double)a.w * a.w;
    }
    for (long long i = (n4 << 2) + blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n;
         i += (long long)gridDim.x * blockDim.x)
        acc += (double)v[i] * v[i];
    __shared__ double sh[8];
    __shared__ bool last;
    double total;
    if (ordered_total(acc, partials, counter, sh, &last, total)) *out = total;
}

int launch_sumsq(const float *d_v, int64_t n, double *d_out, double *d_partials, unsigned int *d_counter,
                 cudaStream_t st) {
    int blocks = (int)((n / 4 + 255) / 256);
    if (blocks > kReduceBlocks) blocks = kReduceBlocks;
    if (blocks < 1) blocks = 1;
    sumsq_kernel<<<blocks, 256, 0, st>>>(d_v, (long long)n, d_out, d_partials, d_counter);
    CBCT_LAUNCH_CHECK();
    return CBCT_OK;
}

// step 2: alpha = gamma / ||q||^2, or flag breakdown and make the updates no-ops
__global__ void cgls_alpha_kernel(double *s, int *flag) {
    if (s[S_GAMMA] == 0.0 || s[S_QQ] == 0.0 || *flag) { *flag = 1; s[S_ALPHA] = 0.0; }
    else s[S_ALPHA] = s[S_GAMMA] / s[S_QQ];
}
// steps 5-6: beta = gamma'/gamma; gamma <- gamma'
__global__ void cgls_beta_kernel(double *s, const int *flag) {
    if (*flag) { s[S_BETA] = 0.0; return; }
    s[S_BETA] = s[S_GAMMA_NEW] / s[S_GAMMA];
    s[S_GAMMA] = s[S_GAMMA_NEW];
}

// y[i] += sign * alpha * x[i]   (step 3; alpha read from the device)
__global__ void __launch_bounds__(256) axpy_dev_kernel(float *__restrict__ y, const float *__restrict__ x, long long n,
                                                       const double *s, float sign) {
    const float a = sign * (float)s[S_ALPHA];
    const long long n4 = aligned16(y, x) ? n >> 2 : 0;
    float4 *y4 = reinterpret_cast<float4 *>(y);
    const float4 *x4 = reinterpret_cast<const float4 *>(x);
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n4; i += (long long)gridDim.x * blockDim.x) {
        float4 yy = y4[i];
        const float4 xx = __ldg(x4 + i);
        yy.x = fmaf(a, xx.x, yy.x); yy.y = fmaf(a, xx.y, yy.y); yy.z = fmaf(a, xx.z, yy.z); yy.w = fmaf(a, xx.w, yy.w);
        y4[i] = yy;
    }
    for (long long i = (n4 << 2) + blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n;
         i += (long long)gridDim.x * blockDim.x)
        y[i] = fmaf(a, x[i], y[i]);
}

// p = s + beta p   (step 7); untouched on breakdown
__global__ void __launch_bounds__(256) p_update_kernel(float *__restrict__ p, const float *__restrict__ sv, long long n,
                                                       const double *s, const int *flag) {
    if (*flag) return;
    const float b = (float)s[S_BETA];
    const long long n4 = aligned16(p, sv) ? n >> 2 : 0;
    float4 *p4 = reinterpret_cast<float4 *>(p);
    const float4 *s4 = reinterpret_cast<const float4 *>(sv);
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n4; i += (long long)gridDim.x * blockDim.x) {
        float4 pp = p4[i];
        const float4 ss = __ldg(s4 + i);
        pp.x = fmaf(b, pp.x, ss.x); pp.y = fmaf(b, pp.y, ss.y); pp.z = fmaf(b, pp.z, ss.z); pp.w = fmaf(b, pp.w, ss.w);
        p4[i] = pp;
    }
    for (long long i = (n4 << 2) + blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n;
         i += (long long)gridDim.x * blockDim.x)
        p[i] = fmaf(b, p[i], sv[i]);
}

// r = g - q   (initialisation)
__global__ void __launch_bounds__(256) residual_kernel(float *__restrict__ r, const float *__restrict__ gq,
                                                       const float *__restrict__ q, long long n) {
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        r[i] = gq[i] - q[i];
}

__global__ void cgls_reset_kernel(double *s, int *flag) {
    for (int i = 0; i < S_COUNT; ++i) s[i] = 0.0;
    *flag = 0;
}
__global__ void cgls_set_gamma_kernel(double *s) { s[S_GAMMA] = s[S_GAMMA_NEW]; }

static inline int ew_blocks(long long n) {
    long long b = (n / 4 + 255) / 256;
    if (b > 148LL * 16) b = 148LL * 16;
    return (int)(b < 1 ? 1 : b);
}

}  // namespace cbct

using namespace cbct;

extern "C" int cbct_cgls_create(const cbct_geometry *G, cbct_cgls **out) {
    if (!G || !out) return CBCT_E_INVALID;
    *out = nullptr;
    cbct_cgls *cg = new (std::nothrow) cbct_cgls();
    if (!cg) return CBCT_E_INVALID;
    cg->geom = G;
    cg->d_q = cg->d_s = nullptr; cg->d_scal = nullptr; cg->d_flag = nullptr; cg->d_partials = nullptr; cg->d_counter = nullptr;
    cudaError_t e = cudaMalloc(&cg->d_q, sizeof(float) * G->n_rays);
    if (e == cudaSuccess) e = cudaMalloc(&cg->d_s, sizeof(float) * G->n_vox);
    if (e == cudaSuccess) e = cudaMalloc(&cg->d_scal, sizeof(double) * S_COUNT);
    if (e == cudaSuccess) e = cudaMalloc(&cg->d_flag, sizeof(int));
    if (e == cudaSuccess) e = cudaMalloc(&cg->d_partials, sizeof(double) * kReduceBlocks);
    if (e == cudaSuccess) e = cudaMalloc(&cg->d_counter, sizeof(unsigned int));
    if (e == cudaSuccess) e = cudaMemset(cg->d_counter, 0, sizeof(unsigned int));
    if (e == cudaSuccess) e = cudaMemset(cg->d_scal, 0, sizeof(double) * S_COUNT);
    if (e == cudaSuccess) e = cudaMemset(cg->d_flag, 0, sizeof(int));
    if (e != cudaSuccess) { cbct_cgls_destroy(cg); return set_cuda_error(e); }
    *out = cg;
    return CBCT_OK;
}

extern "C" int cbct_cgls_destroy(cbct_cgls *cg) {
    if (!cg) return CBCT_OK;
    cudaFree(cg->d_q); cudaFree(cg->d_s); cudaFree(cg->d_scal); cudaFree(cg->d_flag);
    cudaFree(cg->d_partials); cudaFree(cg->d_counter);
    (void)cudaGetLastError();
    delete cg;
    return CBCT_OK;
}

extern "C" int cbct_cgls_init(cbct_cgls *cg, const float *d_g, const float *d_x, float *d_r, float *d_p, void *stream) {
    if (!cg || !d_g || !d_x || !d_r || !d_p) return CBCT_E_INVALID;
    cudaStream_t st = as_stream(stream);
    const cbct_geometry *G = cg->geom;
    CBCT_TRY(device_error_pending(G));
    cgls_reset_kernel<<<1, 1, 0, st>>>(cg->d_scal, cg->d_flag);
    CBCT_LAUNCH_CHECK();
    CBCT_TRY(launch_forward(G, d_x, cg->d_q, st));                                   // q = P x0
    residual_kernel<<<ew_blocks(G->n_rays), 256, 0, st>>>(d_r, d_g, cg->d_q, G->n_rays);   // r = g - P x0
    CBCT_LAUNCH_CHECK();
    bool fused = false;
    CBCT_TRY(launch_backproject(G, d_r, d_p, st, cg->d_scal + S_GAMMA_NEW, &fused));  // p = s = P^T r, ||s||^2 from its conversion pass
    if (!fused) CBCT_TRY(launch_sumsq(d_p, G->n_vox, cg->d_scal + S_GAMMA_NEW, cg->d_partials, cg->d_counter, st));
    cgls_set_gamma_kernel<<<1, 1, 0, st>>>(cg->d_scal);                              // gamma = ||s||^2
    CBCT_LAUNCH_CHECK();
    return CBCT_OK;
}

extern "C" int cbct_cgls_step(cbct_cgls *cg, float *d_x, float *d_r, float *d_p, void *stream) {
    if (!cg || !d_x || !d_r || !d_p) return CBCT_E_INVALID;
    cudaStream_t st = as_stream(stream);
    const cbct_geometry *G = cg->geom;
    bool fused = false;
    CBCT_TRY(launch_forward(G, d_p, cg->d_q, st, cg->d_scal + S_QQ, &fused));                        // 1. q = P p, ||q||^2 from its epilogue
    if (!fused) CBCT_TRY(launch_sumsq(cg->d_q, G->n_rays, cg->d_scal + S_QQ, cg->d_partials, cg->d_counter, st));
    cgls_alpha_kernel<<<1, 1, 0, st>>>(cg->d_scal, cg->d_flag);                                      // 2. alpha
    CBCT_LAUNCH_CHECK();
    axpy_dev_kernel<<<ew_blocks(G->n_vox), 256, 0, st>>>(d_x, d_p, G->n_vox, cg->d_scal, 1.f);       // 3. x += alpha p
    CBCT_LAUNCH_CHECK();
    axpy_dev_kernel<<<ew_blocks(G->n_rays), 256, 0, st>>>(d_r, cg->d_q, G->n_rays, cg->d_scal, -1.f); //    r -= alpha q
    CBCT_LAUNCH_CHECK();
    CBCT_TRY(launch_backproject(G, d_r, cg->d_s, st, cg->d_scal + S_GAMMA_NEW, &fused));             // 4. s = P^T r, 5. ||s||^2
    if (!fused) CBCT_TRY(launch_sumsq(cg->d_s, G->n_vox, cg->d_scal + S_GAMMA_NEW, cg->d_partials, cg->d_counter, st));
    cgls_beta_kernel<<<1, 1, 0, st>>>(cg->d_scal, cg->d_flag);                                       // 6. beta
    CBCT_LAUNCH_CHECK();
    p_update_kernel<<<ew_blocks(G->n_vox), 256, 0, st>>>(d_p, cg->d_s, G->n_vox, cg->d_scal, cg->d_flag);    // 7.
    CBCT_LAUNCH_CHECK();
    return CBCT_OK;
}

extern "C" int cbct_cgls_scalars(cbct_cgls *cg, const float *d_r, double out[5], void *stream) {
    if (!cg || !out) return CBCT_E_INVALID;
    cudaStream_t st = as_stream(stream);
    if (d_r) CBCT_TRY(launch_sumsq(d_r, cg->geom->n_rays, cg->d_scal + S_RR, cg->d_partials, cg->d_counter, st));
    double h[S_COUNT];
    int flag = 0;
    CBCT_CUDA_TRY(cudaMemcpyAsync(h, cg->d_scal, sizeof(h), cudaMemcpyDeviceToHost, st));
    CBCT_CUDA_TRY(cudaMemcpyAsync(&flag, cg->d_flag, sizeof(int), cudaMemcpyDeviceToHost, st));
    CBCT_CUDA_TRY(cudaStreamSynchronize(st));
    out[0] = h[S_GAMMA]; out[1] = h[S_QQ]; out[2] = h[S_ALPHA]; out[3] = h[S_BETA]; out[4] = d_r ? h[S_RR] : -1.0;
    return flag ? CBCT_BREAKDOWN : CBCT_OK;
}
