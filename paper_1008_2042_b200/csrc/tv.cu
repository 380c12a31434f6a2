// tv.cu -- the paper's COMPARISON regulariser: total variation through the Rudin-Osher-Fatemi
// sub-problem, PAPER.md:236-238 (§2.3): argmin_f ||f - u||^2 + mu_TV ||f||_TV "by a simple gradient descent method ... with
// an adaptively adjusted step length", stopped "when the energy function value decreases less than ... 0.1%".
// include/cbct.h: tv_rof, tv_rof_workspace_bytes, tv_rof_result.  Readings T1-T6 (the paper gives no
// discretisation): forward differences with zero rows at the last faces, isotropic TV smoothed by eps,
//   E(f) = sum (f-u)^2 + mu sum sqrt(|Df|^2 + eps^2),   grad E = 2 (f-u) + mu D^T( Df / sqrt(|Df|^2 + eps^2) ),
// a trial step f - tau grad E is accepted iff it lowers E (then tau *= 1.2, else tau /= 2), descent from f = u with
// tau = 0.25, stop at the first accepted step whose relative decrease is below rel_tol or after max_iter trials.
// The descent is data dependent, yet nothing is read back: the control state (E, tau, which of the two buffers holds the
// iterate, done) lives in device memory, the host issues max_iter x {trial, energy, decide} launches and every kernel
// returns at once when `done` is set, so the whole regulariser is one asynchronous stream of kernels like the rest of
// the path.  Energies are accumulated in fp64 in a fixed order (block partials summed by the last block), so the
// accept / reject decisions are reproducible and are taken in the precision the oracle takes them in.
#include <new>

#include "common.cuh"

namespace cbct {

struct TvState {
    double E, Et;          // energy of the iterate, of the trial
    float tau;
    int cur;               // buffer holding the iterate: 0 = the caller's d_f, 1 = the workspace volume
    int done, trials, accepted;
    unsigned counter;      // last-block detection of the energy reduction
};

__device__ __forceinline__ float tv_at(const float *__restrict__ f, int x, int y, int z, int nx, int ny) {
    return __ldg(f + ((size_t)z * ny + y) * nx + x);
}
// forward differences at (x,y,z), zero across the last faces (T1), and 1 / sqrt(|Df|^2 + eps^2)
__device__ __forceinline__ void tv_diffs(const float *__restrict__ f, int x, int y, int z, int nx, int ny, int nz, float eps2, float &gx,
                                         float &gy, float &gz, float &inv) {
    const float c = tv_at(f, x, y, z, nx, ny);
    gx = x + 1 < nx ? tv_at(f, x + 1, y, z, nx, ny) - c : 0.f;
    gy = y + 1 < ny ? tv_at(f, x, y + 1, z, nx, ny) - c : 0.f;
    gz = z + 1 < nz ? tv_at(f, x, y, z + 1, nx, ny) - c : 0.f;
    inv = 1.f / sqrtf(fmaf(gx, gx, fmaf(gy, gy, fmaf(gz, gz, eps2))));
}

__global__ void tv_init_kernel(TvState *s) {
    s->E = 0.0; s->Et = 0.0; s->tau = 0.25f; s->cur = 0; s->done = 0; s->trials = 0; s->accepted = 0; s->counter = 0u;
}

// which = 0: energy of the iterate -> s->E (the start of the descent);  which = 1: energy of the trial -> s->Et
__global__ void __launch_bounds__(256) tv_energy_kernel(const float *__restrict__ buf0, const float *__restrict__ buf1,
                                                        const float *__restrict__ u, TvState *s, int which, float mu, float eps2,
                                                        int nx, int ny, int nz, double *partials) {
    if (s->done) return;
    const float *f = ((s->cur ^ which) & 1) ? buf1 : buf0;
    double acc = 0.0;
    // linear block index -> (row tile, plane): 256 threads = 32 (x) x 8 (y), x strides over the row, blocks stride over (y-tile, z)
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5, ytiles = (ny + 7) >> 3;
    for (int job = blockIdx.x; job < ytiles * nz; job += gridDim.x) {
        const int z = job / ytiles, y = (job - z * ytiles) * 8 + ty;
        if (y >= ny) continue;
        const size_t row = ((size_t)z * ny + y) * nx;
        for (int x = tx; x < nx; x += 32) {
            float gx, gy, gz, inv;
            tv_diffs(f, x, y, z, nx, ny, nz, eps2, gx, gy, gz, inv);
            const float d = __ldg(f + row + x) - __ldg(u + row + x);
            acc += (double)d * d + (double)mu * (double)sqrtf(fmaf(gx, gx, fmaf(gy, gy, fmaf(gz, gz, eps2))));
        }
    }
    __shared__ double sh[8];
    __shared__ bool last;
    double t;
    if (ordered_total(acc, partials, &s->counter, sh, &last, t)) {
        if (which) s->Et = t; else { s->E = t; if (t == 0.0) s->done = 1; }       // E(u) = 0: nothing to do (T6)
    }
}

// trial = f - tau grad E(f),  f = the iterate's buffer, trial = the other one
__global__ void __launch_bounds__(256) tv_trial_kernel(float *__restrict__ buf0, float *__restrict__ buf1, const float *__restrict__ u,
                                                       const TvState *s, float mu, float eps2, int nx, int ny, int nz) {
    if (s->done) return;
    const float *f = s->cur ? buf1 : buf0;
    float *t = s->cur ? buf0 : buf1;
    const float tau = s->tau;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5, ytiles = (ny + 7) >> 3;
    for (int job = blockIdx.x; job < ytiles * nz; job += gridDim.x) {
        const int z = job / ytiles, y = (job - z * ytiles) * 8 + ty;
        if (y >= ny) continue;
        const size_t row = ((size_t)z * ny + y) * nx;
        for (int x = tx; x < nx; x += 32) {
            float gx, gy, gz, inv, a, b, c, ninv;
            tv_diffs(f, x, y, z, nx, ny, nz, eps2, gx, gy, gz, inv);
            // (D^T p)[i] = sum_a ( p_a[i - e_a] - p_a[i] ),  p = Df / sqrt(|Df|^2 + eps^2)
            float div = -(gx + gy + gz) * inv;
            if (x > 0) { tv_diffs(f, x - 1, y, z, nx, ny, nz, eps2, a, b, c, ninv); div = fmaf(a, ninv, div); }
            if (y > 0) { tv_diffs(f, x, y - 1, z, nx, ny, nz, eps2, a, b, c, ninv); div = fmaf(b, ninv, div); }
            if (z > 0) { tv_diffs(f, x, y, z - 1, nx, ny, nz, eps2, a, b, c, ninv); div = fmaf(c, ninv, div); }
            const float fi = __ldg(f + row + x);
            const float grad = fmaf(mu, div, 2.f * (fi - __ldg(u + row + x)));
            t[row + x] = fmaf(-tau, grad, fi);
        }
    }
}

// T5 / T6 on the device
__global__ void tv_decide_kernel(TvState *s, float rel_tol) {
    if (s->done) return;
    s->trials += 1;
    if (s->Et < s->E) {
        const double rel = (s->E - s->Et) / s->E;
        s->E = s->Et;
        s->cur ^= 1;
        s->accepted += 1;
        s->tau *= 1.2f;
        if (rel < (double)rel_tol) s->done = 1;
    } else {
        s->tau *= 0.5f;
    }
}

// the result -> d_f (= buf0), optionally clamped at zero (positivity H)
__global__ void __launch_bounds__(256) tv_finish_kernel(float *__restrict__ buf0, const float *__restrict__ buf1, const TvState *s,
                                                        int clamp, long long n) {
    const bool from1 = s->cur != 0;
    if (!from1 && !clamp) return;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        float v = from1 ? __ldg(buf1 + i) : buf0[i];
        if (clamp) v = fmaxf(v, 0.f);
        buf0[i] = v;
    }
}

static inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }
static inline int tv_blocks(long long n) {
    long long b = (n + 255) / 256;
    if (b > kReduceBlocks) b = kReduceBlocks;
    return (int)(b < 1 ? 1 : b);
}
// trial / energy kernels: one block job = 8 rows of one plane (32 x 8 threads, x strides over the row)
static inline int tv_jobs(int ny, int nz) {
    long long b = (long long)((ny + 7) >> 3) * nz;
    if (b > kReduceBlocks) b = kReduceBlocks;
    return (int)(b < 1 ? 1 : b);
}

}  // namespace cbct

using namespace cbct;

extern "C" size_t tv_rof_workspace_bytes(int nx, int ny, int nz) {
    if (nx <= 0 || ny <= 0 || nz <= 0) return 0;
    return align_up(sizeof(float) * (size_t)nx * ny * nz, 256) + 256 + sizeof(double) * kReduceBlocks;
}

extern "C" int tv_rof(const float *d_u, float *d_f, void *d_work, float mu_tv, float eps, int max_iter, float rel_tol,
                      int clamp_nonneg, int nx, int ny, int nz, void *stream) {
    if (!d_u || !d_f || !d_work || d_u == d_f || nx <= 0 || ny <= 0 || nz <= 0) return CBCT_E_INVALID;
    if (!(mu_tv >= 0.f) || !(eps > 0.f) || max_iter < 0 || !(rel_tol >= 0.f)) return CBCT_E_INVALID;
    if ((long long)nx * ny * nz > (1LL << 31) - 1) return CBCT_E_INVALID;
    CBCT_TRY(device_supported());
    cudaStream_t st = as_stream(stream);
    const long long n = (long long)nx * ny * nz;
    unsigned char *w = static_cast<unsigned char *>(d_work);
    float *buf1 = reinterpret_cast<float *>(w);
    TvState *s = reinterpret_cast<TvState *>(w + align_up(sizeof(float) * (size_t)n, 256));
    double *partials = reinterpret_cast<double *>(w + align_up(sizeof(float) * (size_t)n, 256) + 256);
    const int blocks = tv_blocks(n), jobs = tv_jobs(ny, nz);
    const float eps2 = eps * eps;
    CBCT_CUDA_TRY(cudaMemcpyAsync(d_f, d_u, sizeof(float) * (size_t)n, cudaMemcpyDeviceToDevice, st));      // descent starts from f = u
    tv_init_kernel<<<1, 1, 0, st>>>(s);
    CBCT_LAUNCH_CHECK();
    tv_energy_kernel<<<jobs, 256, 0, st>>>(d_f, buf1, d_u, s, 0, mu_tv, eps2, nx, ny, nz, partials);
    CBCT_LAUNCH_CHECK();
    for (int it = 0; it < max_iter; ++it) {
        tv_trial_kernel<<<jobs, 256, 0, st>>>(d_f, buf1, d_u, s, mu_tv, eps2, nx, ny, nz);
        CBCT_LAUNCH_CHECK();
        tv_energy_kernel<<<jobs, 256, 0, st>>>(d_f, buf1, d_u, s, 1, mu_tv, eps2, nx, ny, nz, partials);
        CBCT_LAUNCH_CHECK();
        tv_decide_kernel<<<1, 1, 0, st>>>(s, rel_tol);
        CBCT_LAUNCH_CHECK();
    }
    tv_finish_kernel<<<blocks, 256, 0, st>>>(d_f, buf1, s, clamp_nonneg, n);
    CBCT_LAUNCH_CHECK();
    return CBCT_OK;
}

extern "C" int tv_rof_result(const void *d_work, int nx, int ny, int nz, int *trials, int *accepted, double *energy, void *stream) {
    if (!d_work || nx <= 0 || ny <= 0 || nz <= 0) return CBCT_E_INVALID;
    const unsigned char *w = static_cast<const unsigned char *>(d_work);
    TvState h;
    cudaStream_t st = as_stream(stream);
    CBCT_CUDA_TRY(cudaMemcpyAsync(&h, w + align_up(sizeof(float) * (size_t)nx * ny * nz, 256), sizeof(h), cudaMemcpyDeviceToHost, st));
    CBCT_CUDA_TRY(cudaStreamSynchronize(st));
    if (trials) *trials = h.trials;
    if (accepted) *accepted = h.accepted;
    if (energy) *energy = h.E;
    return CBCT_OK;
}
