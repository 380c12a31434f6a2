// microbench.cu -- the per-SM rates the projector kernels are bound by, measured on the device the library runs on
// (include/cbct.h: cbct_microbench).  SURVEY.md §8(d): MEASURED_PEAKS.json holds only HBM and bf16 peaks, while P and
// P^T are bound by instruction issue and shared-memory wavefronts, and the Siddon pair by L2 requests; these kernels
// supply the missing denominators: fp32 FMA issue (scalar FFMA and packed FFMA2), conflict-free LDS and ATOMS.ADD
// wavefronts, L1-hit LDG, L2 read bandwidth on a 64 MB set, and L2 integer reductions (RED.ADD.S32).
// Rates per SM are measured with clock64() inside the kernel (one CTA of 1024 threads per SM, the slowest warp counts),
// so they do not depend on knowing the SM clock; bandwidths are measured with CUDA events on the launching stream.
#include <algorithm>

#include "../../include/cbct_debug.h"
#include "common.cuh"
#include "ptx.cuh"

namespace cbct {

constexpr int MB_UNROLL = 64;

// kind 0: FFMA, kind 1: FFMA2 (8 independent accumulators per thread: the chain never limits issue)
template <int KIND>
__global__ void __launch_bounds__(1024) mb_fma_kernel(int iters, float seed, long long *cycles, float *sink) {
    float a[8];
    f32x2 p[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) { a[i] = seed + i; p[i] = pack2(seed + i, seed - i); }
    const float m = 1.0000001f;
    const f32x2 m2 = pack2(m, m), c2 = pack2(seed, seed);
    __syncthreads();
    const long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < MB_UNROLL / 8; ++u) {
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                if (KIND == 0) a[i] = fmaf(a[i], m, seed);
                else p[i] = fma2(p[i], m2, c2);
            }
        }
    }
    const long long t1 = clock64();
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) { float lo, hi; unpack2(p[i], lo, hi); s += a[i] + lo + hi; }
    if (s == 123.456f) sink[0] = s;                                    // never true: keeps the chains alive
    if ((threadIdx.x & 31) == 0) cycles[blockIdx.x * 32 + (threadIdx.x >> 5)] = t1 - t0;
}

// kind 2: LDS.32, kind 3: ATOMS.ADD.S32; lane l touches word (l + k) of a 4 KB window: 32 distinct banks per instruction
// kind 7: ATOMS.ADD.64, lane l touches the 8-byte word l of an 8 KB window (256 contiguous bytes per instruction)
template <int KIND>
__global__ void __launch_bounds__(1024) mb_smem_kernel(int iters, long long *cycles, float *sink) {
    __shared__ __align__(16) int buf[2048 + 128];
    for (int i = threadIdx.x; i < 2048 + 128; i += blockDim.x) buf[i] = i;
    __syncthreads();
    const unsigned base = smem_u32(buf) + (KIND == 7 ? 8u : 4u) * (threadIdx.x & 31);
    float acc = 0.f;
    const long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
        const unsigned a = base + 128u * (unsigned)(it & 7);
#pragma unroll
        for (int u = 0; u < MB_UNROLL; ++u) {
            if (KIND == 2) acc += lds_f32(a + 128u * (u & 15));
            else if (KIND == 3) red_s32(a + 128u * (u & 15), 1);
            else red_u64(a + 256u * (u & 15), 1ull);
        }
    }
    const long long t1 = clock64();
    if (acc == 123.456f) sink[0] = acc;
    if ((threadIdx.x & 31) == 0) cycles[blockIdx.x * 32 + (threadIdx.x >> 5)] = t1 - t0;
}

// kind 4: LDG.32 hitting L1 (each warp re-reads its own 128-byte line set of 8 KB per CTA)
__global__ void __launch_bounds__(1024) mb_ldg_kernel(int iters, const float *__restrict__ src, long long *cycles, float *sink) {
    const float *p = src + (size_t)blockIdx.x * 2048 + (threadIdx.x & 31);
    float acc = 0.f;
    for (int u = 0; u < 64; ++u) acc += __ldg(p + 32 * u);             // warm the lines
    __syncthreads();
    const long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < MB_UNROLL; ++u) acc += __ldg(p + 32 * ((u + it) & 63));
    }
    const long long t1 = clock64();
    if (acc == 123.456f) sink[0] = acc;
    if ((threadIdx.x & 31) == 0) cycles[blockIdx.x * 32 + (threadIdx.x >> 5)] = t1 - t0;
}

// kind 5: L2 read bandwidth: float4 grid-stride reads of a set that fits L2 (64 MB), repeated
__global__ void __launch_bounds__(256) mb_l2_read_kernel(const float4 *__restrict__ src, long long n4, int reps, float *sink) {
    float acc = 0.f;
    for (int r = 0; r < reps; ++r)
        for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n4; i += (long long)gridDim.x * blockDim.x) {
            const float4 v = ldg_cg_f4(src + i);                          // .cg: served by L2, not kept in L1
            acc += v.x + v.y + v.z + v.w;
        }
    if (acc == 123.456f) sink[0] = acc;
}

// kind 6: L2 integer reductions: every lane adds 1 to its own word of a 64 MB int32 set (coalesced RED.ADD.S32)
__global__ void __launch_bounds__(256) mb_l2_red_kernel(int *dst, long long n, int reps) {
    for (int r = 0; r < reps; ++r)
        for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) atomicAdd(dst + i, 1);
}

}  // namespace cbct

using namespace cbct;

// out[0] = the rate, out[1] = seconds (event time of the measured launch), out[2] = work items of that launch
extern "C" int cbct_microbench(int kind, int iters_arg, double out[3], void *stream) {
    if (!out || kind < 0 || kind > 7) return CBCT_E_INVALID;
    CBCT_TRY(device_supported());
    cudaStream_t st = as_stream(stream);
    // a caller may shorten the timed loops (host-side checks of the kernels); the default is what is reported
    const int n_sm = 148, iters = iters_arg > 0 ? iters_arg : 2000;
    const int reps_rd = iters >= 2000 ? 20 : 1, reps_red = iters >= 2000 ? 4 : 1;
    struct Scratch {                                                   // released on every return path
        long long *cycles = nullptr;
        float *sink = nullptr, *buf = nullptr;
        cudaEvent_t e0 = nullptr, e1 = nullptr;
        ~Scratch() {
            if (e0) cudaEventDestroy(e0);
            if (e1) cudaEventDestroy(e1);
            cudaFree(cycles); cudaFree(sink); cudaFree(buf);
        }
    } sc;
    long long *&d_cycles = sc.cycles;
    float *&d_sink = sc.sink, *&d_buf = sc.buf;
    const size_t set_bytes = (size_t)64 << 20;
    CBCT_CUDA_TRY(cudaMalloc(&d_cycles, sizeof(long long) * n_sm * 32));
    CBCT_CUDA_TRY(cudaMalloc(&d_sink, 256));
    CBCT_CUDA_TRY(cudaMalloc(&d_buf, set_bytes));
    CBCT_CUDA_TRY(cudaMemsetAsync(d_buf, 0, set_bytes, st));
    cudaEvent_t &e0 = sc.e0, &e1 = sc.e1;
    CBCT_CUDA_TRY(cudaEventCreate(&e0));
    CBCT_CUDA_TRY(cudaEventCreate(&e1));
    double work = 0;
    for (int pass = 0; pass < 2; ++pass) {                             // pass 0 warms up, pass 1 is measured
        CBCT_CUDA_TRY(cudaEventRecord(e0, st));
        switch (kind) {
            case 0: mb_fma_kernel<0><<<n_sm, 1024, 0, st>>>(iters, 1.5f, d_cycles, d_sink); break;
            case 1: mb_fma_kernel<1><<<n_sm, 1024, 0, st>>>(iters, 1.5f, d_cycles, d_sink); break;
            case 2: mb_smem_kernel<2><<<n_sm, 1024, 0, st>>>(iters, d_cycles, d_sink); break;
            case 3: mb_smem_kernel<3><<<n_sm, 1024, 0, st>>>(iters, d_cycles, d_sink); break;
            case 7: mb_smem_kernel<7><<<n_sm, 1024, 0, st>>>(iters, d_cycles, d_sink); break;
            case 4: mb_ldg_kernel<<<n_sm, 1024, 0, st>>>(iters, d_buf, d_cycles, d_sink); break;
            case 5: mb_l2_read_kernel<<<n_sm * 8, 256, 0, st>>>(reinterpret_cast<const float4 *>(d_buf), (long long)(set_bytes / 16), reps_rd, d_sink); break;
            case 6: mb_l2_red_kernel<<<n_sm * 8, 256, 0, st>>>(reinterpret_cast<int *>(d_buf), (long long)(set_bytes / 4), reps_red); break;
        }
        CBCT_LAUNCH_CHECK();
        CBCT_CUDA_TRY(cudaEventRecord(e1, st));
    }
    CBCT_CUDA_TRY(cudaEventSynchronize(e1));
    float ms = 0.f;
    CBCT_CUDA_TRY(cudaEventElapsedTime(&ms, e0, e1));
    if (kind <= 4 || kind == 7) {
        std::vector<long long> cyc(n_sm * 32);
        CBCT_CUDA_TRY(cudaMemcpy(cyc.data(), d_cycles, sizeof(long long) * cyc.size(), cudaMemcpyDeviceToHost));
        long long worst = 1;
        for (long long c : cyc) worst = c > worst ? c : worst;
        work = 32.0 * iters * MB_UNROLL;                                // warp instructions per SM
        out[0] = work / (double)worst;                                  // warp instructions per clock per SM
    } else if (kind == 5) {
        work = (double)reps_rd * (double)set_bytes;
        out[0] = work / (ms * 1e-3) / 1e9;                              // GB/s
    } else {
        work = (double)reps_red * (double)(set_bytes / 4);
        out[0] = work / (ms * 1e-3) / 1e9;                              // G reductions per second
    }
    out[1] = ms * 1e-3;
    out[2] = work;
    return CBCT_OK;
}
