// tests/cpu_shim/include/cuda_runtime.h -- TEST INFRASTRUCTURE, not product code.
// Stand-in for the CUDA runtime header: lets the UNCHANGED kernel sources of paper_1008_2042_b200/csrc compile
// with g++ so that `-m "not gpu"` tests can execute every kernel on the host, one fiber per CUDA thread, with
// guard pages around every allocation, bounds checks on shared-memory addresses and hardware-rule checks on the
// TMA calls (tests/cpu_shim/README.md).  It exists to catch indexing, alignment and synchronisation mistakes
// when no GPU is at hand; it is never built, loaded or imported by the package.
#pragma once
#include <stddef.h>
#include <stdint.h>

#include <cmath>
#include <cstdlib>
#include <chrono>
#include <cstring>
#include <functional>
#include <tuple>

// ---- qualifiers -------------------------------------------------------------------------------------------
#define __global__
#define __device__
#define __host__
#define __forceinline__ inline __attribute__((always_inline))
#define __launch_bounds__(...)
#define __grid_constant__
#define __constant__ static
#define __align__(n) alignas(n)
// `__shared__` declarations and `<<<...>>>` launches are rewritten by tests/cpu_shim/cu2cpp.py

// ---- vector types -----------------------------------------------------------------------------------------------
struct float2 { float x, y; };
struct alignas(16) float4 { float x, y, z, w; };
struct alignas(16) double2 { double x, y; };
struct alignas(16) int4 { int x, y, z, w; };
struct alignas(8) int2 { int x, y; };
struct uint3 { unsigned x, y, z; };
struct dim3 {
    unsigned x, y, z;
    constexpr dim3(unsigned x_ = 1, unsigned y_ = 1, unsigned z_ = 1) : x(x_), y(y_), z(z_) {}
};
static inline float2 make_float2(float x, float y) { return float2{x, y}; }
static inline float4 make_float4(float x, float y, float z, float w) { return float4{x, y, z, w}; }
static inline double2 make_double2(double x, double y) { return double2{x, y}; }
static inline int4 make_int4(int x, int y, int z, int w) { return int4{x, y, z, w}; }

extern thread_local uint3 threadIdx, blockIdx;
extern thread_local dim3 blockDim, gridDim;
constexpr int warpSize = 32;

// ---- runtime API (everything is synchronous; streams and events are inert) ------------------------------------------
typedef int cudaError_t;
enum { cudaSuccess = 0, cudaErrorInvalidValue = 1, cudaErrorMemoryAllocation = 2 };
typedef struct shim_stream *cudaStream_t;
typedef struct shim_event *cudaEvent_t;
enum cudaMemcpyKind { cudaMemcpyHostToHost = 0, cudaMemcpyHostToDevice = 1, cudaMemcpyDeviceToHost = 2, cudaMemcpyDeviceToDevice = 3 };
enum cudaDeviceAttr { cudaDevAttrComputeCapabilityMajor = 75 };
enum cudaFuncAttribute { cudaFuncAttributeMaxDynamicSharedMemorySize = 8 };
enum { cudaEnableDefault = 0 };
enum cudaDriverEntryPointQueryResult { cudaDriverEntryPointSuccess = 0, cudaDriverEntryPointSymbolNotFound = 1 };

namespace shim {
void *dev_malloc(size_t bytes);          // guard page right after the (16-byte rounded) end, contents poisoned with 0xFF
void dev_free(void *p);
}
template <class T>
static inline cudaError_t cudaMalloc(T **p, size_t bytes) {
    *p = static_cast<T *>(shim::dev_malloc(bytes));
    return *p ? cudaSuccess : cudaErrorMemoryAllocation;
}
static inline cudaError_t cudaFree(void *p) { shim::dev_free(p); return cudaSuccess; }
enum { cudaHostAllocMapped = 2 };
static inline cudaError_t cudaHostAlloc(void **p, size_t bytes, unsigned) { *p = shim::dev_malloc(bytes); return *p ? cudaSuccess : cudaErrorMemoryAllocation; }
static inline cudaError_t cudaHostGetDevicePointer(void **dp, void *hp, unsigned) { *dp = hp; return cudaSuccess; }   // one address space
static inline cudaError_t cudaFreeHost(void *p) { shim::dev_free(p); return cudaSuccess; }
static inline cudaError_t cudaGetLastError() { return cudaSuccess; }
static inline cudaError_t cudaMemcpy(void *d, const void *s, size_t n, cudaMemcpyKind) { std::memcpy(d, s, n); return cudaSuccess; }
static inline cudaError_t cudaMemcpyAsync(void *d, const void *s, size_t n, cudaMemcpyKind, cudaStream_t = nullptr) {
    std::memmove(d, s, n);
    return cudaSuccess;
}
static inline cudaError_t cudaMemset(void *d, int v, size_t n) { std::memset(d, v, n); return cudaSuccess; }
static inline cudaError_t cudaMemsetAsync(void *d, int v, size_t n, cudaStream_t = nullptr) { std::memset(d, v, n); return cudaSuccess; }
static inline cudaError_t cudaStreamSynchronize(cudaStream_t) { return cudaSuccess; }
static inline cudaError_t cudaDeviceSynchronize() { return cudaSuccess; }
static inline cudaError_t cudaGetDevice(int *d) { *d = 0; return cudaSuccess; }
static inline cudaError_t cudaDeviceGetAttribute(int *v, cudaDeviceAttr, int) { *v = 10; return cudaSuccess; }
// events are wall-clock timestamps: every launch is synchronous here, so "device time between two events" is host time
struct shim_event { double ms; };
static inline cudaError_t cudaEventCreate(cudaEvent_t *e) { *e = new shim_event{0.0}; return cudaSuccess; }
static inline cudaError_t cudaEventDestroy(cudaEvent_t e) { delete e; return cudaSuccess; }
static inline cudaError_t cudaEventRecord(cudaEvent_t e, cudaStream_t = nullptr) {
    if (!e) return cudaErrorInvalidValue;
    e->ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now().time_since_epoch()).count();
    return cudaSuccess;
}
static inline cudaError_t cudaEventSynchronize(cudaEvent_t) { return cudaSuccess; }
static inline cudaError_t cudaEventElapsedTime(float *ms, cudaEvent_t a, cudaEvent_t b) {
    if (!a || !b) return cudaErrorInvalidValue;
    *ms = (float)(b->ms - a->ms);
    return cudaSuccess;
}
cudaError_t cudaFuncSetAttribute(const void *func, cudaFuncAttribute, int value);   // records the opt-in per kernel
template <class F>
static inline cudaError_t cudaFuncSetAttribute(F *func, cudaFuncAttribute a, int value) {
    return cudaFuncSetAttribute(reinterpret_cast<const void *>(func), a, value);
}
cudaError_t cudaGetDriverEntryPoint(const char *symbol, void **fn, int flags, cudaDriverEntryPointQueryResult *q);

// ---- kernel launch, barriers, warp collectives (tests/cpu_shim/shim_runtime.cpp) ------------------------------------------
namespace shim {
void launch(const void *func, dim3 grid, dim3 block, size_t smem_bytes, const std::function<void()> &thread_body);
template <class K, class... A>
static inline void launch_kernel(K *kernel, dim3 grid, dim3 block, size_t smem, cudaStream_t, A... args) {
    auto pack = std::make_tuple(args...);
    launch(reinterpret_cast<const void *>(kernel), grid, block, smem, [&]() { std::apply(kernel, pack); });
}
void *dyn_smem();                                   // this block's dynamic shared memory (exactly smem_bytes, then a guard)
void *static_smem(const void *key, size_t bytes, size_t align);   // one guarded allocation per `__shared__` declaration
template <class T>
static inline T *sh(const void *key) { return static_cast<T *>(static_smem(key, sizeof(T), alignof(T))); }
void syncthreads();
enum WarpOp { W_MIN_S32, W_MAX_S32, W_MAX_U32, W_MIN_U32, W_ADD_S32, W_SHFL_XOR, W_SHFL_DOWN, W_SHFL_IDX, W_BALLOT };
uint64_t warp_collective(unsigned mask, WarpOp op, uint64_t payload, int arg);
[[noreturn]] void fail(const char *fmt, ...);
}
#define SHIM_LAUNCH(...) ::shim::launch_kernel(__VA_ARGS__)
static inline void __syncthreads() { shim::syncthreads(); }
namespace shim { int syncthreads_or(int pred); }
static inline int __syncthreads_or(int pred) { return shim::syncthreads_or(pred); }
static inline void __threadfence_system() { __atomic_thread_fence(__ATOMIC_SEQ_CST); }
static inline void __syncwarp(unsigned mask = 0xffffffffu) { shim::warp_collective(mask, shim::W_BALLOT, 0, 0); }
static inline long long clock64() { return (long long)__builtin_ia32_rdtsc(); }
static inline void __threadfence() { __atomic_thread_fence(__ATOMIC_SEQ_CST); }

static inline int __reduce_min_sync(unsigned m, int v) { return (int)shim::warp_collective(m, shim::W_MIN_S32, (uint64_t)(int64_t)v, 0); }
static inline int __reduce_max_sync(unsigned m, int v) { return (int)shim::warp_collective(m, shim::W_MAX_S32, (uint64_t)(int64_t)v, 0); }
static inline unsigned __reduce_max_sync(unsigned m, unsigned v) { return (unsigned)shim::warp_collective(m, shim::W_MAX_U32, v, 0); }
static inline unsigned __reduce_min_sync(unsigned m, unsigned v) { return (unsigned)shim::warp_collective(m, shim::W_MIN_U32, v, 0); }
static inline int __reduce_add_sync(unsigned m, int v) { return (int)shim::warp_collective(m, shim::W_ADD_S32, (uint64_t)(int64_t)v, 0); }
static inline int __ffs(int v) { return __builtin_ffs(v); }
static inline unsigned __ballot_sync(unsigned m, int pred) { return (unsigned)shim::warp_collective(m, shim::W_BALLOT, pred ? 1 : 0, 0); }
template <class T>
static inline T shim_shfl(unsigned m, shim::WarpOp op, T v, int arg) {
    static_assert(sizeof(T) <= 8, "shuffle payload");
    uint64_t bits = 0;
    std::memcpy(&bits, &v, sizeof(T));
    bits = shim::warp_collective(m, op, bits, arg);
    std::memcpy(&v, &bits, sizeof(T));
    return v;
}
template <class T> static inline T __shfl_xor_sync(unsigned m, T v, int lane_mask) { return shim_shfl(m, shim::W_SHFL_XOR, v, lane_mask); }
template <class T> static inline T __shfl_down_sync(unsigned m, T v, int delta) { return shim_shfl(m, shim::W_SHFL_DOWN, v, delta); }
template <class T> static inline T __shfl_sync(unsigned m, T v, int src) { return shim_shfl(m, shim::W_SHFL_IDX, v, src); }

// ---- atomics (blocks run on several OS threads, so these are real atomics) -------------------------------------------------
static inline int atomicAdd(int *p, int v) { return __atomic_fetch_add(p, v, __ATOMIC_RELAXED); }
static inline unsigned atomicAdd(unsigned *p, unsigned v) { return __atomic_fetch_add(p, v, __ATOMIC_RELAXED); }
static inline unsigned long long atomicAdd(unsigned long long *p, unsigned long long v) { return __atomic_fetch_add(p, v, __ATOMIC_RELAXED); }
static inline float atomicAdd(float *p, float v) {
    float old = *p, want;
    do { want = old + v; } while (!__atomic_compare_exchange(p, &old, &want, true, __ATOMIC_RELAXED, __ATOMIC_RELAXED));
    return old;
}
template <class T>
static inline T shim_atomic_minmax(T *p, T v, bool is_max) {
    T old = __atomic_load_n(p, __ATOMIC_RELAXED);
    while ((is_max ? v > old : v < old) && !__atomic_compare_exchange_n(p, &old, v, true, __ATOMIC_RELAXED, __ATOMIC_RELAXED)) {}
    return old;
}
static inline int atomicOr(int *p, int v) { return __atomic_fetch_or(p, v, __ATOMIC_RELAXED); }
static inline int atomicMax(int *p, int v) { return shim_atomic_minmax(p, v, true); }
static inline unsigned atomicMax(unsigned *p, unsigned v) { return shim_atomic_minmax(p, v, true); }
static inline int atomicMin(int *p, int v) { return shim_atomic_minmax(p, v, false); }
static inline unsigned atomicMin(unsigned *p, unsigned v) { return shim_atomic_minmax(p, v, false); }
static inline unsigned atomicInc(unsigned *p, unsigned limit) {
    unsigned old = __atomic_load_n(p, __ATOMIC_RELAXED), want;
    do { want = old >= limit ? 0 : old + 1; } while (!__atomic_compare_exchange_n(p, &old, want, true, __ATOMIC_SEQ_CST, __ATOMIC_RELAXED));
    return old;
}

// ---- device intrinsics -----------------------------------------------------------------------------------------------
namespace shim { void check_align(const void *p, size_t a, const char *what); }
template <class T>
static inline T __ldg(const T *p) { shim::check_align(p, alignof(T), "__ldg"); return *p; }
static inline float __uint_as_float(unsigned u) { float f; std::memcpy(&f, &u, 4); return f; }
static inline float __int_as_float(int u) { float f; std::memcpy(&f, &u, 4); return f; }
static inline unsigned __float_as_uint(float f) { unsigned u; std::memcpy(&u, &f, 4); return u; }
static inline int __float_as_int(float f) { int u; std::memcpy(&u, &f, 4); return u; }
static inline int __float2int_rn(float f) { return (int)std::lrintf(f); }
static inline int __float2int_rd(float f) { return (int)std::floor(f); }
static inline float __frcp_rn(float x) { return 1.0f / x; }
static inline float __fdividef(float a, float b) { return a / b; }
static inline float __fadd_rd(float a, float b) {          // a + b rounded towards -inf: the fp64 sum of two floats is exact
    const double s = (double)a + (double)b;
    float r = (float)s;
    if ((double)r > s) r = std::nextafterf(r, -INFINITY);
    return r;
}
static inline float __fmul_rn(float a, float b) { volatile float r = a * b; return r; }
static inline float __fadd_rn(float a, float b) { volatile float r = a + b; return r; }
static inline double rsqrt(double x) { return 1.0 / std::sqrt(x); }
static inline float rsqrtf(float x) { return 1.0f / std::sqrt(x); }
static inline float __saturatef(float x) { return x < 0.f ? 0.f : (x > 1.f ? 1.f : x); }
static inline size_t __cvta_generic_to_shared(const void *p);

// min / max overloads as CUDA offers them in the global namespace
static inline int max(int a, int b) { return a > b ? a : b; }
static inline int min(int a, int b) { return a < b ? a : b; }
static inline unsigned max(unsigned a, unsigned b) { return a > b ? a : b; }
static inline unsigned min(unsigned a, unsigned b) { return a < b ? a : b; }
static inline long long max(long long a, long long b) { return a > b ? a : b; }
static inline long long min(long long a, long long b) { return a < b ? a : b; }
static inline long max(long a, long b) { return a > b ? a : b; }
static inline long min(long a, long b) { return a < b ? a : b; }
static inline unsigned long max(unsigned long a, unsigned long b) { return a > b ? a : b; }
static inline unsigned long min(unsigned long a, unsigned long b) { return a < b ? a : b; }
static inline float max(float a, float b) { return std::fmax(a, b); }
static inline float min(float a, float b) { return std::fmin(a, b); }
static inline double max(double a, double b) { return std::fmax(a, b); }
static inline double min(double a, double b) { return std::fmin(a, b); }

namespace shim { unsigned cvta_shared(const void *p); void *shared_ptr_of(unsigned addr, size_t bytes, const char *what); }
static inline size_t __cvta_generic_to_shared(const void *p) { return shim::cvta_shared(p); }
