// tests/cpu_shim/include/shim_ptx.h -- TEST INFRASTRUCTURE, not product code.
// Host emulation of the wrappers in paper_1008_2042_b200/csrc/ptx.cuh (same names, same signatures).  It is
// force-included before the kernel sources and pre-defines ptx.cuh's include guard, so ptx.cuh contributes nothing.
// Semantics follow the PTX ISA as used by the kernels: mbarrier phases with transaction counts, tiled 3-D bulk
// tensor copies with zero fill of out-of-range elements, tensor reductions that skip them, bulk async-groups.
// Hardware rules the emulation ENFORCES (a violation aborts the test with a message instead of faulting a GPU):
// 128-byte aligned shared-memory box address, 16-byte aligned global address and strides, inner box extent a
// multiple of 16 bytes, box extents <= 256, transaction bytes == box bytes, non-negative reduction coordinates,
// shared addresses inside the launch's shared memory, no shared memory released under an unfinished bulk group.
#pragma once
#define CBCT_PTX_CUH_
#include <cuda.h>
#include <cuda_runtime.h>

namespace shim {
void mbar_init(unsigned bar, unsigned count);
void mbar_expect_tx(unsigned bar, unsigned bytes);
bool mbar_try_wait(unsigned bar, unsigned parity);   // one poll: lets the other fibers run, true once the phase completed
unsigned long long globaltimer_ns();                 // virtual clock of the block: jumps ahead when every live fiber only polls
void tma_load_3d(unsigned dst, const CUtensorMap *map, int c0, int c1, int c2, unsigned bar);
void tma_reduce_add_3d(const CUtensorMap *map, int c0, int c1, int c2, unsigned src);
void bulk_commit();
void bulk_wait(int pending_allowed, bool read_only);
void bank_record(unsigned addr, unsigned kind);       // kind 0: ld.shared, 1: red.shared (bank statistics, off by default)
}  // namespace shim

namespace cbct {

static inline unsigned smem_u32(const void *p) { return shim::cvta_shared(p); }
static inline void mbar_init(unsigned bar, unsigned count) { shim::mbar_init(bar, count); }
static inline void fence_mbar_init() {}
static inline void mbar_expect_tx(unsigned bar, unsigned bytes) { shim::mbar_expect_tx(bar, bytes); }
static inline bool mbar_try_wait(unsigned bar, unsigned parity) { return shim::mbar_try_wait(bar, parity); }
static inline unsigned long long globaltimer_ns() { return shim::globaltimer_ns(); }
static inline void tma_load_3d(unsigned dst, const CUtensorMap *map, int c0, int c1, int c2, unsigned bar) {
    shim::tma_load_3d(dst, map, c0, c1, c2, bar);
}
static inline void tma_reduce_add_3d(const CUtensorMap *map, int c0, int c1, int c2, unsigned src) {
    shim::tma_reduce_add_3d(map, c0, c1, c2, src);
}
static inline void bulk_commit() { shim::bulk_commit(); }
static inline void bulk_wait_read0() { shim::bulk_wait(0, true); }
static inline void bulk_wait0() { shim::bulk_wait(0, false); }
static inline void fence_async_smem() {}

static inline float lds_f32(unsigned addr) { shim::bank_record(addr, 0); return *static_cast<const float *>(shim::shared_ptr_of(addr, 4, "ld.shared.f32")); }
template <int OFF>
static inline float lds_f32_off(unsigned addr) { return lds_f32(addr + (unsigned)OFF); }
static inline void red_s32(unsigned addr, int v) { shim::bank_record(addr, 1); *static_cast<int *>(shim::shared_ptr_of(addr, 4, "red.shared.add.s32")) += v; }
template <int OFF>
static inline void red_s32_off(unsigned addr, int v) { red_s32(addr + (unsigned)OFF, v); }

static inline void red_u64(unsigned addr, unsigned long long v) { *static_cast<unsigned long long *>(shim::shared_ptr_of(addr, 8, "red.shared.add.u64")) += v; }
template <int BF, int BS>
static inline void red_s32_x8_if(unsigned addr, const int (&v)[8], bool pred) {
    const unsigned off[8] = {0, 4, 4 * BF, 4 * BF + 4, 4 * BF * BS, 4 * BF * BS + 4, 4 * BF * BS + 4 * BF, 4 * BF * BS + 4 * BF + 4};
    for (int i = 0; i < 8; ++i) {
        if (pred) red_s32(addr + off[i], v[i]);
        else shim::bank_record(0xffffffffu, 2);          // keeps the lane's instruction ordinal aligned with its warp
    }
}
static inline float4 ldg_cg_f4(const float4 *p) { shim::check_align(p, 16, "ld.global.cg.v4"); return *p; }

// packed fp32 pairs: two independent IEEE operations
typedef unsigned long long f32x2;
static inline f32x2 pack2(float lo, float hi) { f32x2 r; float v[2] = {lo, hi}; std::memcpy(&r, v, 8); return r; }
static inline void unpack2(f32x2 p, float &lo, float &hi) { float v[2]; std::memcpy(v, &p, 8); lo = v[0]; hi = v[1]; }
static inline f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) {
    float a0, a1, b0, b1, c0, c1;
    unpack2(a, a0, a1); unpack2(b, b0, b1); unpack2(c, c0, c1);
    return pack2(std::fmaf(a0, b0, c0), std::fmaf(a1, b1, c1));
}
static inline f32x2 add2(f32x2 a, f32x2 b) { float a0, a1, b0, b1; unpack2(a, a0, a1); unpack2(b, b0, b1); return pack2(__fadd_rn(a0, b0), __fadd_rn(a1, b1)); }
static inline f32x2 sub2(f32x2 a, f32x2 b) { float a0, a1, b0, b1; unpack2(a, a0, a1); unpack2(b, b0, b1); return pack2(__fadd_rn(a0, -b0), __fadd_rn(a1, -b1)); }
static inline f32x2 mul2(f32x2 a, f32x2 b) { float a0, a1, b0, b1; unpack2(a, a0, a1); unpack2(b, b0, b1); return pack2(__fmul_rn(a0, b0), __fmul_rn(a1, b1)); }
static inline f32x2 add2_rd(f32x2 a, f32x2 b) { float a0, a1, b0, b1; unpack2(a, a0, a1); unpack2(b, b0, b1); return pack2(__fadd_rd(a0, b0), __fadd_rd(a1, b1)); }

}  // namespace cbct
