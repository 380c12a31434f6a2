// tests/cpu_shim/shim_runtime.cpp -- TEST INFRASTRUCTURE, not product code (see README.md in this directory).
// Executes CUDA kernels on the host: one fiber (ucontext) per CUDA thread, the fibers of a block scheduled round-robin
// on one OS thread, blocks spread over OS threads.  __syncthreads, warp collectives, mbarriers and bulk async-groups
// are scheduling points.  Every allocation ends at a guard page; shared-memory addresses are bounds-checked; the
// TMA emulation enforces the hardware's alignment and size rules.  The first violation is recorded (shim_last_error)
// and the launch is abandoned, so a test fails with a message where a GPU would raise Xid 13 / hang.
#include <cuda.h>
#include <cuda_runtime.h>
#include <cxxabi.h>
#include <dlfcn.h>
#include <execinfo.h>
#include <fcntl.h>
#include <omp.h>
#include <signal.h>
#include <stdarg.h>
#include <stdio.h>
#include <sys/mman.h>
#include <ucontext.h>
#include <unistd.h>

#include <algorithm>
#include <map>
#include <mutex>
#include <string>
#include <unordered_map>
#include <vector>

thread_local uint3 threadIdx, blockIdx;
thread_local dim3 blockDim, gridDim;

namespace shim {

// ---- error record -------------------------------------------------------------------------------------------------
static std::mutex g_err_mu;
static std::string g_error;
static volatile bool g_failed = false;
static void record_error(const char *msg) {
    std::lock_guard<std::mutex> lk(g_err_mu);
    if (g_error.empty()) g_error = msg;
    g_failed = true;
}

// ---- guarded memory ---------------------------------------------------------------------------------------------
struct Alloc { void *map; size_t map_bytes; size_t bytes; };
static std::mutex g_mem_mu;
static std::map<uintptr_t, Alloc> g_allocs;          // keyed by user pointer
static const size_t PAGE = 4096;

static void *guarded(size_t bytes, size_t align, Alloc *rec) {
    const size_t rounded = (bytes + align - 1) / align * align;
    const size_t body = (rounded + PAGE - 1) / PAGE * PAGE;
    unsigned char *m = static_cast<unsigned char *>(mmap(nullptr, body + 2 * PAGE, PROT_READ | PROT_WRITE, MAP_PRIVATE | MAP_ANONYMOUS, -1, 0));
    if (m == MAP_FAILED) return nullptr;
    mprotect(m, PAGE, PROT_NONE);                     // guard below (not tight) and right above the end (tight)
    mprotect(m + PAGE + body, PAGE, PROT_NONE);
    unsigned char *user = m + PAGE + body - rounded;
    std::memset(m + PAGE, 0xFF, body);                // NaN / -1: reads of never-written memory show up in results
    if (rec) *rec = Alloc{m, body + 2 * PAGE, bytes};
    return user;
}

void *dev_malloc(size_t bytes) {
    Alloc a;
    void *p = guarded(bytes ? bytes : 1, 256, &a);
    if (!p) return nullptr;
    std::lock_guard<std::mutex> lk(g_mem_mu);
    g_allocs[reinterpret_cast<uintptr_t>(p)] = a;
    return p;
}
void dev_free(void *p) {
    if (!p) return;
    std::lock_guard<std::mutex> lk(g_mem_mu);
    auto it = g_allocs.find(reinterpret_cast<uintptr_t>(p));
    if (it == g_allocs.end()) { record_error("cudaFree of a pointer cudaMalloc did not return"); return; }
    munmap(it->second.map, it->second.map_bytes);
    g_allocs.erase(it);
}

// a fault on a guard page is the whole point of the guards: say which allocation, which kernel thread, and where
static thread_local const char *t_kernel = "";
static int g_fault_fd = 2;                              // pytest captures fd 2 and _exit loses the capture: SHIM_FAULT_LOG names a file
static void on_segv(int, siginfo_t *si, void *) {
    char buf[512];
    if (const char *path = getenv("SHIM_FAULT_LOG")) {
        const int fd = open(path, O_WRONLY | O_CREAT | O_TRUNC, 0644);
        if (fd >= 0) g_fault_fd = fd;
    }
    const uintptr_t a = reinterpret_cast<uintptr_t>(si->si_addr);
    int n = snprintf(buf, sizeof buf, "\ncpu_shim: SIGSEGV at %p in kernel '%s' block (%u,%u,%u) thread (%u,%u,%u)\n", si->si_addr, t_kernel,
                     blockIdx.x, blockIdx.y, blockIdx.z, threadIdx.x, threadIdx.y, threadIdx.z);
    if (write(g_fault_fd, buf, n) < 0) {}
    for (auto &kv : g_allocs) {                        // no lock: we are crashing anyway
        const uintptr_t lo = reinterpret_cast<uintptr_t>(kv.second.map), hi = lo + kv.second.map_bytes;
        if (a >= lo && a < hi) {
            n = snprintf(buf, sizeof buf, "cpu_shim: the address is %lld bytes past the END of a cudaMalloc'ed buffer of %zu bytes (base %p)\n",
                         (long long)(a - (kv.first + kv.second.bytes)), kv.second.bytes, reinterpret_cast<void *>(kv.first));
            if (write(g_fault_fd, buf, n) < 0) {}
        }
    }
    void *frames[48];
    backtrace_symbols_fd(frames, backtrace(frames, 48), g_fault_fd);
    _exit(139);
}
static void install_segv_handler() {                   // per OS thread: its own alternate stack; the action is process-wide
    stack_t ss;
    ss.ss_sp = malloc(64 * 1024); ss.ss_size = 64 * 1024; ss.ss_flags = 0;
    sigaltstack(&ss, nullptr);
    struct sigaction sa;
    memset(&sa, 0, sizeof sa);
    sa.sa_sigaction = on_segv;
    sa.sa_flags = SA_SIGINFO | SA_ONSTACK;
    sigaction(SIGSEGV, &sa, nullptr);
}

// ---- per-OS-thread worker state ------------------------------------------------------------------------------------------
enum State { READY, WAIT_BLOCK, WAIT_WARP, SPIN, DONE };
struct BulkOp { CUtensorMap map; int c[3]; unsigned src; };
struct Fiber {
    ucontext_t ctx;
    State state;
    uint3 tid;
    int lin;
    unsigned wmask; WarpOp wop; uint64_t wpayload, wresult; int warg;
    unsigned seq;                                     // ordinal of the next shared-memory instruction since the last barrier
    std::vector<BulkOp> open_group;                   // tensor reductions issued since the last commit
    std::vector<std::vector<BulkOp>> groups;          // committed, not yet executed (lazy mode), oldest first
};
struct PendingLoad { CUtensorMap map; int c[3]; unsigned dst, bar; };
struct BankRec { unsigned warp, seq, addr, kind; };     // one lane of one shared-memory instruction (bank statistics)
struct StaticShared { const void *key; unsigned char *ptr; size_t bytes; unsigned vaddr; };
struct Worker {
    std::vector<Fiber> fibers;
    unsigned char *stack_region = nullptr;
    ucontext_t sched;
    int cur = -1, live = 0, nthreads = 0;
    bool progress = false, aborted = false;
    const std::function<void()> *body = nullptr;
    unsigned char *dyn_region = nullptr;              // 256 KiB + guard, allocated once
    unsigned char *dyn_base = nullptr;
    size_t dyn_bytes = 0;
    std::vector<StaticShared> statics;
    unsigned static_next = 0x100;
    std::vector<PendingLoad> loads;                   // lazy mode: issued, not yet performed
    std::vector<BankRec> bank;                        // bank statistics of the running block
    unsigned epoch = 0;                               // __syncthreads count: re-aligns the lanes' instruction ordinals
    int or_acc[2] = {0, 0};                           // __syncthreads_or: predicate accumulators of this / the next barrier
    unsigned long long vclock = 0;                    // %globaltimer of the block (ns): advances only when the block would idle
    bool timed_wait = false;                          // some fiber polls against the clock: idling advances it instead of deadlocking
    int clock_jumps = 0;
};
static thread_local Worker *tw = nullptr;
static const size_t STACK_BYTES = 256 * 1024, DYN_MAX = 232448;       // 227 KiB
static const unsigned DYN_VADDR = 0x100000;
static int g_order = 0;                                // SHIM_ORDER: 0 ascending, 1 reverse, 2 random (seeded per block)
static bool g_lazy = false;                            // SHIM_TMA=lazy: async copies land at the last legal moment

// Workers are pooled: OpenMP may retire and re-create its threads between launches, so a worker (fiber stacks,
// shared-memory allocations) is borrowed for the duration of one launch and handed back.
static std::mutex g_pool_mu;
static std::vector<Worker *> g_pool;
static thread_local bool t_altstack = false;
static Worker *acquire_worker() {
    if (!t_altstack) { install_segv_handler(); t_altstack = true; }
    {
        std::lock_guard<std::mutex> lk(g_pool_mu);
        if (!g_pool.empty()) { Worker *w = g_pool.back(); g_pool.pop_back(); return tw = w; }
    }
    Worker *w = new Worker();
    Alloc a;
    w->dyn_region = static_cast<unsigned char *>(guarded(DYN_MAX, 128, &a));
    // one mapping for the 1024 fiber stacks (touched lazily)
    w->stack_region = static_cast<unsigned char *>(mmap(nullptr, 1024 * STACK_BYTES, PROT_READ | PROT_WRITE,
                                                        MAP_PRIVATE | MAP_ANONYMOUS | MAP_NORESERVE, -1, 0));
    if (!w->dyn_region || w->stack_region == MAP_FAILED) { fprintf(stderr, "cpu_shim: out of address space\n"); abort(); }
    return tw = w;
}
static void release_worker(Worker *w) {
    tw = nullptr;
    std::lock_guard<std::mutex> lk(g_pool_mu);
    g_pool.push_back(w);
}
static inline Fiber &me() { return tw->fibers[tw->cur]; }

static void yield_to_scheduler() {
    Worker *w = tw;
    Fiber &f = w->fibers[w->cur];
    swapcontext(&f.ctx, &w->sched);
}

[[noreturn]] void fail(const char *fmt, ...) {
    char buf[1024];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    char where[256] = "";
    if (tw && tw->cur >= 0)
        snprintf(where, sizeof where, " [block (%u,%u,%u) thread (%u,%u,%u)]", blockIdx.x, blockIdx.y, blockIdx.z, threadIdx.x,
                 threadIdx.y, threadIdx.z);
    record_error((std::string(buf) + where).c_str());
    if (tw && tw->cur >= 0) {
        tw->aborted = true;
        me().state = DONE;
        yield_to_scheduler();
    }
    fprintf(stderr, "cpu_shim: %s\n", buf);
    abort();
}

void check_align(const void *p, size_t a, const char *what) {
    if (reinterpret_cast<uintptr_t>(p) & (a - 1)) fail("%s: address %p is not %zu-byte aligned", what, p, a);
}

static void fiber_entry() {
    Worker *w = tw;
    (*w->body)();
    Fiber &f = w->fibers[w->cur];
    if (!f.open_group.empty() || !f.groups.empty())
        fail("thread exits with an unfinished bulk async-group (cp.async.bulk.wait_group missing: shared memory would be "
             "released under the TMA unit)");
    f.state = DONE;
    yield_to_scheduler();
}

void *dyn_smem() { return tw->dyn_base; }

void *static_smem(const void *key, size_t bytes, size_t align) {
    Worker *w = tw;
    for (auto &s : w->statics)
        if (s.key == key) return s.ptr;
    Alloc a;
    StaticShared s;
    s.key = key; s.bytes = bytes;
    s.ptr = static_cast<unsigned char *>(guarded(bytes, align < 16 ? 16 : align, &a));
    w->static_next = (w->static_next + 127) & ~127u;
    s.vaddr = w->static_next;
    w->static_next += (unsigned)bytes;
    w->statics.push_back(s);
    return s.ptr;
}

unsigned cvta_shared(const void *p) {
    Worker *w = tw;
    const unsigned char *q = static_cast<const unsigned char *>(p);
    if (q >= w->dyn_base && q <= w->dyn_base + w->dyn_bytes) return DYN_VADDR + (unsigned)(q - w->dyn_base);
    for (auto &s : w->statics)
        if (q >= s.ptr && q < s.ptr + s.bytes) return s.vaddr + (unsigned)(q - s.ptr);
    fail("__cvta_generic_to_shared: %p is not in this block's shared memory", p);
}

// ---- shared-memory bank statistics (shim_bank_stats_enable) ----------------------------------------------------------------------
// A warp's lanes execute the k-th ld.shared / red.shared after a barrier together (lanes that have run out of loop
// iterations are masked off), so grouping the recorded lane addresses by (warp, barrier epoch, ordinal) reconstructs the
// warp instructions.  Wavefronts of one instruction = the largest number of requests falling on one of the 32 banks:
// for loads, lanes reading the same word share a request (broadcast); for atomic reductions every lane is a request
// (measured on B200: 32 clk when all lanes hit one word, profiles/README.md).
static bool g_bank_on = false;
static std::mutex g_bank_mu;
static double g_bank_tot[4] = {0, 0, 0, 0};             // ld instr, ld wavefronts, red instr, red wavefronts
void bank_record(unsigned addr, unsigned kind) {
    if (!g_bank_on) return;
    Worker *w = tw;
    Fiber &f = w->fibers[w->cur];
    if (kind == 2) { ++f.seq; return; }                 // a lane predicated off: the ordinal advances, no request
    w->bank.push_back(BankRec{(unsigned)f.lin >> 5, (w->epoch << 18) | (f.seq++ & 0x3ffff), addr, kind});
}
static void bank_flush(Worker *w) {
    if (w->bank.empty()) return;
    std::sort(w->bank.begin(), w->bank.end(), [](const BankRec &a, const BankRec &b) {
        return a.warp != b.warp ? a.warp < b.warp : (a.seq != b.seq ? a.seq < b.seq : a.addr < b.addr);
    });
    double tot[4] = {0, 0, 0, 0};
    for (size_t i = 0; i < w->bank.size();) {
        size_t j = i;
        int per_bank[32] = {0};
        unsigned last_word[32];
        for (; j < w->bank.size() && w->bank[j].warp == w->bank[i].warp && w->bank[j].seq == w->bank[i].seq; ++j) {
            const unsigned word = w->bank[j].addr >> 2, b = word & 31;
            if (w->bank[i].kind == 0 && per_bank[b] && last_word[b] == word) continue;       // broadcast (sorted by address)
            ++per_bank[b]; last_word[b] = word;
        }
        int wf = 0;
        for (int b = 0; b < 32; ++b) wf = std::max(wf, per_bank[b]);
        tot[2 * w->bank[i].kind] += 1; tot[2 * w->bank[i].kind + 1] += wf;
        i = j;
    }
    w->bank.clear();
    std::lock_guard<std::mutex> lk(g_bank_mu);
    for (int k = 0; k < 4; ++k) g_bank_tot[k] += tot[k];
}

void *shared_ptr_of(unsigned addr, size_t bytes, const char *what) {
    Worker *w = tw;
    if (addr >= DYN_VADDR) {
        const size_t off = addr - DYN_VADDR;
        if (off + bytes > w->dyn_bytes) fail("%s: shared address +%zu (%zu bytes) is outside the %zu bytes of dynamic shared memory", what, off, bytes, w->dyn_bytes);
        if (off & (bytes < 16 ? bytes - 1 : 15)) fail("%s: shared address +%zu is misaligned for %zu bytes", what, off, bytes);
        return w->dyn_base + off;
    }
    for (auto &s : w->statics)
        if (addr >= s.vaddr && addr + bytes <= s.vaddr + s.bytes) return s.ptr + (addr - s.vaddr);
    fail("%s: shared address 0x%x is outside every shared allocation of this block", what, addr);
}

// ---- barriers and warp collectives -------------------------------------------------------------------------------------------
void syncthreads() {
    me().state = WAIT_BLOCK;
    yield_to_scheduler();
}

int syncthreads_or(int pred) {
    Worker *w = tw;
    const unsigned slot = w->epoch & 1;               // the slot of the NEXT barrier was cleared when this epoch began
    if (pred) w->or_acc[slot] = 1;
    me().state = WAIT_BLOCK;
    yield_to_scheduler();
    return w->or_acc[slot];
}

static void spin() {                                  // give the other fibers a turn, then re-test the caller's condition
    me().state = SPIN;
    yield_to_scheduler();
}

uint64_t warp_collective(unsigned mask, WarpOp op, uint64_t payload, int arg) {
    Fiber &f = me();
    if (!(mask >> (f.lin & 31) & 1)) fail("warp collective: the calling lane is not in the mask 0x%x", mask);
    f.wmask = mask; f.wop = op; f.wpayload = payload; f.warg = arg;
    f.state = WAIT_WARP;
    yield_to_scheduler();
    return me().wresult;
}

static void complete_warp(Worker *w, int warp) {
    const int lo = warp * 32, hi = std::min(lo + 32, w->nthreads);
    int waiting = 0, alive = 0;
    for (int i = lo; i < hi; ++i) {
        alive += w->fibers[i].state != DONE;
        waiting += w->fibers[i].state == WAIT_WARP;
    }
    if (!waiting || waiting < alive) return;
    const Fiber &first = *[&]() { for (int i = lo; i < hi; ++i) if (w->fibers[i].state == WAIT_WARP) return &w->fibers[i]; return (Fiber *)nullptr; }();
    int64_t smin = INT64_MAX, smax = INT64_MIN;
    uint64_t umax = 0, umin = UINT64_MAX, ballot = 0, sadd = 0;      // sadd wraps (payloads of other collectives are arbitrary bits)
    for (int i = lo; i < hi; ++i) {
        Fiber &g = w->fibers[i];
        if (g.state != WAIT_WARP) continue;
        if (g.wop != first.wop || g.wmask != first.wmask) {
            record_error("warp collective: lanes of one warp wait in different collectives (divergent *_sync call)");
            w->aborted = true;
            return;
        }
        const int64_t s = (int64_t)g.wpayload;
        smin = std::min(smin, s); smax = std::max(smax, s); sadd += (uint64_t)s;
        umax = std::max(umax, g.wpayload); umin = std::min(umin, g.wpayload);
        if (g.wpayload) ballot |= 1ull << (i - lo);
    }
    for (int i = lo; i < hi; ++i) {
        Fiber &g = w->fibers[i];
        if (g.state != WAIT_WARP) continue;
        int src = -1;
        switch (g.wop) {
            case W_MIN_S32: g.wresult = (uint64_t)smin; break;
            case W_MAX_S32: g.wresult = (uint64_t)smax; break;
            case W_ADD_S32: g.wresult = sadd; break;
            case W_MAX_U32: g.wresult = umax; break;
            case W_MIN_U32: g.wresult = umin; break;
            case W_BALLOT: g.wresult = ballot; break;
            case W_SHFL_XOR: src = (i - lo) ^ g.warg; break;
            case W_SHFL_DOWN: src = (i - lo) + g.warg; break;
            case W_SHFL_IDX: src = g.warg & 31; break;
        }
        if (g.wop == W_SHFL_XOR || g.wop == W_SHFL_DOWN || g.wop == W_SHFL_IDX) {
            const bool ok = src >= 0 && src < 32 && lo + src < hi && w->fibers[lo + src].state == WAIT_WARP;
            g.wresult = ok ? w->fibers[lo + src].wpayload : g.wpayload;
        }
    }
    for (int i = lo; i < hi; ++i)
        if (w->fibers[i].state == WAIT_WARP) w->fibers[i].state = READY;
    w->progress = true;
}

// ---- launch ------------------------------------------------------------------------------------------------------------
static std::mutex g_attr_mu;
static std::unordered_map<const void *, int> g_max_dyn;
static std::string g_cur_kernel;
static long long g_block_stride = 1;                   // statistics runs: execute every n-th block only (outputs incomplete)
static std::string g_kernel_log;                       // demangled names of the kernels launched, one per line

static void log_kernel(const void *func, dim3 grid, dim3 block, size_t smem) {
    Dl_info info;
    std::string name = "?";
    if (dladdr(func, &info) && info.dli_sname) {
        int st = 0;
        char *d = abi::__cxa_demangle(info.dli_sname, nullptr, nullptr, &st);
        name = st == 0 && d ? d : info.dli_sname;
        free(d);
        const size_t paren = name.find('(');               // keep "ns::kernel<args>", drop the parameter list
        if (paren != std::string::npos) name.resize(paren);
        const size_t sp = name.rfind(' ');                 // templates demangle as "void ns::kernel<...>"
        if (sp != std::string::npos && name.compare(0, 5, "void ") == 0) name = name.substr(5);
    }
    char buf[160];
    snprintf(buf, sizeof buf, " grid=(%u,%u,%u) block=(%u,%u,%u) smem=%zu\n", grid.x, grid.y, grid.z, block.x, block.y, block.z, smem);
    std::lock_guard<std::mutex> lk(g_attr_mu);
    g_kernel_log += name + buf;
    g_cur_kernel = name;
    if (getenv("SHIM_TRACE")) fprintf(stderr, "cpu_shim launch: %s%s", name.c_str(), buf);
}

static void run_block(Worker *w, const std::function<void()> &body, dim3 grid, dim3 block, uint3 bid, size_t smem) {
    const int n = (int)(block.x * block.y * block.z);
    w->nthreads = n; w->live = n; w->body = &body; w->aborted = false;
    t_kernel = g_cur_kernel.c_str();
    w->dyn_bytes = smem;
    w->dyn_base = w->dyn_region + DYN_MAX - ((smem + 127) & ~(size_t)127);
    if (smem) std::memset(w->dyn_base, 0xFF, smem);
    w->loads.clear();
    w->bank.clear(); w->epoch = 0;
    w->or_acc[0] = w->or_acc[1] = 0; w->vclock = 0; w->timed_wait = false; w->clock_jumps = 0;
    if ((int)w->fibers.size() < n) w->fibers.resize(n);
    gridDim = grid; blockDim = block; blockIdx = bid;
    for (int i = 0; i < n; ++i) {
        Fiber &f = w->fibers[i];
        f.state = READY; f.lin = i; f.seq = 0;
        f.tid = uint3{(unsigned)i % block.x, ((unsigned)i / block.x) % block.y, (unsigned)i / (block.x * block.y)};
        f.open_group.clear(); f.groups.clear();
        getcontext(&f.ctx);
        f.ctx.uc_stack.ss_sp = w->stack_region + (size_t)i * STACK_BYTES;
        f.ctx.uc_stack.ss_size = STACK_BYTES;
        f.ctx.uc_link = nullptr;
        makecontext(&f.ctx, fiber_entry, 0);
    }
    int idle_passes = 0;
    unsigned long long rng = 0x9e3779b97f4a7c15ull ^ ((unsigned long long)bid.x << 40) ^ ((unsigned long long)bid.y << 20) ^ bid.z;
    while (w->live > 0 && !w->aborted && !g_failed) {
        w->progress = false;
        rng = rng * 6364136223846793005ull + 1442695040888963407ull;
        const unsigned rot = (unsigned)(rng >> 33) % (unsigned)n, rdir = (unsigned)(rng >> 20) & 1u;
        for (int k = 0; k < n && !w->aborted; ++k) {
            // SHIM_ORDER=reverse: the last thread of the block runs first; random: a different rotation and direction per pass
            const int i = g_order == 1 ? n - 1 - k : (g_order == 2 ? (int)((rot + (unsigned)(rdir ? k : n - 1 - k)) % (unsigned)n) : k);
            Fiber &f = w->fibers[i];
            if (f.state != READY && f.state != SPIN) continue;
            const bool was_spin = f.state == SPIN;
            f.state = READY;
            w->cur = i;
            threadIdx = f.tid;
            swapcontext(&w->sched, &f.ctx);
            w->cur = -1;
            if (f.state == DONE) { --w->live; w->progress = true; complete_warp(w, i / 32); }
            else if (f.state == WAIT_WARP) { w->progress = true; complete_warp(w, i / 32); }
            else if (f.state == WAIT_BLOCK) w->progress = true;
            else if (f.state == SPIN && !was_spin) w->progress = true;
        }
        int waiting = 0;
        for (int i = 0; i < n; ++i) waiting += w->fibers[i].state == WAIT_BLOCK;
        if (waiting && waiting == w->live) {
            for (int i = 0; i < n; ++i)
                if (w->fibers[i].state == WAIT_BLOCK) { w->fibers[i].state = READY; w->fibers[i].seq = 0; }
            ++w->epoch;
            w->or_acc[w->epoch & 1] = 0;
            w->progress = true;
        }
        idle_passes = w->progress ? 0 : idle_passes + 1;
        if (idle_passes > 4 && w->timed_wait && w->clock_jumps < 64) {
            // every live fiber only polls, and at least one polls against %globaltimer: let (virtual) time pass so that
            // its bound expires -- a bounded wait must END as an error path, which is what the tests check
            w->vclock += 1000ull * 1000ull * 1000ull;
            ++w->clock_jumps;
            idle_passes = 0;
            continue;
        }
        if (idle_passes > 4) {
            char buf[256];
            int nb = 0, nw = 0, ns = 0;
            for (int i = 0; i < n; ++i) { nb += w->fibers[i].state == WAIT_BLOCK; nw += w->fibers[i].state == WAIT_WARP; ns += w->fibers[i].state == SPIN; }
            snprintf(buf, sizeof buf, "deadlock in block (%u,%u,%u): %d threads at __syncthreads, %d in a warp collective, %d spinning on an "
                     "mbarrier / bulk group, %d alive", bid.x, bid.y, bid.z, nb, nw, ns, w->live);
            record_error(buf);
            w->aborted = true;
        }
    }
    if (!w->loads.empty() && !w->aborted && !g_failed) record_error("block ends with a TMA load in flight that nobody waited for");
    bank_flush(w);
}

void launch(const void *func, dim3 grid, dim3 block, size_t smem, const std::function<void()> &body) {
    if (g_failed) return;
    log_kernel(func, grid, block, smem);
    const char *mode = getenv("SHIM_TMA");
    g_lazy = mode && !strcmp(mode, "lazy");
    const char *order = getenv("SHIM_ORDER");
    g_order = !order ? 0 : (!strcmp(order, "reverse") ? 1 : (!strcmp(order, "random") ? 2 : 0));
    const size_t nthreads = (size_t)block.x * block.y * block.z;
    if (!nthreads || nthreads > 1024 || block.z > 64) { record_error("launch: invalid block size"); return; }
    if (!grid.x || !grid.y || !grid.z || grid.y > 65535 || grid.z > 65535) { record_error("launch: invalid grid size (y, z <= 65535)"); return; }
    {
        std::lock_guard<std::mutex> lk(g_attr_mu);
        auto it = g_max_dyn.find(func);
        const size_t allowed = it == g_max_dyn.end() ? 48 * 1024 : (size_t)it->second;
        if (smem > allowed || smem > DYN_MAX) {
            record_error("launch: dynamic shared memory above 48 KiB without cudaFuncSetAttribute(MaxDynamicSharedMemorySize), or above 227 KiB");
            return;
        }
    }
    const long long nblocks = (long long)grid.x * grid.y * grid.z;
    const char *nt = getenv("SHIM_THREADS");
    int threads = nt ? atoi(nt) : omp_get_max_threads();
    if (threads < 1) threads = 1;
    if (nblocks < threads) threads = (int)nblocks;
#pragma omp parallel num_threads(threads)
    {
        Worker *w = acquire_worker();
#pragma omp for schedule(dynamic, 1)
        for (long long b = 0; b < nblocks; ++b) {
            if (g_failed || (g_block_stride > 1 && b % g_block_stride)) continue;
            const uint3 bid{(unsigned)(b % grid.x), (unsigned)((b / grid.x) % grid.y), (unsigned)(b / ((long long)grid.x * grid.y))};
            run_block(w, body, grid, block, bid, smem);
        }
        release_worker(w);
    }
}

// ---- mbarrier -------------------------------------------------------------------------------------------------------
struct MBar { uint8_t phase, init, pending, armed; int32_t tx; };
static_assert(sizeof(MBar) == 8, "mbarrier is one 64-bit word");
static MBar *bar_at(unsigned bar) {
    if (bar & 7) fail("mbarrier address 0x%x is not 8-byte aligned", bar);
    return static_cast<MBar *>(shared_ptr_of(bar, 8, "mbarrier"));
}
static void bar_check(MBar *b) {
    if (b->pending == 0 && b->tx == 0) { b->phase ^= 1; b->pending = b->init; }
}
void mbar_init(unsigned bar, unsigned count) {
    MBar *b = bar_at(bar);
    if (!count || count > 255) fail("mbarrier.init: count %u", count);
    b->phase = 0; b->init = (uint8_t)count; b->pending = (uint8_t)count; b->armed = 0xA5; b->tx = 0;
}
void mbar_expect_tx(unsigned bar, unsigned bytes) {
    MBar *b = bar_at(bar);
    if (b->armed != 0xA5) fail("mbarrier.arrive.expect_tx on a barrier that was never initialised");
    if (!b->pending) fail("mbarrier.arrive: more arrivals than the barrier's count");
    b->tx += (int32_t)bytes;
    --b->pending;
    bar_check(b);
}
static void perform_load(const PendingLoad &l);
bool mbar_try_wait(unsigned bar, unsigned parity) {
    MBar *b = bar_at(bar);
    if (b->armed != 0xA5) fail("mbarrier.try_wait on a barrier that was never initialised");
    Worker *w = tw;
    for (size_t i = 0; i < w->loads.size();) {        // lazy mode: the copy lands when somebody first needs it
        if (w->loads[i].bar == bar) {
            const PendingLoad l = w->loads[i];
            w->loads.erase(w->loads.begin() + i);
            perform_load(l);
        } else ++i;
    }
    if (b->phase != (parity & 1)) return true;
    spin();                                           // the hardware instruction blocks for a time slice: others run
    return bar_at(bar)->phase != (parity & 1);
}
unsigned long long globaltimer_ns() {
    tw->timed_wait = true;
    return tw->vclock;
}

// ---- tensor maps and bulk tensor operations ------------------------------------------------------------------------------------
struct MapRec { uint64_t magic; unsigned char *base; uint64_t dims[3]; uint64_t strides[2]; uint32_t box[3]; int32_t dtype; };
static_assert(sizeof(MapRec) <= sizeof(CUtensorMap), "record fits the opaque map");
static const uint64_t MAP_MAGIC = 0x43424354544d4150ull;

static CUresult encode_tiled(CUtensorMap *m, CUtensorMapDataType dtype, cuuint32_t rank, void *base, const cuuint64_t *dims,
                             const cuuint64_t *strides, const cuuint32_t *box, const cuuint32_t *estr, CUtensorMapInterleave il,
                             CUtensorMapSwizzle sw, CUtensorMapL2promotion, CUtensorMapFloatOOBfill) {
    if (!m || rank != 3 || !base || il != CU_TENSOR_MAP_INTERLEAVE_NONE || sw != CU_TENSOR_MAP_SWIZZLE_NONE) return CUDA_ERROR_INVALID_VALUE;
    if (dtype != CU_TENSOR_MAP_DATA_TYPE_FLOAT32 && dtype != CU_TENSOR_MAP_DATA_TYPE_INT32) return CUDA_ERROR_INVALID_VALUE;
    if (reinterpret_cast<uintptr_t>(m) & 63) return CUDA_ERROR_INVALID_VALUE;
    if (reinterpret_cast<uintptr_t>(base) & 15) return CUDA_ERROR_INVALID_VALUE;
    for (int i = 0; i < 3; ++i) {
        if (!dims[i] || dims[i] > (1ull << 32)) return CUDA_ERROR_INVALID_VALUE;
        if (!box[i] || box[i] > 256 || estr[i] != 1) return CUDA_ERROR_INVALID_VALUE;
    }
    for (int i = 0; i < 2; ++i)
        if (!strides[i] || (strides[i] & 15) || strides[i] >= (1ull << 40)) return CUDA_ERROR_INVALID_VALUE;
    if ((box[0] * 4) & 15) return CUDA_ERROR_INVALID_VALUE;
    MapRec r;
    r.magic = MAP_MAGIC; r.base = static_cast<unsigned char *>(base); r.dtype = dtype;
    for (int i = 0; i < 3; ++i) { r.dims[i] = dims[i]; r.box[i] = box[i]; }
    r.strides[0] = strides[0]; r.strides[1] = strides[1];
    std::memset(m, 0, sizeof(*m));
    std::memcpy(m, &r, sizeof r);
    return CUDA_SUCCESS;
}

static MapRec map_rec(const CUtensorMap *map, const char *what) {
    if (reinterpret_cast<uintptr_t>(map) & 63) fail("%s: the tensor map is not 64-byte aligned", what);
    MapRec r;
    std::memcpy(&r, map, sizeof r);
    if (r.magic != MAP_MAGIC) fail("%s: not an encoded tensor map", what);
    return r;
}
static inline size_t box_bytes(const MapRec &r) { return (size_t)r.box[0] * r.box[1] * r.box[2] * 4; }

static void perform_load(const PendingLoad &l) {
    const MapRec r = map_rec(&l.map, "cp.async.bulk.tensor (load)");
    uint32_t *dst = static_cast<uint32_t *>(shared_ptr_of(l.dst, box_bytes(r), "cp.async.bulk.tensor destination"));
    for (uint32_t z = 0; z < r.box[2]; ++z)
        for (uint32_t y = 0; y < r.box[1]; ++y)
            for (uint32_t x = 0; x < r.box[0]; ++x) {
                const long long gx = (long long)l.c[0] + x, gy = (long long)l.c[1] + y, gz = (long long)l.c[2] + z;
                uint32_t v = 0;                        // out-of-range elements are zero-filled
                if (gx >= 0 && gy >= 0 && gz >= 0 && gx < (long long)r.dims[0] && gy < (long long)r.dims[1] && gz < (long long)r.dims[2])
                    v = *reinterpret_cast<const uint32_t *>(r.base + gz * r.strides[1] + gy * r.strides[0] + gx * 4);
                dst[((size_t)z * r.box[1] + y) * r.box[0] + x] = v;
            }
    MBar *b = bar_at(l.bar);
    b->tx -= (int32_t)box_bytes(r);
    bar_check(b);
}

void tma_load_3d(unsigned dst, const CUtensorMap *map, int c0, int c1, int c2, unsigned bar) {
    const MapRec r = map_rec(map, "cp.async.bulk.tensor (load)");
    if (dst & 127) fail("cp.async.bulk.tensor: shared destination 0x%x is not 128-byte aligned", dst);
    (void)shared_ptr_of(dst, box_bytes(r), "cp.async.bulk.tensor destination");
    MBar *b = bar_at(bar);
    if (b->armed != 0xA5) fail("cp.async.bulk.tensor: completes on an mbarrier that was never initialised");
    // SHIM_ALLOW_TX_MISMATCH=1: let the mismatch through, so that a test can watch the kernel's own bounded wait expire
    if (b->tx != (int32_t)box_bytes(r) && !getenv("SHIM_ALLOW_TX_MISMATCH"))
        fail("cp.async.bulk.tensor: the barrier expects %d bytes but the box holds %zu (the wait would hang)", b->tx, box_bytes(r));
    PendingLoad l;
    l.map = *map; l.c[0] = c0; l.c[1] = c1; l.c[2] = c2; l.dst = dst; l.bar = bar;
    if (g_lazy) tw->loads.push_back(l);
    else perform_load(l);
}

static void perform_reduce(const BulkOp &op) {
    const MapRec r = map_rec(&op.map, "cp.reduce.async.bulk.tensor");
    const uint32_t *src = static_cast<const uint32_t *>(shared_ptr_of(op.src, box_bytes(r), "cp.reduce.async.bulk.tensor source"));
    for (uint32_t z = 0; z < r.box[2]; ++z)
        for (uint32_t y = 0; y < r.box[1]; ++y)
            for (uint32_t x = 0; x < r.box[0]; ++x) {
                const long long gx = (long long)op.c[0] + x, gy = (long long)op.c[1] + y, gz = (long long)op.c[2] + z;
                if (gx >= (long long)r.dims[0] || gy >= (long long)r.dims[1] || gz >= (long long)r.dims[2]) continue;   // skipped
                unsigned char *g = r.base + gz * r.strides[1] + gy * r.strides[0] + gx * 4;
                const uint32_t v = src[((size_t)z * r.box[1] + y) * r.box[0] + x];
                if (r.dtype == CU_TENSOR_MAP_DATA_TYPE_INT32) __atomic_fetch_add(reinterpret_cast<int *>(g), (int)v, __ATOMIC_RELAXED);
                else { float f; std::memcpy(&f, &v, 4); atomicAdd(reinterpret_cast<float *>(g), f); }
            }
}

void tma_reduce_add_3d(const CUtensorMap *map, int c0, int c1, int c2, unsigned src) {
    const MapRec r = map_rec(map, "cp.reduce.async.bulk.tensor");
    if (src & 127) fail("cp.reduce.async.bulk.tensor: shared source 0x%x is not 128-byte aligned", src);
    if (c0 < 0 || c1 < 0 || c2 < 0) fail("cp.reduce.async.bulk.tensor: negative start coordinate (%d, %d, %d)", c0, c1, c2);
    (void)shared_ptr_of(src, box_bytes(r), "cp.reduce.async.bulk.tensor source");
    BulkOp op;
    op.map = *map; op.c[0] = c0; op.c[1] = c1; op.c[2] = c2; op.src = src;
    if (g_lazy) me().open_group.push_back(op);
    else perform_reduce(op);
}
void bulk_commit() {
    Fiber &f = me();
    if (!f.open_group.empty()) { f.groups.push_back(f.open_group); f.open_group.clear(); }
}
void bulk_wait(int pending_allowed, bool) {
    Fiber &f = me();
    while ((int)f.groups.size() > pending_allowed) {
        for (const BulkOp &op : f.groups.front()) perform_reduce(op);
        f.groups.erase(f.groups.begin());
    }
}

}  // namespace shim

cudaError_t cudaFuncSetAttribute(const void *func, cudaFuncAttribute, int value) {
    if (value > (int)shim::DYN_MAX) return cudaErrorInvalidValue;
    std::lock_guard<std::mutex> lk(shim::g_attr_mu);
    shim::g_max_dyn[func] = value;
    return cudaSuccess;
}
cudaError_t cudaGetDriverEntryPoint(const char *symbol, void **fn, int, cudaDriverEntryPointQueryResult *q) {
    if (!strcmp(symbol, "cuTensorMapEncodeTiled")) {
        *fn = reinterpret_cast<void *>(&shim::encode_tiled);
        if (q) *q = cudaDriverEntryPointSuccess;
        return cudaSuccess;
    }
    *fn = nullptr;
    if (q) *q = cudaDriverEntryPointSymbolNotFound;
    return cudaSuccess;
}

// ---- C entry points for the Python test helper -------------------------------------------------------------------------------
extern "C" {
void *shim_malloc(size_t bytes) { return shim::dev_malloc(bytes); }
void shim_free(void *p) { shim::dev_free(p); }
const char *shim_last_error(void) {                     // "" when every launch so far obeyed the rules
    static thread_local std::string copy;
    std::lock_guard<std::mutex> lk(shim::g_err_mu);
    copy = shim::g_error;
    return copy.c_str();
}
const char *shim_kernel_log(int clear) {               // what was launched since the last clear
    static thread_local std::string copy;
    std::lock_guard<std::mutex> lk(shim::g_attr_mu);
    copy = shim::g_kernel_log;
    if (clear) shim::g_kernel_log.clear();
    return copy.c_str();
}
void shim_bank_stats_enable(int on, long long block_stride) {   // block_stride > 1: run every n-th block only (statistics, not results)
    shim::g_bank_on = on != 0;
    shim::g_block_stride = block_stride > 1 ? block_stride : 1;
    std::lock_guard<std::mutex> lk(shim::g_bank_mu);
    for (double &v : shim::g_bank_tot) v = 0;
}
void shim_bank_stats(double out[4]) {                   // {ld.shared instr, wavefronts, red.shared instr, wavefronts} per warp
    std::lock_guard<std::mutex> lk(shim::g_bank_mu);
    for (int k = 0; k < 4; ++k) out[k] = shim::g_bank_tot[k];
}
void shim_clear_error(void) {
    std::lock_guard<std::mutex> lk(shim::g_err_mu);
    shim::g_error.clear();
    shim::g_failed = false;
}
}
