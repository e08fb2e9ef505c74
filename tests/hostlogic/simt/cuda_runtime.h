// tests/hostlogic/simt/cuda_runtime.h -- TEST INFRASTRUCTURE, not product code.
//
// A small SIMT emulator that lets g++ compile a .cu file of paper_1901_02492_b200/csrc and run its
// kernels on the CPU, so that the device-side LOGIC of a kernel (indices, barrier phases, queue and
// ring bookkeeping, warp collectives) can be checked against the oracle without a GPU.  This file
// stands in for <cuda_runtime.h> when the test build puts this directory first on the include
// path.  What it models:
//   * every CUDA thread of a CTA is a fiber (ucontext) on one OS thread; CTAs run one after the
//     other.  A fiber runs until it blocks (a warp collective, __syncthreads, a failed mbarrier
//     poll); the scheduler then resumes another one, in an order chosen by simt::cfg().order
//     (forward, reverse, pseudo-random), so lanes of a warp are NOT in lockstep between
//     collectives -- code that needs __syncwarp for memory ordering and omits it fails here;
//   * shared memory is one byte array addressed by 32-bit offsets, bounds-checked and filled
//     with 0xFF (NaN patterns) at CTA start; mbarriers (init / arrive / expect_tx / complete_tx /
//     try_wait.parity) and tiled 3-D TMA loads with zero fill (simt_ptx.h), whose completion is
//     delayed by a configurable number of scheduler steps to model asynchrony;
//   * the handful of runtime calls the launch code makes (memcpy/memset on "streams", attribute
//     queries, the driver entry point for cuTensorMapEncodeTiled).
// What it does not model: memory-ordering subtleties between proxies, instruction-level hardware
// faults (e.g. alignment rules are asserted here only where this file knows them), performance.
#pragma once
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <ucontext.h>

#include <functional>
#include <map>
#include <vector>

#define KBMOD_SIMT_EMUL_ACTIVE 1

// AddressSanitizer build (tests/test_simt_sanitized.py): the part of the CTA's shared-memory array
// beyond the launch's dynamic size is poisoned while the CTA runs, so that a plain-pointer access
// past the size the launch asked for traps exactly as one past a heap block does.
#if defined(__SANITIZE_ADDRESS__)
#include <sanitizer/asan_interface.h>
#define SIMT_ASAN_POISON(p, n) ASAN_POISON_MEMORY_REGION((p), (n))
#define SIMT_ASAN_UNPOISON(p, n) ASAN_UNPOISON_MEMORY_REGION((p), (n))
#else
#define SIMT_ASAN_POISON(p, n) ((void)0)
#define SIMT_ASAN_UNPOISON(p, n) ((void)0)
#endif

// ---- keywords
#define __global__
#define __device__
#define __host__
#define __forceinline__ inline
#define __launch_bounds__(...)
#define __grid_constant__
#define __shared__
#define __align__(n)

// ---- vector types
// CUDA's alignment (8 / 16 bytes): a vector load or store through a misaligned pointer is a
// "misaligned address" fault on the GPU (Xid 13); with these attributes UBSan's alignment check
// reports it in the sanitized build (tests/test_simt_sanitized.py)
struct alignas(8) float2 { float x, y; };
struct alignas(16) float4 { float x, y, z, w; };
struct alignas(16) int4 { int x, y, z, w; };
struct uint3 { unsigned x, y, z; };
struct dim3 {
    unsigned x, y, z;
    dim3(unsigned x_ = 1, unsigned y_ = 1, unsigned z_ = 1) : x(x_), y(y_), z(z_) {}
};
static inline float2 make_float2(float x, float y) { return float2{x, y}; }
static inline float4 make_float4(float x, float y, float z, float w) { return float4{x, y, z, w}; }

// ---- runtime API subset
typedef void* cudaStream_t;
typedef int cudaError_t;
enum { cudaSuccess = 0 };
enum cudaMemcpyKind { cudaMemcpyHostToDevice = 1, cudaMemcpyDeviceToHost = 2, cudaMemcpyDeviceToDevice = 3 };
enum cudaFuncAttribute { cudaFuncAttributeMaxDynamicSharedMemorySize = 8 };
enum cudaDeviceAttr { cudaDevAttrMultiProcessorCount = 16 };
enum cudaDriverEntryPointQueryResult { cudaDriverEntryPointSuccess = 0 };
enum { cudaEnableDefault = 0 };

// ---- fiber context switch: hand-written on x86-64 (swapcontext makes a sigprocmask system call per
// switch, which dominates the run time), ucontext elsewhere
#if defined(__x86_64__)
extern "C" void simt_switch(void** save_sp, void* load_sp);
asm(".text\n.weak simt_switch\n.type simt_switch,@function\nsimt_switch:\n"
    "pushq %rbp\npushq %rbx\npushq %r12\npushq %r13\npushq %r14\npushq %r15\n"
    "movq %rsp, (%rdi)\nmovq %rsi, %rsp\n"
    "popq %r15\npopq %r14\npopq %r13\npopq %r12\npopq %rbx\npopq %rbp\nret\n"
    ".size simt_switch, .-simt_switch\n");
namespace simt {
struct Context { void* sp = nullptr; };
inline void ctx_switch(Context& from, Context& to) { simt_switch(&from.sp, to.sp); }
inline void ctx_make(Context& c, char* stack, size_t bytes, void (*entry)()) {
    uintptr_t top = ((uintptr_t)stack + bytes) & ~(uintptr_t)15;
    void** sp = reinterpret_cast<void**>(top);
    *--sp = nullptr;                       // keeps rsp = 8 (mod 16) at entry, as after a call
    *--sp = reinterpret_cast<void*>(entry);
    for (int k = 0; k < 6; ++k) *--sp = nullptr;
    c.sp = sp;
}
}  // namespace simt
#else
namespace simt {
struct Context { ucontext_t uc; };
inline void ctx_switch(Context& from, Context& to) { swapcontext(&from.uc, &to.uc); }
inline void ctx_make(Context& c, char* stack, size_t bytes, void (*entry)()) {
    getcontext(&c.uc);
    c.uc.uc_stack.ss_sp = stack;
    c.uc.uc_stack.ss_size = bytes;
    c.uc.uc_link = nullptr;
    makecontext(&c.uc, entry, 0);
}
}  // namespace simt
#endif

namespace simt {

constexpr unsigned FULL = 0xFFFFFFFFu;
constexpr size_t STACK_BYTES = 512 * 1024;
constexpr size_t SMEM_MAX = 227 * 1024;
constexpr unsigned SMEM_BASE = 0x400;          // shared-window offset of byte 0 (catches null addresses)

struct Config {
    int order = 0;          // 0 forward, 1 reverse, 2 pseudo-random (seeded)
    unsigned seed = 1;
    int sms = 3;            // cudaDevAttrMultiProcessorCount reported to the launch code
    int tma_delay = 0;      // a TMA load completes after up to this many scheduler steps
    long long clock_step = 1ll << 22;   // clock64() advances a fiber's clock by this much per call
};
inline Config& cfg() { static Config c; return c; }

struct MBar { int expected = 0, pending = 0; long long tx = 0; unsigned phase = 0; bool init = false; };

struct Fiber {
    Context ctx;
    char* stack = nullptr;
    bool done = false;
    uint3 tid{0, 0, 0};
    unsigned wgen = 0;      // warp-collective generation of this lane
    unsigned bgen = 0;      // __syncthreads generation
    long long clock = 0;    // this thread's clock64()
    const char* where = "";  // what the fiber last blocked on (deadlock report)
    unsigned where_a = 0, where_b = 0;
};

struct WarpSlot { unsigned gen[2] = {~0u, ~0u}; unsigned arrived[2] = {0, 0}; unsigned long long vals[2][32]; };

struct PendingTma { int due; std::function<void()> fn; };

struct State {
    std::vector<Fiber> fibers;
    std::vector<WarpSlot> warps;
    std::vector<char*> stacks;
    unsigned char* smem = nullptr;      // the CTA's shared memory: set by the test driver (SMEM_MAX + 64 bytes)
    size_t smem_size = 0;               // dynamic shared memory of the running launch
    std::map<unsigned, MBar> bars;
    std::vector<PendingTma> tma;
    Context sched;
    Fiber* cur = nullptr;
    uint3 bid{0, 0, 0};
    dim3 gdim, bdim;
    unsigned bar_count = 0, bar_gen = 0;
    long long steps = 0;
    unsigned rng = 1;
    std::function<void()> body;
    // statistics / faults
    long long smem_faults = 0, launches = 0, tma_loads = 0, tma_faults = 0;
};
inline State& S() { static State s; return s; }

[[noreturn]] inline void fatal(const char* what) {
    fprintf(stderr, "simt: fatal: %s\n", what);
    abort();
}

inline void yield() { State& s = S(); ctx_switch(s.cur->ctx, s.sched); }

inline void fiber_main() {
    State& s = S();
    s.body();
    s.cur->done = true;
    ctx_switch(s.cur->ctx, s.sched);
    fatal("finished fiber resumed");
}

inline unsigned next_rand() { State& s = S(); s.rng = s.rng * 1664525u + 1013904223u; return s.rng >> 8; }

inline void run_due_tma(bool force) {
    State& s = S();
    for (size_t k = 0; k < s.tma.size();) {
        if (force || --s.tma[k].due <= 0) {
            auto fn = std::move(s.tma[k].fn);
            s.tma.erase(s.tma.begin() + k);
            fn();
        } else {
            ++k;
        }
    }
}

// Runs one CTA to completion.  Returns false if the CTA deadlocked (no fiber can make progress
// and nothing is pending); the kernels under test bound their own waits, so this is a test failure.
inline bool run_cta(unsigned nthreads, size_t smem_bytes) {
    State& s = S();
    if (!s.smem || smem_bytes > SMEM_MAX) fatal("shared memory not set up or launch asks for more than 227 KB");
    s.smem_size = smem_bytes;
    SIMT_ASAN_UNPOISON(s.smem, SMEM_MAX + 64);
    memset(s.smem, 0xFF, SMEM_MAX + 64);
    // the scratch tail [SMEM_MAX, SMEM_MAX + 64) stays addressable: smem_ptr() redirects a faulting
    // access there and counts it, which the tests assert on
    SIMT_ASAN_POISON(s.smem + smem_bytes, SMEM_MAX - smem_bytes);
    s.bars.clear();
    s.tma.clear();
    s.bar_count = 0;
    s.bar_gen = 0;
    s.fibers.assign(nthreads, Fiber());
    s.warps.assign((nthreads + 31) / 32, WarpSlot());
    for (unsigned t = 0; t < nthreads; ++t) {
        Fiber& f = s.fibers[t];
        if (s.stacks.size() <= t) s.stacks.push_back(static_cast<char*>(malloc(STACK_BYTES)));
        f.stack = s.stacks[t];           // stacks are pooled across CTAs and launches
        f.tid = uint3{t % s.bdim.x, t / s.bdim.x, 0};
        ctx_make(f.ctx, f.stack, STACK_BYTES, fiber_main);
    }
    unsigned live = nthreads;
    std::vector<unsigned> order(nthreads);
    long long idle_passes = 0;
    while (live > 0) {
        for (unsigned t = 0; t < nthreads; ++t) order[t] = cfg().order == 1 ? nthreads - 1 - t : t;
        if (cfg().order == 2)
            for (unsigned t = nthreads - 1; t > 0; --t) std::swap(order[t], order[next_rand() % (t + 1)]);
        const long long before = s.steps;
        for (unsigned k = 0; k < nthreads; ++k) {
            Fiber& f = s.fibers[order[k]];
            if (f.done) continue;
            s.cur = &f;
            ctx_switch(s.sched, f.ctx);
            if (f.done) { --live; ++s.steps; }
            run_due_tma(false);
        }
        if (s.steps == before) {
            if (!s.tma.empty()) { run_due_tma(true); continue; }
            if (++idle_passes > 8192) break;        // clock64() keeps advancing: bounded waits expire first
        } else {
            idle_passes = 0;
        }
    }
    if (live > 0 && getenv("SIMT_DEBUG")) {
        for (unsigned t = 0; t < nthreads; t += 1) {
            const Fiber& f = s.fibers[t];
            if (!f.done && ((t & 31) == 0 || f.where_a != s.fibers[t & ~31u].where_a || f.where != s.fibers[t & ~31u].where))
                fprintf(stderr, "simt: cta %u thread %u blocked in %s (%u, %u) wgen %u\n", s.bid.x, t, f.where, f.where_a - SMEM_BASE, f.where_b, f.wgen);
        }
        for (auto& kv : s.bars)
            fprintf(stderr, "simt: mbarrier @%u expected %d pending %d tx %lld phase %u\n", kv.first - SMEM_BASE, kv.second.expected, kv.second.pending, kv.second.tx, kv.second.phase);
    }
    s.fibers.clear();
    SIMT_ASAN_UNPOISON(s.smem, SMEM_MAX + 64);
    return live == 0;
}

inline dim3 as_dim3(dim3 d) { return d; }
inline dim3 as_dim3(unsigned v) { return dim3(v); }
inline dim3 as_dim3(int v) { return dim3((unsigned)v); }
inline dim3 as_dim3(long long v) { return dim3((unsigned)v); }

// grids and blocks of up to two dimensions (threadIdx.x fastest, as on the device)
template <class Kern, class... Args>
inline void launch(Kern kern, dim3 grid, dim3 block, size_t smem_bytes, Args... args) {
    State& s = S();
    if (grid.z != 1 || block.z != 1) fatal("3-D launches are not modelled");
    ++s.launches;
    s.gdim = grid;
    s.bdim = block;
    s.rng = cfg().seed;
    for (unsigned by = 0; by < grid.y; ++by)
        for (unsigned bx = 0; bx < grid.x; ++bx) {
            s.bid = uint3{bx, by, 0};
            s.body = [&]() { kern(args...); };
            if (!run_cta(block.x * block.y, smem_bytes)) fatal("CTA deadlocked");
        }
}

// ---- shared memory access (32-bit shared-window addresses)
inline unsigned char* smem_ptr(unsigned a, unsigned bytes, unsigned align) {
    State& s = S();
    const unsigned off = a - SMEM_BASE;
    if (a < SMEM_BASE || (size_t)off + bytes > s.smem_size || (a & (align - 1))) {
        ++s.smem_faults;
        return s.smem + SMEM_MAX;                       // scratch tail: keep running, report later
    }
    return s.smem + off;
}

// ---- warp collectives: every lane deposits a value; all lanes see all values
inline const unsigned long long* warp_exchange(unsigned mask, unsigned long long v) {
    if (mask != FULL) fatal("warp collective with a partial mask (not modelled)");
    State& s = S();
    Fiber* f = s.cur;
    const unsigned t = (unsigned)(f - s.fibers.data());
    WarpSlot& w = s.warps[t >> 5];
    const unsigned lane = t & 31, g = f->wgen++, sl = g & 1;
    if (w.gen[sl] != g) { w.gen[sl] = g; w.arrived[sl] = 0; }
    w.vals[sl][lane] = v;
    w.arrived[sl] |= 1u << lane;
    ++s.steps;
    f->where = "warp collective"; f->where_a = SMEM_BASE; f->where_b = g;
    while (!(w.gen[sl] == g && w.arrived[sl] == FULL)) yield();
    return w.vals[sl];
}

}  // namespace simt

#define threadIdx (::simt::S().cur->tid)
#define blockIdx (::simt::S().bid)
#define gridDim (::simt::S().gdim)
#define blockDim (::simt::S().bdim)

// ---- intrinsics
template <class T> static inline T __ldg(const T* p) { return *p; }
template <class T> static inline T __ldcg(const T* p) { return *p; }
template <class T> static inline void __stcg(T* p, T v) { *p = v; }
static inline float __fadd_rn(float a, float b) { volatile float r = a + b; return r; }
static inline float __fsub_rn(float a, float b) { volatile float r = a - b; return r; }
static inline float __fmul_rn(float a, float b) { volatile float r = a * b; return r; }
static inline float __fdiv_rn(float a, float b) { volatile float r = a / b; return r; }
static inline float __fsqrt_rn(float a) { return sqrtf(a); }
static inline float __int2float_rn(int a) { return (float)a; }
static inline float rsqrtf(float a) { return 1.0f / sqrtf(a); }
static inline float2 __fadd2_rn(float2 a, float2 b) { return float2{__fadd_rn(a.x, b.x), __fadd_rn(a.y, b.y)}; }
static inline float __uint_as_float(unsigned u) { float f; memcpy(&f, &u, 4); return f; }
static inline unsigned __float_as_uint(float f) { unsigned u; memcpy(&u, &f, 4); return u; }
static inline float __int_as_float(int u) { float f; memcpy(&f, &u, 4); return f; }
static inline int __float_as_int(float f) { int u; memcpy(&u, &f, 4); return u; }
static inline int __popc(unsigned v) { return __builtin_popcount(v); }
static inline int __ffs(unsigned v) { return __builtin_ffs((int)v); }
static inline unsigned __funnelshift_l(unsigned lo, unsigned hi, unsigned sh) {
    sh &= 31;
    return sh ? (hi << sh) | (lo >> (32 - sh)) : hi;
}
static inline int min(int a, int b) { return a < b ? a : b; }
static inline unsigned min(unsigned a, unsigned b) { return a < b ? a : b; }
static inline int max(int a, int b) { return a > b ? a : b; }
static inline long long clock64() { return ::simt::S().cur->clock += ::simt::cfg().clock_step; }
static inline int atomicExch(int* p, int v) { const int o = *p; *p = v; return o; }
// fibers never pre-empt one another inside a plain statement, so read-modify-write is atomic here
static inline unsigned long long atomicAdd(unsigned long long* p, unsigned long long v) {
    const unsigned long long o = *p;
    *p = o + v;
    return o;
}

static inline void __syncwarp(unsigned mask = ::simt::FULL) { ::simt::warp_exchange(mask, 0); }
static inline unsigned __ballot_sync(unsigned mask, int pred) {
    const unsigned long long* v = ::simt::warp_exchange(mask, pred ? 1 : 0);
    unsigned r = 0;
    for (int l = 0; l < 32; ++l) r |= v[l] ? (1u << l) : 0u;
    return r;
}
static inline int __all_sync(unsigned mask, int pred) { return __ballot_sync(mask, pred) == ::simt::FULL; }
static inline int __any_sync(unsigned mask, int pred) { return __ballot_sync(mask, pred) != 0; }
static inline int __shfl_sync(unsigned mask, int v, int src) {
    return (int)(unsigned)::simt::warp_exchange(mask, (unsigned)v)[src & 31];
}
static inline unsigned __match_any_sync(unsigned mask, int v) {
    const unsigned long long* a = ::simt::warp_exchange(mask, (unsigned)v);
    const unsigned lane = (unsigned)(::simt::S().cur - ::simt::S().fibers.data()) & 31;
    unsigned r = 0;
    for (int l = 0; l < 32; ++l) r |= (a[l] == a[lane]) ? (1u << l) : 0u;
    return r;
}
static inline void __syncthreads() {
    ::simt::State& s = ::simt::S();
    ::simt::Fiber* f = s.cur;
    const unsigned g = f->bgen++;
    unsigned nthreads = s.bdim.x * s.bdim.y * s.bdim.z;
    if (++s.bar_count == nthreads) { s.bar_count = 0; ++s.bar_gen; }
    ++s.steps;
    while (s.bar_gen <= g) ::simt::yield();
}

// ---- runtime calls used by the launch code ("device" memory is host memory)
static inline cudaError_t cudaMemcpyAsync(void* d, const void* s, size_t n, cudaMemcpyKind, cudaStream_t) {
    memcpy(d, s, n);
    return cudaSuccess;
}
static inline cudaError_t cudaMemsetAsync(void* d, int v, size_t n, cudaStream_t) { memset(d, v, n); return cudaSuccess; }
static inline cudaError_t cudaGetLastError() { return cudaSuccess; }
static inline cudaError_t cudaStreamSynchronize(cudaStream_t) { return cudaSuccess; }
template <class F> static inline cudaError_t cudaFuncSetAttribute(F, cudaFuncAttribute, int) { return cudaSuccess; }
static inline cudaError_t cudaGetDevice(int* d) { *d = 0; return cudaSuccess; }
static inline cudaError_t cudaDeviceGetAttribute(int* v, cudaDeviceAttr, int) { *v = ::simt::cfg().sms; return cudaSuccess; }
static inline cudaError_t cudaGetDeviceCount(int* n) { *n = 1; return cudaSuccess; }
cudaError_t cudaGetDriverEntryPoint(const char* name, void** fn, int flags, cudaDriverEntryPointQueryResult* qr);
