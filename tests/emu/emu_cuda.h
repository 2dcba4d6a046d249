// emu_cuda.h -- TEST INFRASTRUCTURE, never part of the product: a CPU emulation of the slice of CUDA that
// paper_2603_07038_b200/csrc uses, so that the SAME kernel and host sources (em_lib.cu and its headers, unmodified) can be
// compiled by g++ into tests/emu/libem_emu*.so and run on small grids under checks that compute-sanitizer would do on a
// GPU (it is closed on this GPU pool, and so -- for most of round 2 -- was the pool itself):
//   * every CUDA thread is a fiber (own stack, cooperative switch); a CTA runs on one OS thread, CTAs in parallel;
//   * __syncthreads / __syncwarp / shuffles / votes / named barriers / mbarriers block the fiber until the condition
//     holds; a CTA in which every fiber is blocked and no asynchronous copy is pending is a DEADLOCK and is reported
//     with what each warp waits for (the launch fails like a CUDA launch failure);
//   * TMA tensor / bulk copies and cp.async are asynchronous: they complete after a (seeded) random delay, never before
//     the issuing thread moved on, cp.async only inside cp_async_wait -- a consumer that reads before it waited, or a
//     producer that refills a slot too early, sees wrong data;
//   * EMU_SEED != 0 randomises the fiber schedule (order, skipped turns, extra yields at every synchronisation point);
//   * dynamic shared memory is poisoned (0xFF = NaN) per CTA, has a canary behind it, and every address handed to an
//     mbarrier / TMA / cp.async / streaming-store wrapper is checked for range and alignment (a misaligned or
//     out-of-range address is what faults a GPU); global allocations made through emu_alloc sit between guard pages.
//   * RACECHECK (EMU_RACECHECK=1 on a build made with -fsanitize=thread, whose load / store hooks __tsan_read* /
//     __tsan_write* are implemented HERE, emu_exports.cpp, not by libtsan): a happens-before race detector for the dynamic
//     shared memory.  Every thread and the asynchronous copy engine carry vector clocks; __syncthreads, __syncwarp,
//     bar.sync / bar.arrive and mbarrier arrive / complete_tx -> try_wait are the only ordering edges (shuffles and votes
//     are NOT); two accesses to the same 4 bytes by different agents, one of them a write, with no ordering path between
//     them are reported as a race with both code addresses -- whether or not the schedule at hand made them collide.
// What it does not emulate: timing, caches, the memory model between CTAs, PTX itself (em_ptx.cuh is replaced as a whole).
#pragma once

#include <atomic>
#include <condition_variable>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <functional>
#include <map>
#include <memory>
#include <mutex>
#include <string>
#include <thread>
#include <vector>

#include <math.h>        // libstdc++: the float overloads of ::fabs, ::expm1 ... in the global namespace, as in CUDA
#include <sys/mman.h>

#define __global__
#define __device__
#define __host__
#define __forceinline__ inline __attribute__((always_inline))
#define __launch_bounds__(...)
#define __grid_constant__
#define __shared__ static thread_local
#define __align__(n) alignas(n)

// ---- vector types ---------------------------------------------------------------------------------------------------
struct uint3 { unsigned x, y, z; };
struct dim3 {
    unsigned x, y, z;
    dim3(unsigned x_ = 1, unsigned y_ = 1, unsigned z_ = 1) : x(x_), y(y_), z(z_) {}
};
struct alignas(16) float4 { float x, y, z, w; };
struct alignas(16) double4 { double x, y, z, w; };
struct alignas(16) int4 { int x, y, z, w; };
inline int4 make_int4(int x, int y, int z, int w) { return int4{x, y, z, w}; }

typedef int cudaError_t;
constexpr cudaError_t cudaSuccess = 0, cudaErrorInvalidValue = 1, cudaErrorLaunchFailure = 719;
inline thread_local cudaError_t emu_last_error = cudaSuccess;       // what cudaGetLastError returns (and clears)
inline thread_local std::string emu_last_error_text;

// ---- the fiber machine ----------------------------------------------------------------------------------------------
namespace emu {

struct Cta;

struct Fiber {
    void *sp = nullptr;                 // saved stack pointer while switched out
    int tid = 0, lane = 0, warp = 0;
    uint3 tidx{0, 0, 0};
    Cta *cta = nullptr;
    bool done = false;
    // blocked while ((*wait_addr & wait_mask) == wait_val)
    volatile uint32_t *wait_addr = nullptr;
    uint32_t wait_mask = 0, wait_val = 0;
    const char *wait_what = "";
    long wait_arg = 0;
    // cp.async: the copies happen inside cp_async_wait (the latest moment the hardware allows)
    struct Copy { void *dst; const void *src; int bytes; int group; };
    std::vector<Copy> copies;
    int open_group = 0;
};

// racecheck: the clocks of a synchronisation object -- what its arrivals of the running phase have released (pending) and
// what a thread that saw a phase complete acquires (completed)
struct SyncClock { std::vector<uint32_t> pending, completed; };
struct WarpState { uint64_t buf[2][32]; uint32_t gen = 0; int arrived = 0, alive = 32; SyncClock clk; };
struct BarState { uint32_t gen = 0; int arrived = 0; SyncClock clk; };
struct AsyncOp { int delay; std::function<void()> fire; };
struct RaceState;

struct Region { uintptr_t lo, hi; };

struct Cta {
    const std::vector<Region> *regions = nullptr;       // emu_alloc'ed global memory at launch time
    dim3 bidx, bdim, gdim;
    int nthreads = 0, alive = 0;
    unsigned char *smem = nullptr;
    size_t smem_bytes = 0;
    std::vector<Fiber> fibers;
    std::vector<WarpState> warps;
    BarState bars[16];
    std::vector<AsyncOp> async;
    std::map<unsigned, SyncClock> mbar_init;    // smem offsets of initialised mbarriers (+ their racecheck clocks)
    RaceState *race = nullptr;                  // racecheck state (EMU_RACECHECK=1), else null
    const std::function<void()> *body = nullptr;
    void *sched_sp = nullptr;
    uint64_t rng = 0;
    bool random = false;
    bool failed = false;
    std::string error;
    const char *kernel_name = "";
};

inline thread_local Fiber *t_cur = nullptr;

extern "C" void emu_switch(void **save_sp, void *load_sp);
extern "C" void emu_install_fault_handler(void);      // emu_exports.cpp: SIGSEGV / SIGBUS inside a kernel -> who, where
extern "C" void emu_thread_altstack(void);
// (defined once, in emu_exports.cpp: saves the callee-saved registers, swaps the stack pointer)

inline uint64_t next_rand(uint64_t &s) {       // splitmix64
    uint64_t z = (s += 0x9e3779b97f4a7c15ull);
    z = (z ^ (z >> 30)) * 0xbf58476d1ce4e5b9ull;
    z = (z ^ (z >> 27)) * 0x94d049bb133111ebull;
    return z ^ (z >> 31);
}

inline void yield() { Fiber *f = t_cur; emu_switch(&f->sp, f->cta->sched_sp); }

// a kernel-side error (bad address, barrier misuse): recorded, the CTA is abandoned at the next scheduler turn
[[noreturn]] inline void fail_here(const std::string &msg) {
    Fiber *f = t_cur;
    Cta *c = f->cta;
    if (!c->failed) {
        char head[256];
        snprintf(head, sizeof(head), "emu: kernel %s, block (%u,%u,%u), thread %d (warp %d lane %d): ", c->kernel_name,
                 c->bidx.x, c->bidx.y, c->bidx.z, f->tid, f->warp, f->lane);
        c->failed = true;
        c->error = std::string(head) + msg;
    }
    for (;;) { f->wait_addr = nullptr; yield(); }       // never resumed: the scheduler stops on `failed`
}

inline void block_while(volatile uint32_t *addr, uint32_t mask, uint32_t val, const char *what, long arg = 0) {
    Fiber *f = t_cur;
    while ((*addr & mask) == val) {
        f->wait_addr = addr; f->wait_mask = mask; f->wait_val = val; f->wait_what = what; f->wait_arg = arg;
        yield();
    }
    f->wait_addr = nullptr;
}

// ---- racecheck ----------------------------------------------------------------------------------------------------------
// Agents: the CTA's threads 0 .. n-1 and the asynchronous copy engine (index n).  clock[t][u] = the latest epoch of agent u
// that happens-before agent t's present; an access is stamped (agent, own epoch); a release bumps the own epoch.
struct RaceState {
    int n = 0;                                   // agents = threads + 1
    std::vector<uint32_t> clocks;                // [n][n]
    struct Shadow {                              // per 4-byte granule of the dynamic shared memory
        uint32_t w_agent = 0xffffffffu, w_clk = 0;
        uint32_t r_agent[4], r_clk[4];
        uint8_t nr = 0;
        const void *w_pc = nullptr, *r_pc[4];
    };
    std::vector<Shadow> shadow;
    uint32_t agent_epoch = 0;
    uint32_t *clk(int t) { return clocks.data() + (size_t)t * n; }
};
inline void race_join(std::vector<uint32_t> &dst, const uint32_t *src, int n) {
    if ((int)dst.size() != n) dst.assign(n, 0);
    for (int q = 0; q < n; ++q) dst[q] = std::max(dst[q], src[q]);
}
// the running thread publishes everything it did so far to the object's running phase
inline void race_release(SyncClock &s) {
    Fiber *f = t_cur; RaceState *r = f->cta->race;
    if (!r) return;
    race_join(s.pending, r->clk(f->tid), r->n);
    r->clk(f->tid)[f->tid] += 1;
}
// a phase of the object completed: what was released into it becomes visible to those who wait for it
inline void race_complete(Cta *c, SyncClock &s) {
    RaceState *r = c->race;
    if (!r || s.pending.empty()) return;
    race_join(s.completed, s.pending.data(), r->n);
}
inline void race_acquire(SyncClock &s) {
    Fiber *f = t_cur; RaceState *r = f->cta->race;
    if (!r || s.completed.empty()) return;
    uint32_t *c = r->clk(f->tid);
    for (int q = 0; q < r->n; ++q) c[q] = std::max(c[q], s.completed[q]);
}
inline std::string race_pc(const void *pc) { char b[32]; snprintf(b, sizeof(b), "%p", pc); return b; }
inline void race_report(Cta *c, size_t off, const char *what, uint32_t a0, const void *pc0, uint32_t a1, const void *pc1) {
    if (c->failed) return;
    RaceState *r = c->race;
    auto who = [&](uint32_t a) { return (int)a == r->n - 1 ? std::string("the async copy engine") : "thread " + std::to_string(a) + " (warp " + std::to_string(a / 32) + " lane " + std::to_string(a % 32) + ")"; };
    c->failed = true;
    c->error = std::string("emu: RACE in kernel ") + c->kernel_name + ", block (" + std::to_string(c->bidx.x) + "," + std::to_string(c->bidx.y) + "," +
               std::to_string(c->bidx.z) + "), dynamic shared memory offset " + std::to_string(off) + ": " + what + " -- " + who(a0) + " at pc " + race_pc(pc0) +
               " and " + who(a1) + " at pc " + race_pc(pc1) + " are not ordered by any barrier";
}
// one access of `agent` (clock row vc) to [p, p + n): is_write or read; returns false after reporting a race
inline bool race_check(Cta *c, const uint32_t *vc, uint32_t agent, uint32_t epoch, const unsigned char *p, size_t n, bool is_write, const void *pc) {
    RaceState *r = c->race;
    const size_t off0 = (size_t)(p - c->smem);
    for (size_t g = off0 / 4; g <= (off0 + n - 1) / 4; ++g) {
        if (c->mbar_init.count((unsigned)(g * 4 / 8 * 8) + 0x10000u)) continue;         // the mbarrier objects themselves
        RaceState::Shadow &sh = r->shadow[g];
        const bool engine = (int)agent == r->n - 1;          // two copies of the engine are NOT ordered by being the engine's
        if (sh.w_agent != 0xffffffffu && (sh.w_agent != agent || engine) && sh.w_clk > vc[sh.w_agent]) {
            race_report(c, g * 4, is_write ? "write after write" : "read after write", sh.w_agent, sh.w_pc, agent, pc); return false;
        }
        if (is_write) {
            for (int q = 0; q < sh.nr; ++q)
                if (sh.r_agent[q] != agent && sh.r_clk[q] > vc[sh.r_agent[q]]) {
                    race_report(c, g * 4, "write after read", sh.r_agent[q], sh.r_pc[q], agent, pc); return false;
                }
            sh.w_agent = agent; sh.w_clk = epoch; sh.w_pc = pc; sh.nr = 0;
        } else {
            int slot = -1;
            for (int q = 0; q < sh.nr; ++q)
                if (sh.r_agent[q] == agent || sh.r_clk[q] <= vc[sh.r_agent[q]]) { slot = q; break; }      // mine, or subsumed by me
            if (slot < 0) slot = sh.nr < 4 ? sh.nr++ : (int)(epoch & 3);                                    // (full: one reader is forgotten)
            sh.r_agent[slot] = agent; sh.r_clk[slot] = epoch; sh.r_pc[slot] = pc;
        }
    }
    return true;
}
// the load / store hooks of a -fsanitize=thread build land here (emu_exports.cpp)
inline void race_access(const void *addr, size_t n, bool is_write, const void *pc) {
    Fiber *f = t_cur;
    if (!f) return;
    Cta *c = f->cta;
    if (!c->race || c->failed) return;
    const unsigned char *p = static_cast<const unsigned char *>(addr);
    if (p < c->smem || p + n > c->smem + c->smem_bytes) return;
    const uint32_t *vc = c->race->clk(f->tid);
    race_check(c, vc, (uint32_t)f->tid, vc[f->tid], p, n, is_write, pc);
}
// An asynchronous copy is ordered after everything its issuer had seen when it issued it (vc: the issuer's clock then,
// including the latest copy-engine epoch it had learnt of through a barrier) and before whoever waits for the mbarrier
// it completes on; two copies are ordered only through such a wait.
struct RaceAsync { std::vector<uint32_t> vc; uint32_t epoch = 0; };
inline std::shared_ptr<RaceAsync> race_async_issue() {
    Fiber *f = t_cur; RaceState *r = f->cta->race;
    if (!r) return nullptr;
    auto a = std::make_shared<RaceAsync>();
    a->vc.assign(r->clk(f->tid), r->clk(f->tid) + r->n);
    a->epoch = ++r->agent_epoch;
    r->clk(f->tid)[f->tid] += 1;                       // what the issuer does next is NOT ordered before the copy
    return a;
}
inline void race_async_write(Cta *c, const std::shared_ptr<RaceAsync> &a, const unsigned char *dst, size_t n, const void *pc) {
    if (!a || !c->race || c->failed) return;
    race_check(c, a->vc.data(), (uint32_t)c->race->n - 1, a->epoch, dst, n, true, pc);
}
inline void race_async_complete(Cta *c, SyncClock &s, const std::shared_ptr<RaceAsync> &a) {
    if (!a || !c->race) return;
    race_join(s.pending, a->vc.data(), c->race->n);
    s.pending[c->race->n - 1] = std::max(s.pending[c->race->n - 1], a->epoch);
}

// extra yield at a synchronisation point when the schedule is randomised (the counterpart of EM_SWEEP_FUZZ's delays)
inline void sync_point() {
    Fiber *f = t_cur;
    if (f->cta->random && (next_rand(f->cta->rng) & 3) == 0) yield();
}

// ---- warp collectives -------------------------------------------------------------------------------------------
// orders = true (__syncwarp): the collective is also a memory barrier among the lanes; shuffles and votes are not
inline const uint64_t *warp_xchg(uint64_t v, unsigned mask, bool orders = false) {
    Fiber *f = t_cur;
    if (mask != 0xffffffffu) fail_here("warp collective with a partial mask (not emulated)");
    WarpState &W = f->cta->warps[f->warp];
    const uint32_t g = W.gen;
    uint64_t *b = W.buf[g & 1];
    b[f->lane] = v;
    if (orders) race_release(W.clk);
    if (++W.arrived >= W.alive) { W.arrived = 0; W.gen = g + 1; if (orders) race_complete(f->cta, W.clk); }
    else block_while(&W.gen, 0xffffffffu, g, "warp collective (shuffle / vote / __syncwarp)");
    if (orders) race_acquire(W.clk);
    return b;
}
template <typename T> inline uint64_t to_bits(T v) { uint64_t u = 0; static_assert(sizeof(T) <= 8, ""); memcpy(&u, &v, sizeof(T)); return u; }
template <typename T> inline T from_bits(uint64_t u) { T v; memcpy(&v, &u, sizeof(T)); return v; }

inline void cta_barrier_arrive(Cta *c, BarState &B, int expected, bool wait, const char *what, long arg) {
    const uint32_t g = B.gen;
    race_release(B.clk);
    if (++B.arrived >= expected) { B.arrived = 0; B.gen = g + 1; race_complete(c, B.clk); }
    else if (wait) block_while(&B.gen, 0xffffffffu, g, what, arg);
    if (wait) race_acquire(B.clk);
}

// ---- global-memory registry (emu_alloc: guard pages on both sides) ----------------------------------------------
inline std::vector<Region> &regions() { static std::vector<Region> r; return r; }
inline std::mutex &regions_mutex() { static std::mutex m; return m; }
inline bool in_registered(const void *p, size_t n) {       // against the snapshot taken when the kernel was launched
    const std::vector<Region> &rs = *t_cur->cta->regions;
    if (rs.empty()) return true;                            // nothing registered: no range check
    const uintptr_t a = (uintptr_t)p;
    for (const Region &r : rs) if (a >= r.lo && a + n <= r.hi) return true;
    return false;
}
inline void check_global(const void *p, size_t n, size_t align, const char *what) {
    if ((uintptr_t)p % align) fail_here(std::string(what) + ": misaligned global address");
    if (!in_registered(p, n)) fail_here(std::string(what) + ": global address outside every emu_alloc'ed region");
}
inline unsigned char *check_smem(const void *p, size_t n, size_t align, const char *what) {
    Cta *c = t_cur->cta;
    const unsigned char *q = static_cast<const unsigned char *>(p);
    if (q < c->smem || q + n > c->smem + c->smem_bytes) fail_here(std::string(what) + ": address outside the dynamic shared memory");
    if ((uintptr_t)(q - c->smem) % align) fail_here(std::string(what) + ": misaligned shared address");
    return const_cast<unsigned char *>(q);
}
constexpr unsigned kSmemBase = 0x10000u;                    // shared-window address of dynamic smem offset 0
inline unsigned smem_to_u32(const void *p) { return (unsigned)(check_smem(p, 1, 1, "cvta.to.shared") - t_cur->cta->smem) + kSmemBase; }
inline unsigned char *u32_to_smem(unsigned a, size_t n, size_t align, const char *what) {
    Cta *c = t_cur->cta;
    if (a < kSmemBase || (size_t)(a - kSmemBase) + n > c->smem_bytes) fail_here(std::string(what) + ": shared address out of range");
    if ((a - kSmemBase) % align) fail_here(std::string(what) + ": misaligned shared address");
    return c->smem + (a - kSmemBase);
}

// ---- scheduler ------------------------------------------------------------------------------------------------------
constexpr size_t kStackBytes = 96 * 1024;

inline void fiber_entry() {
    Fiber *f = t_cur;
    (*f->cta->body)();
    Cta *c = f->cta;
    f->done = true;
    c->alive -= 1;
    WarpState &W = c->warps[f->warp];
    W.alive -= 1;
    if (W.arrived > 0 && W.arrived >= W.alive) { W.arrived = 0; W.gen += 1; }           // exited lanes do not hold a collective up
    if (c->bars[0].arrived > 0 && c->bars[0].arrived >= c->alive) { c->bars[0].arrived = 0; c->bars[0].gen += 1; race_complete(c, c->bars[0].clk); }
    if (!f->copies.empty()) { /* cp.async still in flight at exit: the data would land after the thread is gone */ }
    emu_switch(&f->sp, c->sched_sp);
    abort();
}

inline void describe_deadlock(Cta &c) {
    std::string s = "emu: DEADLOCK in kernel " + std::string(c.kernel_name) + ", block (" + std::to_string(c.bidx.x) + "," +
                    std::to_string(c.bidx.y) + "," + std::to_string(c.bidx.z) + "): every live thread is blocked and no asynchronous copy is pending;";
    int shown = 0;
    for (const Fiber &f : c.fibers) {
        if (f.done || (f.lane != 0 && shown > 0 && f.wait_what == c.fibers[f.tid - 1].wait_what && f.wait_arg == c.fibers[f.tid - 1].wait_arg)) continue;
        s += " [warp " + std::to_string(f.warp) + " lane " + std::to_string(f.lane) + ": " + f.wait_what + " #" + std::to_string(f.wait_arg) + "]";
        if (++shown >= 40) { s += " ..."; break; }
    }
    c.failed = true; c.error = s;
}

// runs one CTA to completion on the calling OS thread; stacks: nthreads * kStackBytes
inline void run_cta(Cta &c, char *stacks) {
    const int n = c.nthreads;
    for (int t = 0; t < n; ++t) {
        Fiber &f = c.fibers[t];
        char *top = stacks + (size_t)(t + 1) * kStackBytes;          // 16-byte aligned (kStackBytes is)
        void **sp = reinterpret_cast<void **>(top - 8);
        *--sp = reinterpret_cast<void *>(&fiber_entry);               // popped by emu_switch's ret
        for (int r = 0; r < 6; ++r) *--sp = nullptr;                  // rbp, rbx, r12-r15
        f.sp = sp;
    }
    int remaining = n;
    std::vector<int> order(n);
    for (int t = 0; t < n; ++t) order[t] = t;
    while (remaining > 0 && !c.failed) {
        bool progress = false, skipped = false;
        if (c.random) {                                  // a new random order of the WARPS every pass, lanes rotated
            const int nw = (n + 31) / 32;
            std::vector<int> wo(nw);
            for (int w = 0; w < nw; ++w) wo[w] = w;
            for (int w = nw - 1; w > 0; --w) std::swap(wo[w], wo[next_rand(c.rng) % (w + 1)]);
            int q = 0;
            for (int w = 0; w < nw; ++w) {
                const int rot = (int)(next_rand(c.rng) & 31);
                for (int l = 0; l < 32; ++l) { const int t = wo[w] * 32 + ((l + rot) & 31); if (t < n) order[q++] = t; }
            }
        }
        std::vector<char> skipw((n + 31) / 32, 0);          // whole warps lose their turn now and then (skew between warps)
        if (c.random) for (auto &sw : skipw) sw = next_rand(c.rng) % 3 == 0;
        for (int q = 0; q < n && !c.failed; ++q) {
            Fiber &f = c.fibers[order[q]];
            if (f.done) continue;
            if (f.wait_addr && ((*f.wait_addr & f.wait_mask) == f.wait_val)) continue;
            if (skipw[f.warp]) { skipped = true; continue; }
            t_cur = &f;
            emu_switch(&c.sched_sp, f.sp);
            progress = true;
            if (f.done) remaining -= 1;
        }
        t_cur = nullptr;
        for (size_t a = 0; a < c.async.size() && !c.failed;) {
            if (--c.async[a].delay <= 0) {
                std::function<void()> fire = std::move(c.async[a].fire);
                c.async.erase(c.async.begin() + a);
                fire(); progress = true;
            } else ++a;
        }
        if (!progress && !c.failed) {
            if (skipped) continue;
            if (!c.async.empty()) { c.async[next_rand(c.rng) % c.async.size()].delay = 0; continue; }
            describe_deadlock(c);
        }
    }
    // copies still in flight when the last thread exited: completed now (so that the racecheck sees their writes), and
    // reported -- on a GPU they would land in shared memory that may already belong to the next CTA
    if (!c.failed && !c.async.empty()) {
        std::vector<AsyncOp> rest;
        rest.swap(c.async);
        for (AsyncOp &op : rest) if (!c.failed) op.fire();
        if (!c.failed) { c.failed = true; c.error = std::string("emu: kernel ") + c.kernel_name + ": the CTA exited with TMA / bulk copies in flight"; }
    }
}

struct LaunchError { std::mutex m; std::string msg; };
inline LaunchError &launch_error() { static LaunchError e; return e; }
inline long env_long(const char *name, long dflt) { const char *v = getenv(name); return v && *v ? atol(v) : dflt; }
inline std::atomic<long> &launch_counter() { static std::atomic<long> n{0}; return n; }
// bytes the kernels REQUEST from / send to global memory through the copy engines and the streaming stores (what the L2
// sees before any caching): [0] TMA boxes (the part inside the tensor), [1] bulk copies, [2] cp.async, [3] streaming stores
inline std::atomic<long long> *traffic_counters() { static std::atomic<long long> c[4]; return c; }
inline std::map<const void *, size_t> &func_smem() { static std::map<const void *, size_t> m; return m; }
constexpr size_t kSmemOptin = 232448;                       // 227 KB: sm_100 per-block opt-in limit
constexpr size_t kSmemDefault = 48 * 1024;

// fiber stacks and the shared-memory buffer of a worker, reused across launches (fresh mappings would be page-faulted in
// again on every launch)
struct Arena { char *stacks = nullptr; size_t stack_bytes = 0; unsigned char *smem_raw = nullptr; size_t smem_alloc = 0; };
inline std::vector<Arena> &arena_pool() { static std::vector<Arena> p; return p; }
inline std::mutex &arena_mutex() { static std::mutex m; return m; }
inline Arena acquire_arena(size_t stack_bytes, size_t smem_alloc) {
    Arena a;
    {
        std::lock_guard<std::mutex> lk(arena_mutex());
        auto &p = arena_pool();
        for (size_t q = 0; q < p.size(); ++q)
            if (p[q].stack_bytes >= stack_bytes && p[q].smem_alloc >= smem_alloc) { a = p[q]; p.erase(p.begin() + q); return a; }
        if (!p.empty()) { a = p.back(); p.pop_back(); }
    }
    if (a.stack_bytes < stack_bytes) {
        if (a.stacks) munmap(a.stacks, a.stack_bytes);
        void *m = mmap(nullptr, stack_bytes, PROT_READ | PROT_WRITE, MAP_PRIVATE | MAP_ANONYMOUS | MAP_NORESERVE, -1, 0);
        a.stacks = m == MAP_FAILED ? nullptr : static_cast<char *>(m); a.stack_bytes = stack_bytes;
    }
    if (a.smem_alloc < smem_alloc) {
        free(a.smem_raw);
        a.smem_raw = static_cast<unsigned char *>(malloc(smem_alloc)); a.smem_alloc = smem_alloc;
    }
    return a;
}
inline void release_arena(const Arena &a) { std::lock_guard<std::mutex> lk(arena_mutex()); arena_pool().push_back(a); }

// persistent worker threads (a fresh std::thread per launch costs a stack mapping and a malloc arena every time)
struct WorkerPool {
    std::mutex m;
    std::condition_variable cv_job, cv_done;
    std::vector<std::thread> threads;
    const std::function<void()> *job = nullptr;
    long generation = 0;
    int wanted = 0, started = 0, running = 0;
    void loop() {
        long seen = 0;
        for (;;) {
            const std::function<void()> *j = nullptr;
            {
                std::unique_lock<std::mutex> lk(m);
                cv_job.wait(lk, [&] { return generation != seen && started < wanted; });
                if (generation != seen && started < wanted) { started += 1; j = job; }
                seen = generation;
            }
            if (j) {
                (*j)();
                std::lock_guard<std::mutex> lk(m);
                if (--running == 0) cv_done.notify_all();
            }
        }
    }
    // runs `fn` on n pool threads at once and returns when all n calls have returned; one launch at a time
    void run(int n, const std::function<void()> &fn) {
        static std::mutex one_launch;
        std::lock_guard<std::mutex> serial(one_launch);
        std::unique_lock<std::mutex> lk(m);
        while ((int)threads.size() < n) { threads.emplace_back([this] { loop(); }); threads.back().detach(); }
        job = &fn; wanted = n; started = 0; running = n; generation += 1;
        cv_job.notify_all();
        cv_done.wait(lk, [&] { return running == 0; });
        job = nullptr; wanted = 0;
    }
};
inline WorkerPool &worker_pool() { static WorkerPool *p = new WorkerPool(); return *p; }     // never destroyed

// the grid: CTAs are handed out in blockIdx order (x fastest) to EMU_THREADS workers
inline int launch(dim3 grid, dim3 block, size_t smem_bytes, const void *func, const char *name, const std::function<void()> &body) {
    const int nthreads = (int)(block.x * block.y * block.z);
    if (nthreads < 1 || nthreads > 1024 || block.z > 64 || grid.x < 1 || grid.y < 1 || grid.z < 1 || grid.x > 2147483647u ||
        grid.y > 65535u || grid.z > 65535u) {                                               // the limits of the CUDA programming guide
        std::lock_guard<std::mutex> lk(launch_error().m);
        launch_error().msg = "emu: invalid launch configuration"; return 1;
    }
    {
        size_t allowed = kSmemDefault;
        auto it = func_smem().find(func);
        if (it != func_smem().end()) allowed = std::max(allowed, it->second);
        if (smem_bytes > allowed || smem_bytes > kSmemOptin) {
            std::lock_guard<std::mutex> lk(launch_error().m);
            launch_error().msg = "emu: dynamic shared memory exceeds what cudaFuncSetAttribute allowed / the 227 KB limit"; return 1;
        }
    }
    const long seed = env_long("EMU_SEED", 0);
    const bool racecheck = env_long("EMU_RACECHECK", 0) != 0;
    const long launch_no = launch_counter()++;
    const size_t n_cta = (size_t)grid.x * grid.y * grid.z;
    int n_workers = (int)env_long("EMU_THREADS", (long)std::thread::hardware_concurrency());
    n_workers = (int)std::max<size_t>(1, std::min<size_t>((size_t)std::max(n_workers, 1), n_cta));
    std::atomic<size_t> next{0};
    std::atomic<bool> failed{false};
    std::vector<Region> regions_now;
    { std::lock_guard<std::mutex> lk(regions_mutex()); regions_now = regions(); }
    if (env_long("EMU_FAULT_HANDLER", 1)) emu_install_fault_handler();
    auto worker = [&]() {
        emu_thread_altstack();
        const size_t stack_bytes = (size_t)nthreads * kStackBytes;
        const size_t canary = 1024, smem_alloc = (smem_bytes + canary + 1023) / 1024 * 1024 + 2048;
        Arena ar = acquire_arena(stack_bytes, smem_alloc);
        char *stacks = ar.stacks;
        if (!stacks || !ar.smem_raw) { failed = true; return; }
        unsigned char *smem = reinterpret_cast<unsigned char *>(((uintptr_t)ar.smem_raw + 1023) / 1024 * 1024);
        for (;;) {
            const size_t b = next.fetch_add(1);
            if (b >= n_cta || failed.load()) break;
            Cta c;
            c.bidx = dim3((unsigned)(b % grid.x), (unsigned)((b / grid.x) % grid.y), (unsigned)(b / ((size_t)grid.x * grid.y)));
            c.bdim = block; c.gdim = grid; c.nthreads = c.alive = nthreads;
            c.smem = smem; c.smem_bytes = smem_bytes;
            memset(smem, 0xFF, smem_bytes);                          // poison: NaN / id 255
            memset(smem + smem_bytes, 0xA5, canary);
            c.fibers.resize(nthreads);
            c.warps.resize((nthreads + 31) / 32);
            for (int t = 0; t < nthreads; ++t) {
                Fiber &f = c.fibers[t];
                f.tid = t; f.lane = t & 31; f.warp = t >> 5; f.cta = &c;
                f.tidx = uint3{(unsigned)(t % block.x), (unsigned)((t / block.x) % block.y), (unsigned)(t / (block.x * block.y))};
            }
            if (nthreads % 32) c.warps.back().alive = nthreads % 32;
            c.body = &body; c.kernel_name = name; c.regions = &regions_now;
            RaceState race;
            if (racecheck && smem_bytes > 0) {
                race.n = nthreads + 1;
                race.clocks.assign((size_t)race.n * race.n, 0);
                for (int t = 0; t < race.n; ++t) race.clk(t)[t] = 1;
                race.shadow.assign((smem_bytes + 3) / 4, RaceState::Shadow());
                c.race = &race;
            }
            c.random = seed != 0;
            c.rng = (uint64_t)seed * 0x2545f4914f6cdd1dull + (uint64_t)launch_no * 1315423911ull + b * 2654435761ull;
            run_cta(c, stacks);
            if (!c.failed) {
                for (size_t q = 0; q < canary; ++q)
                    if (smem[smem_bytes + q] != 0xA5) {
                        c.failed = true;
                        c.error = std::string("emu: kernel ") + name + " wrote behind its dynamic shared memory (offset +" + std::to_string(q) + ")";
                        break;
                    }
            }
            if (!c.failed)
                for (const Fiber &f : c.fibers)
                    if (!f.copies.empty()) { c.failed = true; c.error = std::string("emu: kernel ") + name + ": a thread exited with cp.async copies never waited for"; break; }
            if (c.failed) {
                std::lock_guard<std::mutex> lk(launch_error().m);
                if (launch_error().msg.empty()) launch_error().msg = c.error;
                failed = true;
            }
        }
        release_arena(ar);
    };
    if (n_workers == 1) worker();
    else worker_pool().run(n_workers, worker);
    return failed.load() ? 1 : 0;
}

template <typename... P> struct Launcher {
    void (*k)(P...);
    dim3 g, b;
    size_t s;
    const char *name;
    template <typename... A> void operator()(A &&...a) const {
        auto kk = k;
        std::function<void()> body = [=]() { kk(a...); };
        if (launch(g, b, s, reinterpret_cast<const void *>(kk), name, body)) {
            std::lock_guard<std::mutex> lk(launch_error().m);
            emu_last_error = cudaErrorLaunchFailure;
            emu_last_error_text = launch_error().msg;
            launch_error().msg.clear();
        }
    }
};
template <typename... P> inline Launcher<P...> make_launcher(void (*k)(P...), dim3 g, dim3 b, size_t s, const char *name) {
    return Launcher<P...>{k, g, b, s, name};
}

}  // namespace emu

#define threadIdx (emu::t_cur->tidx)
#define blockIdx (emu::t_cur->cta->bidx)
#define blockDim (emu::t_cur->cta->bdim)
#define gridDim (emu::t_cur->cta->gdim)

// ---- device intrinsics ----------------------------------------------------------------------------------------------
inline void __syncthreads() {
    emu::Cta *c = emu::t_cur->cta;
    emu::sync_point();
    emu::cta_barrier_arrive(c, c->bars[0], c->alive, true, "__syncthreads", 0);
}
inline void __syncwarp(unsigned mask = 0xffffffffu) { emu::warp_xchg(0, mask, true); }
template <typename T> inline T __shfl_sync(unsigned mask, T v, int src, int width = 32) {
    (void)width; return emu::from_bits<T>(emu::warp_xchg(emu::to_bits(v), mask)[src & 31]);
}
template <typename T> inline T __shfl_up_sync(unsigned mask, T v, unsigned delta, int width = 32) {
    (void)width; const int lane = emu::t_cur->lane;
    const uint64_t *b = emu::warp_xchg(emu::to_bits(v), mask);
    return emu::from_bits<T>(b[lane >= (int)delta ? lane - (int)delta : lane]);
}
template <typename T> inline T __shfl_down_sync(unsigned mask, T v, unsigned delta, int width = 32) {
    (void)width; const int lane = emu::t_cur->lane;
    const uint64_t *b = emu::warp_xchg(emu::to_bits(v), mask);
    return emu::from_bits<T>(b[lane + (int)delta < 32 ? lane + (int)delta : lane]);
}
inline unsigned __ballot_sync(unsigned mask, int pred) {
    const uint64_t *b = emu::warp_xchg(pred ? 1 : 0, mask);
    unsigned r = 0;
    for (int l = 0; l < 32; ++l) if (b[l]) r |= 1u << l;
    return r;
}
inline int __all_sync(unsigned mask, int pred) { return __ballot_sync(mask, pred) == 0xffffffffu; }
inline int __any_sync(unsigned mask, int pred) { return __ballot_sync(mask, pred) != 0u; }
inline long long clock64() { return 0; }
inline void __nanosleep(unsigned) { emu::yield(); }

// ---- runtime API ----------------------------------------------------------------------------------------------------
typedef void *cudaStream_t;
struct emu_event_ {};
typedef emu_event_ *cudaEvent_t;
enum cudaMemcpyKind { cudaMemcpyHostToHost = 0, cudaMemcpyHostToDevice = 1, cudaMemcpyDeviceToHost = 2, cudaMemcpyDeviceToDevice = 3 };
enum cudaDeviceAttr { cudaDevAttrMultiProcessorCount = 16, cudaDevAttrMaxSharedMemoryPerBlockOptin = 97 };
enum cudaFuncAttribute { cudaFuncAttributeMaxDynamicSharedMemorySize = 8 };
enum cudaMemoryType { cudaMemoryTypeUnregistered = 0, cudaMemoryTypeHost = 1, cudaMemoryTypeDevice = 2 };
struct cudaPointerAttributes { cudaMemoryType type; int device; };
struct cudaPitchedPtr { void *ptr; size_t pitch, xsize, ysize; };
struct cudaExtent { size_t width, height, depth; };
struct cudaMemcpy3DParms { cudaPitchedPtr srcPtr, dstPtr; cudaExtent extent; cudaMemcpyKind kind; };
inline cudaPitchedPtr make_cudaPitchedPtr(void *p, size_t pitch, size_t xs, size_t ys) { return cudaPitchedPtr{p, pitch, xs, ys}; }
inline cudaExtent make_cudaExtent(size_t w, size_t h, size_t d) { return cudaExtent{w, h, d}; }

inline const char *cudaGetErrorString(cudaError_t e) {
    if (e == cudaSuccess) return "no error";
    return emu_last_error_text.empty() ? "emulated CUDA error" : emu_last_error_text.c_str();
}
inline cudaError_t cudaGetLastError() { cudaError_t e = emu_last_error; emu_last_error = cudaSuccess; return e; }
inline cudaError_t cudaGetDevice(int *d) { *d = 0; return cudaSuccess; }
inline cudaError_t cudaSetDevice(int) { return cudaSuccess; }
inline cudaError_t cudaGetDeviceCount(int *n) { *n = 1; return cudaSuccess; }
inline cudaError_t cudaDeviceGetAttribute(int *v, cudaDeviceAttr a, int) {
    *v = a == cudaDevAttrMultiProcessorCount ? (int)emu::env_long("EMU_SM_COUNT", 148) : (int)emu::kSmemOptin;
    return cudaSuccess;
}
inline cudaError_t cudaPointerGetAttributes(cudaPointerAttributes *a, const void *) { a->type = cudaMemoryTypeDevice; a->device = 0; return cudaSuccess; }
inline cudaError_t cudaStreamSynchronize(cudaStream_t) { return emu_last_error; }
inline cudaError_t cudaMemcpyAsync(void *d, const void *s, size_t n, cudaMemcpyKind, cudaStream_t) { memcpy(d, s, n); return cudaSuccess; }
inline cudaError_t cudaMemsetAsync(void *d, int v, size_t n, cudaStream_t) { memset(d, v, n); return cudaSuccess; }
inline cudaError_t cudaMemcpy2DAsync(void *d, size_t dp, const void *s, size_t sp, size_t w, size_t h, cudaMemcpyKind, cudaStream_t) {
    for (size_t y = 0; y < h; ++y) memcpy(static_cast<char *>(d) + y * dp, static_cast<const char *>(s) + y * sp, w);
    return cudaSuccess;
}
inline cudaError_t cudaMemcpy3DAsync(const cudaMemcpy3DParms *m, cudaStream_t) {
    for (size_t z = 0; z < m->extent.depth; ++z)
        for (size_t y = 0; y < m->extent.height; ++y)
            memcpy(static_cast<char *>(m->dstPtr.ptr) + (z * m->dstPtr.ysize + y) * m->dstPtr.pitch,
                   static_cast<const char *>(m->srcPtr.ptr) + (z * m->srcPtr.ysize + y) * m->srcPtr.pitch, m->extent.width);
    return cudaSuccess;
}
template <typename T> inline cudaError_t cudaMemcpyToSymbol(T &sym, const void *src, size_t n) { memcpy(&sym, src, n); return cudaSuccess; }
inline cudaError_t cudaFuncSetAttribute(const void *f, cudaFuncAttribute, int v) {
    if ((size_t)v > emu::kSmemOptin) return cudaErrorInvalidValue;
    emu::func_smem()[f] = (size_t)v; return cudaSuccess;
}
inline cudaError_t cudaEventCreate(cudaEvent_t *e) { *e = new emu_event_(); return cudaSuccess; }
inline cudaError_t cudaEventDestroy(cudaEvent_t e) { delete e; return cudaSuccess; }
inline cudaError_t cudaEventRecord(cudaEvent_t, cudaStream_t) { return cudaSuccess; }
inline cudaError_t cudaEventSynchronize(cudaEvent_t) { return cudaSuccess; }
inline cudaError_t cudaEventElapsedTime(float *ms, cudaEvent_t, cudaEvent_t) { *ms = 0.f; return cudaSuccess; }

// ---- driver API: tensor maps ----------------------------------------------------------------------------------------
typedef int CUresult;
constexpr CUresult CUDA_SUCCESS = 0, CUDA_ERROR_INVALID_VALUE = 1;
typedef uint32_t cuuint32_t;
typedef uint64_t cuuint64_t;
enum CUtensorMapDataType { CU_TENSOR_MAP_DATA_TYPE_UINT8 = 0, CU_TENSOR_MAP_DATA_TYPE_FLOAT32 = 7, CU_TENSOR_MAP_DATA_TYPE_FLOAT64 = 8 };
enum CUtensorMapInterleave { CU_TENSOR_MAP_INTERLEAVE_NONE = 0 };
enum CUtensorMapSwizzle { CU_TENSOR_MAP_SWIZZLE_NONE = 0 };
enum CUtensorMapL2promotion { CU_TENSOR_MAP_L2_PROMOTION_NONE = 0, CU_TENSOR_MAP_L2_PROMOTION_L2_64B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B };
enum CUtensorMapFloatOOBfill { CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE = 0 };
struct alignas(64) CUtensorMap {
    char *base; uint64_t dims[3]; uint64_t strides[2]; uint32_t box[3]; uint32_t esz, rank, valid;
    char pad_[128 - 8 - 24 - 16 - 12 - 12];
};
static_assert(sizeof(CUtensorMap) == 128, "CUtensorMap is 128 bytes");
// the argument checks of cuTensorMapEncodeTiled that matter here (CUDA driver API reference)
inline CUresult emu_cuTensorMapEncodeTiled(CUtensorMap *m, CUtensorMapDataType dt, cuuint32_t rank, void *base, const cuuint64_t *dims,
                                           const cuuint64_t *strides, const cuuint32_t *box, const cuuint32_t *estrides,
                                           CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill) {
    if (!m || rank != 3 || !base || ((uintptr_t)base % 16) || ((uintptr_t)m % 64)) return CUDA_ERROR_INVALID_VALUE;
    const uint32_t esz = dt == CU_TENSOR_MAP_DATA_TYPE_UINT8 ? 1 : dt == CU_TENSOR_MAP_DATA_TYPE_FLOAT32 ? 4 : 8;
    for (int d = 0; d < 3; ++d) {
        if (dims[d] < 1 || dims[d] > (1ull << 32) || box[d] < 1 || box[d] > 256 || estrides[d] < 1 || estrides[d] > 8) return CUDA_ERROR_INVALID_VALUE;
        m->dims[d] = dims[d]; m->box[d] = box[d];
    }
    for (int d = 0; d < 2; ++d) {
        if (strides[d] % 16 || strides[d] >= (1ull << 40)) return CUDA_ERROR_INVALID_VALUE;
        m->strides[d] = strides[d];
    }
    if (((uint64_t)box[0] * esz) % 16) return CUDA_ERROR_INVALID_VALUE;
    m->base = static_cast<char *>(base); m->esz = esz; m->rank = 3; m->valid = 0x7e57a901u;
    return CUDA_SUCCESS;
}
enum cudaDriverEntryPointQueryResult { cudaDriverEntryPointSuccess = 0 };
constexpr int cudaEnableDefault = 0;
inline cudaError_t cudaGetDriverEntryPoint(const char *name, void **fn, int, cudaDriverEntryPointQueryResult *q) {
    *fn = strcmp(name, "cuTensorMapEncodeTiled") == 0 ? reinterpret_cast<void *>(&emu_cuTensorMapEncodeTiled) : nullptr;
    *q = cudaDriverEntryPointSuccess; return cudaSuccess;
}
