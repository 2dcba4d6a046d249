// emu_exports.cpp -- TEST INFRASTRUCTURE (tests/emu): the fiber switch and the guarded "device" allocator of the emulated
// build; linked with csrc/em_lib.cu into libem_emu*.so.
#include "emu_cuda.h"

#include <signal.h>
#include <unistd.h>

#if defined(__x86_64__)
asm(R"(
.text
.hidden emu_switch
.globl emu_switch
.type emu_switch,@function
emu_switch:
    pushq %rbp
    pushq %rbx
    pushq %r12
    pushq %r13
    pushq %r14
    pushq %r15
    movq %rsp, (%rdi)
    movq %rsi, %rsp
    popq %r15
    popq %r14
    popq %r13
    popq %r12
    popq %rbx
    popq %rbp
    ret
.size emu_switch,.-emu_switch
)");
#else
#error "tests/emu: the fiber switch is written for x86-64"
#endif

// ---- a fault inside an emulated kernel (guard page of the workspace, wild pointer, misaligned SSE access): say where ----
namespace {
void fault_handler(int sig, siginfo_t *si, void *) {
    char buf[1024];
    const emu::Fiber *f = emu::t_cur;
    const uintptr_t a = (uintptr_t)si->si_addr;
    int n;
    if (f && f->cta) {
        const emu::Cta *c = f->cta;
        long smem_off = (a >= (uintptr_t)c->smem && a < (uintptr_t)c->smem + c->smem_bytes + 4096) ? (long)(a - (uintptr_t)c->smem) : -1;
        long best = 0; int where = 0;                                  // distance to the nearest registered region
        if (c->regions)
            for (const emu::Region &r : *c->regions) {
                if (a < r.lo && (where == 0 || (long)(r.lo - a) < best)) { best = (long)(r.lo - a); where = -1; }
                if (a >= r.hi && (where == 0 || (long)(a - r.hi) < best)) { best = (long)(a - r.hi); where = 1; }
            }
        n = snprintf(buf, sizeof(buf), "\nemu: FAULT (signal %d) in kernel %s, block (%u,%u,%u), thread %d (warp %d lane %d): address %p%s",
                     sig, c->kernel_name, c->bidx.x, c->bidx.y, c->bidx.z, f->tid, f->warp, f->lane, si->si_addr,
                     smem_off >= 0 ? " = dynamic shared memory offset " : "");
        if (!si->si_addr) n += snprintf(buf + n, sizeof(buf) - n, " -- no address: a general-protection fault, i.e. almost certainly a MISALIGNED 16-byte "
                                "vector access (what a GPU reports as 'misaligned address'); rebuild with the UBSan traps to get the line");
        else if (smem_off >= 0) n += snprintf(buf + n, sizeof(buf) - n, "%ld (of %zu bytes)", smem_off, c->smem_bytes);
        else if (where && si->si_addr) n += snprintf(buf + n, sizeof(buf) - n, ", %ld bytes %s an emu_alloc'ed region (out-of-bounds global access)", best, where < 0 ? "BEFORE" : "BEHIND");
        n += snprintf(buf + n, sizeof(buf) - n, "\n");
    } else {
        n = snprintf(buf, sizeof(buf), "\nemu: FAULT (signal %d) at address %p outside any emulated kernel\n", sig, si->si_addr);
    }
    if (write(2, buf, (size_t)n) < 0) {}
    _exit(128 + sig);
}
}  // namespace

extern "C" {

// installs the handler (idempotent); every worker thread also gets an alternate signal stack (emu_cuda.h)
void emu_install_fault_handler(void) {
    static bool done = false;
    if (done) return;
    done = true;
    struct sigaction sa;
    memset(&sa, 0, sizeof(sa));
    sa.sa_sigaction = fault_handler;
    sa.sa_flags = SA_SIGINFO | SA_ONSTACK;
    sigemptyset(&sa.sa_mask);
    sigaction(SIGSEGV, &sa, nullptr);
    sigaction(SIGBUS, &sa, nullptr);
}
void emu_thread_altstack(void) {
    static thread_local char *stk = nullptr;
    if (stk) return;
    stk = static_cast<char *>(malloc(64 * 1024));
    stack_t ss; ss.ss_sp = stk; ss.ss_size = 64 * 1024; ss.ss_flags = 0;
    sigaltstack(&ss, nullptr);
}

// bytes of "device memory" between two PROT_NONE guard pages, registered for the range checks of the emulated
// wrappers; the returned pointer is 256-byte aligned and its end is within 255 bytes of the trailing guard page
void *emu_alloc(size_t bytes) {
    const size_t page = (size_t)sysconf(_SC_PAGESIZE);
    const size_t body = (bytes + page - 1) / page * page;
    char *raw = static_cast<char *>(mmap(nullptr, body + 2 * page, PROT_NONE, MAP_PRIVATE | MAP_ANONYMOUS | MAP_NORESERVE, -1, 0));
    if (raw == MAP_FAILED) return nullptr;
    if (mprotect(raw + page, body, PROT_READ | PROT_WRITE) != 0) return nullptr;
    char *p = raw + page + (body - bytes) / 256 * 256;
    std::lock_guard<std::mutex> lk(emu::regions_mutex());
    emu::regions().push_back(emu::Region{(uintptr_t)p, (uintptr_t)p + bytes});
    return p;
}

void emu_free(void *ptr, size_t bytes) {
    const size_t page = (size_t)sysconf(_SC_PAGESIZE);
    const size_t body = (bytes + page - 1) / page * page;
    {
        std::lock_guard<std::mutex> lk(emu::regions_mutex());
        auto &r = emu::regions();
        for (size_t q = 0; q < r.size(); ++q) if (r[q].lo == (uintptr_t)ptr) { r.erase(r.begin() + q); break; }
    }
    char *raw = reinterpret_cast<char *>(((uintptr_t)ptr) / page * page) - page;
    // the body may start up to one page after raw + page only if (body - bytes) >= page, which it never is
    munmap(raw, body + 2 * page);
}

long emu_launch_count(void) { return emu::launch_counter().load(); }
// reads (and clears) the requested-traffic counters of emu_cuda.h: TMA, bulk, cp.async, streaming stores [bytes]
void emu_traffic(long long out[4]) { for (int q = 0; q < 4; ++q) out[q] = emu::traffic_counters()[q].exchange(0); }

// ---- the hooks a -fsanitize=thread build of the kernels calls on every load and store (libtsan is NOT linked: this is
// the emulation's own happens-before race detector for the dynamic shared memory, emu_cuda.h "racecheck") -------------
#define EMU_PC __builtin_return_address(0)
void __tsan_init(void) {}
void __tsan_func_entry(void *) {}
void __tsan_func_exit(void) {}
void __tsan_vptr_update(void **, void *) {}
void __tsan_vptr_read(void **) {}
void __tsan_read1(void *a) { emu::race_access(a, 1, false, EMU_PC); }
void __tsan_read2(void *a) { emu::race_access(a, 2, false, EMU_PC); }
void __tsan_read4(void *a) { emu::race_access(a, 4, false, EMU_PC); }
void __tsan_read8(void *a) { emu::race_access(a, 8, false, EMU_PC); }
void __tsan_read16(void *a) { emu::race_access(a, 16, false, EMU_PC); }
void __tsan_write1(void *a) { emu::race_access(a, 1, true, EMU_PC); }
void __tsan_write2(void *a) { emu::race_access(a, 2, true, EMU_PC); }
void __tsan_write4(void *a) { emu::race_access(a, 4, true, EMU_PC); }
void __tsan_write8(void *a) { emu::race_access(a, 8, true, EMU_PC); }
void __tsan_write16(void *a) { emu::race_access(a, 16, true, EMU_PC); }
void __tsan_unaligned_read2(void *a) { emu::race_access(a, 2, false, EMU_PC); }
void __tsan_unaligned_read4(void *a) { emu::race_access(a, 4, false, EMU_PC); }
void __tsan_unaligned_read8(void *a) { emu::race_access(a, 8, false, EMU_PC); }
void __tsan_unaligned_read16(void *a) { emu::race_access(a, 16, false, EMU_PC); }
void __tsan_unaligned_write2(void *a) { emu::race_access(a, 2, true, EMU_PC); }
void __tsan_unaligned_write4(void *a) { emu::race_access(a, 4, true, EMU_PC); }
void __tsan_unaligned_write8(void *a) { emu::race_access(a, 8, true, EMU_PC); }
void __tsan_unaligned_write16(void *a) { emu::race_access(a, 16, true, EMU_PC); }
void __tsan_read_range(void *a, unsigned long n) { if (n) emu::race_access(a, n, false, EMU_PC); }
void __tsan_write_range(void *a, unsigned long n) { if (n) emu::race_access(a, n, true, EMU_PC); }
// atomics of the emulation's own host code (std::atomic in launch()): plain builtins
#define EMU_ATOMIC(bits, T)                                                                                              \
    T __tsan_atomic##bits##_load(const volatile T *a, int) { return __atomic_load_n(a, __ATOMIC_SEQ_CST); }              \
    void __tsan_atomic##bits##_store(volatile T *a, T v, int) { __atomic_store_n(a, v, __ATOMIC_SEQ_CST); }              \
    T __tsan_atomic##bits##_exchange(volatile T *a, T v, int) { return __atomic_exchange_n(a, v, __ATOMIC_SEQ_CST); }    \
    T __tsan_atomic##bits##_fetch_add(volatile T *a, T v, int) { return __atomic_fetch_add(a, v, __ATOMIC_SEQ_CST); }    \
    T __tsan_atomic##bits##_fetch_sub(volatile T *a, T v, int) { return __atomic_fetch_sub(a, v, __ATOMIC_SEQ_CST); }    \
    int __tsan_atomic##bits##_compare_exchange_strong(volatile T *a, T *e, T v, int, int) {                              \
        return __atomic_compare_exchange_n(a, e, v, 0, __ATOMIC_SEQ_CST, __ATOMIC_SEQ_CST); }                            \
    int __tsan_atomic##bits##_compare_exchange_weak(volatile T *a, T *e, T v, int, int) {                                \
        return __atomic_compare_exchange_n(a, e, v, 1, __ATOMIC_SEQ_CST, __ATOMIC_SEQ_CST); }
EMU_ATOMIC(8, unsigned char)
EMU_ATOMIC(16, unsigned short)
EMU_ATOMIC(32, unsigned int)
EMU_ATOMIC(64, unsigned long)
void __tsan_atomic_thread_fence(int) { __atomic_thread_fence(__ATOMIC_SEQ_CST); }
void __tsan_atomic_signal_fence(int) { __atomic_signal_fence(__ATOMIC_SEQ_CST); }

}  // extern "C"
