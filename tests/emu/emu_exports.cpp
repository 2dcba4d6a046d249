// emu_exports.cpp -- TEST INFRASTRUCTURE (tests/emu): the fiber switch and the guarded "device" allocator of the emulated
// build; linked with csrc/em_lib.cu into libem_emu*.so.
#include "emu_cuda.h"

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

extern "C" {

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

}  // extern "C"
