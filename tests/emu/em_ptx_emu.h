// em_ptx_emu.h -- TEST INFRASTRUCTURE: what csrc/em_ptx.cuh becomes in the emulated build (-DEM_EMULATE, tests/emu): the
// same names and signatures, implemented on the fiber machine of emu_cuda.h with the argument checks the hardware (or
// compute-sanitizer) would make.  The semantics follow the PTX ISA: mbarrier phases with pending-arrival and tx counts,
// try_wait.parity, bar.sync / bar.arrive with a thread count, cp.async groups, bulk / tensor copies that complete_tx on
// an mbarrier, zero fill outside the tensor.
#pragma once
#include "emu_cuda.h"
#include <algorithm>

namespace em {

// (launch_sweep_tma launches through a function pointer called `kern`: the instantiation selected at em_create)
inline const char *kernel_label(const char *s) { return strcmp(s, "kern") == 0 ? "k_sweep_tma" : s; }
#define EM_LAUNCH(kernel, grid, block, smem, stream) ((void)(stream), emu::make_launcher(kernel, dim3(grid), dim3(block), (size_t)(smem), em::kernel_label(#kernel)))
#define EM_DYN_SMEM(name) unsigned char *name = emu::t_cur->cta->smem
#define EM_FUZZ() emu::sync_point()

template <typename T> inline void st_stream16(void *dst, const T &v) {
    static_assert(sizeof(T) == 16, "16-byte vectors only");
    emu::check_global(dst, 16, 16, "st.global.cs.v4");
    emu::traffic_counters()[3].fetch_add(16, std::memory_order_relaxed);
    memcpy(dst, &v, 16);
}
inline float rcp_approx(float x) { return 1.0f / x; }
inline void opaque2(int &, int &) {}

// ---- cp.async: recorded, performed inside cp_async_wait ---------------------------------------------------------------
inline void cp_async_n(void *smem_dst, const void *gsrc, int n) {
    emu::Fiber *f = emu::t_cur;
    emu::check_smem(smem_dst, n, n, "cp.async");
    emu::check_global(gsrc, n, n, "cp.async");
    emu::traffic_counters()[2].fetch_add(n, std::memory_order_relaxed);
    f->copies.push_back(emu::Fiber::Copy{smem_dst, gsrc, n, f->open_group});
}
inline void cp_async16(void *d, const void *s) { cp_async_n(d, s, 16); }
inline void cp_async8(void *d, const void *s) { cp_async_n(d, s, 8); }
inline void cp_async4(void *d, const void *s) { cp_async_n(d, s, 4); }
inline void cp_async_commit() { emu::t_cur->open_group += 1; }
template <int N> inline void cp_async_wait() {
    emu::Fiber *f = emu::t_cur;
    size_t keep = 0;
    for (size_t q = 0; q < f->copies.size(); ++q) {
        const emu::Fiber::Copy &c = f->copies[q];
        if (c.group < f->open_group - N) memcpy(c.dst, c.src, c.bytes);
        else f->copies[keep++] = c;
    }
    f->copies.resize(keep);
}

// ---- mbarrier -----------------------------------------------------------------------------------------------------
// the 8 bytes in shared memory: word 0 = phase parity (bit 0) | pending arrivals (bits 1-15) | expected arrivals
// (bits 16-30), word 1 = pending transaction bytes
struct MBar { volatile uint32_t state; volatile int32_t tx; };
inline unsigned smem_u32(const void *p) { return emu::smem_to_u32(p); }
inline MBar *mbar_at(unsigned bar, const char *what, bool must_be_init = true) {
    MBar *b = reinterpret_cast<MBar *>(emu::u32_to_smem(bar, 8, 8, what));
    if (must_be_init && !emu::t_cur->cta->mbar_init.count(bar)) emu::fail_here(std::string(what) + ": mbarrier was never initialised");
    return b;
}
inline emu::SyncClock &mbar_clock(emu::Cta *c, const MBar *b) {
    return c->mbar_init[(unsigned)(reinterpret_cast<const unsigned char *>(b) - c->smem) + emu::kSmemBase];
}
inline void mbar_complete_if_done(emu::Cta *c, MBar *b) {
    const uint32_t pending = (b->state >> 1) & 0x7fffu, expected = (b->state >> 16) & 0x7fffu;
    if (pending == 0 && b->tx == 0) {
        b->state = (expected << 16) | (expected << 1) | ((b->state & 1u) ^ 1u);
        emu::race_complete(c, mbar_clock(c, b));
    }
}
inline void mbar_init(unsigned bar, unsigned count) {
    MBar *b = mbar_at(bar, "mbarrier.init", false);
    if (count < 1 || count > 0x7fffu) emu::fail_here("mbarrier.init: bad count");
    b->state = (count << 16) | (count << 1); b->tx = 0;
    emu::t_cur->cta->mbar_init[bar] = emu::SyncClock();
}
inline void mbar_fence_init() {}
inline void mbar_arrive_n(MBar *b, const char *what) {
    const uint32_t pending = (b->state >> 1) & 0x7fffu;
    if (pending == 0) emu::fail_here(std::string(what) + ": more arrivals than the barrier expects in this phase");
    emu::race_release(mbar_clock(emu::t_cur->cta, b));
    b->state -= 2u;
    mbar_complete_if_done(emu::t_cur->cta, b);
}
inline void mbar_arrive(unsigned bar) { emu::sync_point(); mbar_arrive_n(mbar_at(bar, "mbarrier.arrive"), "mbarrier.arrive"); }
inline void mbar_expect_tx(unsigned bar, unsigned bytes) {
    MBar *b = mbar_at(bar, "mbarrier.arrive.expect_tx");
    b->tx += (int32_t)bytes;
    mbar_arrive_n(b, "mbarrier.arrive.expect_tx");
}
inline void mbar_wait(unsigned bar, unsigned parity) {
    MBar *b = mbar_at(bar, "mbarrier.try_wait");
    emu::block_while(&b->state, 1u, parity & 1u, "mbarrier.try_wait.parity, smem offset", (long)(bar - emu::kSmemBase));
    emu::race_acquire(mbar_clock(emu::t_cur->cta, b));
    emu::sync_point();
}

// ---- named barriers (ids 1..15) -----------------------------------------------------------------------------------------
inline void pair_arrive(int id) {
    emu::sync_point();
    if (id < 1 || id > 15) emu::fail_here("bar.arrive: barrier id out of range");
    emu::Cta *c = emu::t_cur->cta;
    emu::cta_barrier_arrive(c, c->bars[id], 64, false, "bar.arrive", id);
}
inline void pair_sync(int id) {
    if (id < 1 || id > 15) emu::fail_here("bar.sync: barrier id out of range");
    emu::Cta *c = emu::t_cur->cta;
    emu::cta_barrier_arrive(c, c->bars[id], 64, true, "bar.sync, barrier id", id);
    emu::sync_point();
}

// ---- bulk / tensor copies: queued, completed by the scheduler after a delay --------------------------------------------
template <int POL> inline unsigned long long l2_policy() { return 0; }
inline int async_delay(emu::Cta *c) { return c->random ? (int)(emu::next_rand(c->rng) % 7) : 1; }
inline void async_complete_tx(emu::Cta *c, MBar *b, unsigned bytes, const std::shared_ptr<emu::RaceAsync> &ra) {
    emu::race_async_complete(c, mbar_clock(c, b), ra);
    b->tx -= (int32_t)bytes;
    mbar_complete_if_done(c, b);
}
inline void bulk_load(unsigned dst, const void *src, unsigned bytes, unsigned bar) {
    emu::Cta *c = emu::t_cur->cta;
    if (bytes == 0 || bytes % 16) emu::fail_here("cp.async.bulk: size must be a multiple of 16");
    unsigned char *d = emu::u32_to_smem(dst, bytes, 16, "cp.async.bulk (destination)");
    emu::check_global(src, bytes, 16, "cp.async.bulk (source)");
    MBar *b = mbar_at(bar, "cp.async.bulk (mbarrier)");
    emu::traffic_counters()[1].fetch_add(bytes, std::memory_order_relaxed);
    const std::shared_ptr<emu::RaceAsync> ra = emu::race_async_issue();
    const void *pc = __builtin_return_address(0);
    c->async.push_back(emu::AsyncOp{async_delay(c), [=]() {
        memcpy(d, src, bytes);
        emu::race_async_write(c, ra, d, bytes, pc);
        async_complete_tx(c, b, bytes, ra);
    }});
}
template <int POL>
inline void tma_load_3d(unsigned dst, const CUtensorMap *map, unsigned bar, int x, int y, int z) {
    emu::sync_point();
    emu::Cta *c = emu::t_cur->cta;
    if (((uintptr_t)map % 64) || map->valid != 0x7e57a901u) emu::fail_here("cp.async.bulk.tensor: not a valid (64-byte aligned, encoded) tensor map");
    const CUtensorMap m = *map;
    const size_t bytes = (size_t)m.box[0] * m.box[1] * m.box[2] * m.esz;
    unsigned char *d = emu::u32_to_smem(dst, bytes, 128, "cp.async.bulk.tensor (destination)");
    MBar *b = mbar_at(bar, "cp.async.bulk.tensor (mbarrier)");
    // coordinates may be negative or beyond the extent (zero fill), but the tensor the map describes must lie in
    // registered memory: first and last byte of the part of the box inside the tensor
    {
        long long lo[3], hi[3]; const int co0[3] = {x, y, z}; bool any = true;
        for (int a = 0; a < 3; ++a) {
            lo[a] = std::max<long long>(co0[a], 0); hi[a] = std::min<long long>((long long)co0[a] + m.box[a], (long long)m.dims[a]) - 1;
            if (hi[a] < lo[a]) any = false;
        }
        if (any) {
            emu::traffic_counters()[0].fetch_add((long long)(hi[0] - lo[0] + 1) * (hi[1] - lo[1] + 1) * (hi[2] - lo[2] + 1) * m.esz, std::memory_order_relaxed);
            const char *first = m.base + lo[2] * (long long)m.strides[1] + lo[1] * (long long)m.strides[0] + lo[0] * m.esz;
            const char *last = m.base + hi[2] * (long long)m.strides[1] + hi[1] * (long long)m.strides[0] + hi[0] * m.esz;
            emu::check_global(first, m.esz, 1, "cp.async.bulk.tensor (source, first element)");
            emu::check_global(last, m.esz, 1, "cp.async.bulk.tensor (source, last element)");
        }
    }
    const std::shared_ptr<emu::RaceAsync> ra = emu::race_async_issue();
    const void *pc = __builtin_return_address(0);
    c->async.push_back(emu::AsyncOp{async_delay(c), [=]() {
        const int co[3] = {x, y, z};
        unsigned char *out = d;
        for (uint32_t bz = 0; bz < m.box[2]; ++bz)
            for (uint32_t by = 0; by < m.box[1]; ++by) {
                const long long cz = (long long)co[2] + bz, cy = (long long)co[1] + by;
                const bool row_in = cz >= 0 && cz < (long long)m.dims[2] && cy >= 0 && cy < (long long)m.dims[1];
                for (uint32_t bx = 0; bx < m.box[0]; ++bx, out += m.esz) {
                    const long long cx = (long long)co[0] + bx;
                    if (row_in && cx >= 0 && cx < (long long)m.dims[0])
                        memcpy(out, m.base + cz * (long long)m.strides[1] + cy * (long long)m.strides[0] + cx * m.esz, m.esz);
                    else memset(out, 0, m.esz);
                }
            }
        emu::race_async_write(c, ra, d, bytes, pc);
        async_complete_tx(c, b, (unsigned)bytes, ra);
    }});
}
template <int POL> inline void tma_prefetch_3d(const CUtensorMap *map, int, int, int) {
    if (((uintptr_t)map % 64) || map->valid != 0x7e57a901u) emu::fail_here("cp.async.bulk.prefetch.tensor: not a valid tensor map");
}

}  // namespace em
