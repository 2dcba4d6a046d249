// selftest.cpp -- TEST INFRASTRUCTURE (tests/emu): checks the checker.  Small kernels written against the emulated
// primitives (emu_cuda.h, em_ptx_emu.h), each either correct -- its result is compared with the definition of the PTX
// operation -- or carrying ONE deliberate bug of the kind the emulation exists to catch (a missing wait, a misaligned TMA
// destination, an out-of-range address, a barrier nobody arrives at ...); the bug must be reported.  Driven by
// tests/test_emu_selftest.py through selftest_run(case, message buffer).
#define EM_EMULATE 1
#include "em_ptx_emu.h"
#include "emu_cuda.h"

#include <cstdio>
#include <cstring>
#include <string>

using namespace em;

extern "C" void *emu_alloc(size_t bytes);
extern "C" void emu_free(void *ptr, size_t bytes);

namespace {

struct Args {
    CUtensorMap map;
    float *src;        // [4][8][64] floats
    float *out;        // results
    int bug;
};

constexpr int NX = 64, NY = 8, NZ = 4;

// one 32 x 4 x 1 box of the tensor at (x0, y0, z0) -> shared memory, then every thread copies its elements out
__global__ void k_tma(const __grid_constant__ Args a, int x0, int y0, int z0) {
    EM_DYN_SMEM(sm);
    const int tid = threadIdx.x;
    const unsigned bar = smem_u32(sm + 1024);
    const unsigned dst = smem_u32(sm) + (a.bug == 4 ? 64u : 0u);                    // bug 4: destination not 128-B aligned
    if (tid == 0) {
        if (a.bug != 7) mbar_init(bar, 1);                                           // bug 7: barrier never initialised
        mbar_fence_init();
    }
    __syncthreads();
    if (tid == 0) {
        mbar_expect_tx(bar, a.bug == 3 ? 32 * 4 * 4 + 16 : 32 * 4 * 4);              // bug 3: expects more bytes than arrive
        tma_load_3d<0>(dst, &a.map, bar, x0, y0, z0);
        if (a.bug == 6) mbar_arrive(bar);                                            // bug 6: a second arrival on a count-1 barrier
    }
    if (a.bug != 2) mbar_wait(bar, 0);                                               // bug 2: consumer does not wait
    const float *s = reinterpret_cast<const float *>(sm);
    a.out[tid] = s[tid];
    if (a.bug == 5) sm[2048 + 8 + tid] = 1;                                          // bug 5: writes behind the dynamic shared memory
}

// producer / consumer warps on a named barrier + warp collectives
__global__ void k_pair(float *out, int bug) {
    EM_DYN_SMEM(sm);
    float *row = reinterpret_cast<float *>(sm);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    for (int it = 0; it < 5; ++it) {
        if (w == 0) {
            if (it > 0) pair_sync(2);                     // consumer has read the previous row
            row[lane] = (float)(100 * it + lane);
            pair_arrive(1);
        } else {
            if (bug == 1 && it == 3) { /* bug: consumer skips its wait */ } else pair_sync(1);
            const float v = row[lane];
            const float up = __shfl_up_sync(0xffffffffu, v, 1), dn = __shfl_down_sync(0xffffffffu, v, 1);
            const int all = __all_sync(0xffffffffu, v >= 100.f * it);
            out[it * 32 + lane] = v + 0.25f * (up - dn) + (all ? 1000.f : 0.f);
            if (it < 4) pair_arrive(2);
        }
    }
}

__global__ void k_cpasync(const float *src, float *out, int bug) {
    EM_DYN_SMEM(sm);
    float *slot = reinterpret_cast<float *>(sm) + 4 * threadIdx.x;
    cp_async16(slot, src + 4 * threadIdx.x + (bug == 8 ? 1 : 0));                    // bug 8: misaligned source
    cp_async_commit();
    if (bug != 9) cp_async_wait<0>();                                                // bug 9: never waited for
    out[threadIdx.x] = slot[0] + slot[3];
}

__global__ void k_store(float *dst, int bug) {
    float4 v{1.f, 2.f, 3.f, 4.f};
    st_stream16(dst + 4 * threadIdx.x + (bug == 10 ? 100000 : 0), v);              // bug 10: far outside the allocation
}

__global__ void k_deadlock(float *out) {
    EM_DYN_SMEM(sm);
    const unsigned bar = smem_u32(sm);
    if (threadIdx.x == 0) mbar_init(bar, 2);
    __syncthreads();
    if (threadIdx.x == 0) mbar_arrive(bar);           // one of two expected arrivals
    mbar_wait(bar, 0);
    out[threadIdx.x] = 1.f;
}

// racecheck: lane l writes its slot, a neighbour lane reads it -- ordered by __syncwarp (sync = 1), by a shuffle only
// (sync = 0: NOT an ordering edge) or by nothing (sync = 2)
__global__ void k_warp_order(float *out, int sync) {
    EM_DYN_SMEM(sm);
    float *slot = reinterpret_cast<float *>(sm);
    const int lane = threadIdx.x & 31;
    slot[lane] = (float)lane;
    float carried = 0.f;
    if (sync == 1) __syncwarp();
    else if (sync == 0) carried = __shfl_down_sync(0xffffffffu, (float)lane, 1);
    out[lane] = slot[(lane + 1) & 31] + 0.f * carried;
}

// racecheck: a two-slot staging ring refilled by TMA.  The producer (thread 0) may refill a slot only when every warp has
// arrived on its "empty" mbarrier; early = 1 refills without that wait (WAR on the slot, whatever the schedule).
__global__ void k_ring(const __grid_constant__ Args a, int early) {
    EM_DYN_SMEM(sm);
    const int tid = threadIdx.x, lane = tid & 31;
    const unsigned full = smem_u32(sm + 2048), empty = smem_u32(sm + 2056);
    if (tid == 0) { mbar_init(full, 1); mbar_init(empty, 4); mbar_fence_init(); }
    __syncthreads();
    float acc = 0.f;
    for (int it = 0; it < 4; ++it) {
        if (tid == 0) {
            if (it > 0 && !early) mbar_wait(empty, (unsigned)(it - 1) & 1u);
            mbar_expect_tx(full, 32 * 4 * 4);
            tma_load_3d<0>(smem_u32(sm), &a.map, full, 0, 0, it);
        }
        mbar_wait(full, (unsigned)it & 1u);
        acc += reinterpret_cast<const float *>(sm)[tid];
        __syncwarp();
        if (lane == 0) mbar_arrive(empty);
    }
    a.out[tid] = acc;
}

std::string take_error() {
    std::string s = cudaGetLastError() == cudaSuccess ? "" : cudaGetErrorString(cudaErrorLaunchFailure);
    return s;
}

}  // namespace

// returns 0 when the case behaved as it should; msg = what the emulation reported (or what went wrong)
extern "C" int selftest_run(int which, char *msg, int msg_len) {
    auto say = [&](const std::string &s) { snprintf(msg, (size_t)msg_len, "%s", s.c_str()); };
    const size_t n_src = (size_t)NX * NY * NZ;
    float *src = static_cast<float *>(emu_alloc(n_src * 4)), *out = static_cast<float *>(emu_alloc(4096 * 4));
    for (size_t q = 0; q < n_src; ++q) src[q] = (float)q;
    for (int q = 0; q < 4096; ++q) out[q] = -1.f;
    Args a;
    const cuuint64_t dims[3] = {NX, NY, NZ}, strides[2] = {NX * 4, NX * NY * 4};
    const cuuint32_t box[3] = {32, 4, 1}, ones[3] = {1, 1, 1};
    int rc = 1;
    if (emu_cuTensorMapEncodeTiled(&a.map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, src, dims, strides, box, ones, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                   CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS) {
        say("encode failed"); return 1;
    }
    a.src = src; a.out = out; a.bug = 0;
    auto tma_expected = [&](int tid, int x0, int y0, int z0) -> float {
        const int bx = tid % 32, by = tid / 32, x = x0 + bx, y = y0 + by, z = z0;
        return (x >= 0 && x < NX && y >= 0 && y < NY && z >= 0 && z < NZ) ? src[((size_t)z * NY + y) * NX + x] : 0.f;
    };
    auto run_tma = [&](int bug, int x0, int y0, int z0) { a.bug = bug; EM_LAUNCH(k_tma, 1, 128, 2048, 0)(a, x0, y0, z0); return take_error(); };
    switch (which) {
    case 0: {   // correct TMA box, inside the tensor and hanging over three of its faces (zero fill)
        const int pos[3][3] = {{16, 2, 1}, {-4, -1, 0}, {48, 6, 3}};
        rc = 0;
        for (int t = 0; t < 3 && rc == 0; ++t) {
            const std::string e = run_tma(0, pos[t][0], pos[t][1], pos[t][2]);
            if (!e.empty()) { say(e); rc = 1; break; }
            for (int tid = 0; tid < 128; ++tid)
                if (out[tid] != tma_expected(tid, pos[t][0], pos[t][1], pos[t][2])) { say("TMA box content differs from the definition"); rc = 1; break; }
        }
        if (rc == 0) say("ok");
        break;
    }
    case 2: {   // no wait: the data must NOT be there yet (asynchronous copies never complete before the issuer moves on)
        const std::string e = run_tma(2, 16, 2, 1);
        bool stale = false;
        for (int tid = 0; tid < 128; ++tid) if (!(out[tid] == tma_expected(tid, 16, 2, 1))) stale = true;
        // (the CTA may also end with the copy still in flight, which is reported)
        rc = (stale || !e.empty()) ? 0 : 1; say(stale ? "stale data seen, as it must be" : e);
        break;
    }
    case 3: case 4: case 5: case 6: case 7: {
        const std::string e = run_tma(which, 16, 2, 1);
        const char *want = which == 3 ? "DEADLOCK" : which == 4 ? "misaligned shared address" : which == 5 ? "wrote behind its dynamic shared memory"
                         : which == 6 ? "more arrivals" : "never initialised";
        rc = e.find(want) != std::string::npos ? 0 : 1; say(e.empty() ? "(nothing reported)" : e);
        break;
    }
    case 1: case 11: {   // named-barrier hand-off + collectives: correct (11) and with a skipped wait (1)
        EM_LAUNCH(k_pair, 1, 64, 1024, 0)(out, which == 1 ? 1 : 0);
        const std::string e = take_error();
        bool good = e.empty();
        for (int it = 0; it < 5 && good; ++it)
            for (int lane = 0; lane < 32; ++lane) {
                const float v = 100.f * it + lane, up = lane > 0 ? v - 1 : v, dn = lane < 31 ? v + 1 : v;
                if (out[it * 32 + lane] != v + 0.25f * (up - dn) + 1000.f) good = false;
            }
        if (which == 11) { rc = good ? 0 : 1; say(good ? "ok" : (e.empty() ? "wrong values" : e)); }
        else { rc = good ? 1 : 0; say(good ? "(the skipped wait went unnoticed)" : (e.empty() ? "wrong values seen, as they must be" : e)); }
        break;
    }
    case 8: case 9: case 12: {
        EM_LAUNCH(k_cpasync, 1, 32, 1024, 0)(src, out, which == 12 ? 0 : which);
        const std::string e = take_error();
        if (which == 12) {
            bool good = e.empty();
            for (int t = 0; t < 32 && good; ++t) if (out[t] != src[4 * t] + src[4 * t + 3]) good = false;
            rc = good ? 0 : 1; say(good ? "ok" : e);
        } else {
            const char *want = which == 8 ? "misaligned global address" : "never waited for";
            rc = e.find(want) != std::string::npos ? 0 : 1; say(e.empty() ? "(nothing reported)" : e);
        }
        break;
    }
    case 10: {
        EM_LAUNCH(k_store, 1, 32, 0, 0)(out, 10);
        const std::string e = take_error();
        rc = e.find("outside every emu_alloc'ed region") != std::string::npos ? 0 : 1; say(e.empty() ? "(nothing reported)" : e);
        break;
    }
    case 13: {
        EM_LAUNCH(k_deadlock, 1, 64, 1024, 0)(out);
        const std::string e = take_error();
        rc = e.find("DEADLOCK") != std::string::npos && e.find("mbarrier.try_wait") != std::string::npos ? 0 : 1; say(e.empty() ? "(nothing reported)" : e);
        break;
    }
    case 20: case 21: case 22: {   // racecheck: __syncwarp orders (20), a shuffle does not (21), nothing (22)
        EM_LAUNCH(k_warp_order, 1, 32, 1024, 0)(out, which == 20 ? 1 : which == 21 ? 0 : 2);
        const std::string e = take_error();
        if (which == 20) { rc = e.empty() ? 0 : 1; say(e.empty() ? "ok" : e); }
        else { rc = e.find("RACE") != std::string::npos ? 0 : 1; say(e.empty() ? "(nothing reported)" : e); }
        break;
    }
    case 23: case 24: {   // racecheck: staging ring, refilled after the empty barrier (23) / too early (24)
        a.bug = 0;
        EM_LAUNCH(k_ring, 1, 128, 4096, 0)(a, which == 24 ? 1 : 0);
        const std::string e = take_error();
        if (which == 23) {
            bool good = e.empty();
            for (int tid = 0; tid < 128 && good; ++tid) {
                float want = 0.f;
                for (int it = 0; it < 4; ++it) want += tma_expected(tid, 0, 0, it);
                if (out[tid] != want) good = false;
            }
            rc = good ? 0 : 1; say(good ? "ok" : (e.empty() ? "wrong sums" : e));
        } else { rc = e.find("RACE") != std::string::npos && e.find("async copy engine") != std::string::npos ? 0 : 1; say(e.empty() ? "(nothing reported)" : e); }
        break;
    }
    case 25: {   // racecheck: the hand-off with a skipped bar.sync is a race even if the values happen to come out right
        EM_LAUNCH(k_pair, 1, 64, 1024, 0)(out, 1);
        const std::string e = take_error();
        rc = e.find("RACE") != std::string::npos ? 0 : 1; say(e.empty() ? "(nothing reported)" : e);
        break;
    }
    case 26: {   // racecheck: the consumer that does not wait for the staged box
        const std::string e = run_tma(2, 16, 2, 1);
        rc = e.find("RACE") != std::string::npos ? 0 : 1; say(e.empty() ? "(nothing reported)" : e);
        break;
    }
    default: say("unknown case");
    }
    emu_free(src, n_src * 4); emu_free(out, 4096 * 4);
    return rc;
}
