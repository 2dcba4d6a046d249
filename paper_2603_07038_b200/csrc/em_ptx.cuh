// em_ptx.cuh -- every piece of the kernels that is not plain C++: the inline-PTX wrappers (mbarrier, TMA, bulk copy,
// cp.async, named barriers, L2 policies, streaming stores, MUFU reciprocal), the dynamic shared-memory declaration and
// the kernel-launch syntax.  Gathered in one header so that the TEST build of tests/emu (-DEM_EMULATE: the same kernel
// and host sources compiled by g++ against a fiber-per-thread CPU emulation of these primitives, with bounds, alignment
// and deadlock checks -- the stand-in for compute-sanitizer, which is closed on this GPU pool) can replace exactly this
// file.  EM_EMULATE is never defined in a product build: libem.so has no CPU path.
#pragma once

#if defined(EM_EMULATE)
#include "em_ptx_emu.h"          // tests/emu/ (test infrastructure)
#else

#include <cuda.h>
#include <cuda_runtime.h>

namespace em {

// kernel<<<grid, block, dynamic shared bytes, stream>>>(args...)  ==  EM_LAUNCH((kernel), grid, block, bytes, stream)(args...)
#define EM_LAUNCH(kernel, grid, block, smem, stream) kernel<<<(grid), (block), (smem), (stream)>>>
// the dynamic shared memory of a kernel
#define EM_DYN_SMEM(name) extern __shared__ __align__(1024) unsigned char name[]

// 16-byte store with the streaming (evict-first) L2 policy: output planes are never re-read within a step,
// so they should not displace the halo rows the neighbouring tiles are about to re-read
template <typename T> __device__ __forceinline__ void st_stream16(void *dst, const T &v) {
    static_assert(sizeof(T) == 16, "16-byte vectors only");
    __stcs(reinterpret_cast<float4 *>(dst), *reinterpret_cast<const float4 *>(&v));
}

// MUFU.RCP (<= 1 ulp): the seed of rcp<float> (em_common.cuh); x is a positive normal number there
__device__ __forceinline__ float rcp_approx(float x) {
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

// ---- cp.async ----------------------------------------------------------------------------------------------------
__device__ __forceinline__ void cp_async16(void *smem_dst, const void *gsrc) {
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async4(void *smem_dst, const void *gsrc) {
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;\n" ::"r"(s), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async8(void *smem_dst, const void *gsrc) {
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"(s), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

// keeps two values opaque to the optimiser (no instruction is emitted)
__device__ __forceinline__ void opaque2(int &a, int &b) { asm volatile("" : "+r"(a), "+r"(b)); }

// ---- schedule fuzzing (test builds only: -DEM_SWEEP_FUZZ, libem_fuzz.so) ---------------------------------------------
// The plane loop of the sweep orders its shared-memory hazards with mbarriers and named barriers instead of CTA barriers.
// compute-sanitizer is closed on this GPU pool, so the evidence that no ordering edge is missing is a stress test: with a
// non-zero seed every synchronisation point (and every phase boundary) delays its warp by a pseudo-random 0-8 us -- a
// few plane-times -- and the results must stay bit-identical to the normal build (tests/test_gpu_fuzz.py).
#ifdef EM_SWEEP_FUZZ
__device__ unsigned g_em_fuzz_seed = 0;
__device__ __forceinline__ void em_fuzz() {
    const unsigned seed = g_em_fuzz_seed;
    if (seed == 0) return;
    unsigned x = ((unsigned)(clock64() >> 7) * 2654435761u) ^ seed ^ (blockIdx.x * 97u + (threadIdx.x >> 5) * 131u);
    x ^= x >> 15; x *= 2246822519u; x ^= x >> 13;
    if ((x & 3u) == 0u) __nanosleep((x >> 8) & 8191u);
}
#define EM_FUZZ() em_fuzz()
#else
#define EM_FUZZ() ((void)0)
#endif

// ---- mbarrier / TMA ----------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_arrive(unsigned bar) {
    EM_FUZZ();
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "W_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@!p bra W_%=;\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
    EM_FUZZ();
}
// 1-D bulk copy global -> shared counted on an mbarrier (bytes: multiple of 16)
__device__ __forceinline__ void bulk_load(unsigned dst, const void *src, unsigned bytes, unsigned bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
// producer / consumer named barrier of two warps (ids 1..15; id 0 is __syncthreads)
__device__ __forceinline__ void pair_arrive(int id) { EM_FUZZ(); asm volatile("bar.arrive %0, 64;" ::"r"(id) : "memory"); }
__device__ __forceinline__ void pair_sync(int id) { asm volatile("bar.sync %0, 64;" ::"r"(id) : "memory"); EM_FUZZ(); }

template <int POL> __device__ __forceinline__ unsigned long long l2_policy() {
    unsigned long long pol;
    if (POL == 1) asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    else if (POL == 2) asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    else asm volatile("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
// one box of a 3-D tensor map global -> shared, counted on an mbarrier, with an L2 cache policy
template <int POL>
__device__ __forceinline__ void tma_load_3d(unsigned dst, const CUtensorMap *map, unsigned bar, int x, int y, int z) {
    EM_FUZZ();
    const unsigned long long pol = l2_policy<POL>();
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3, %4}], [%5], %6;"
        ::"r"(dst), "l"(map), "r"(x), "r"(y), "r"(z), "r"(bar), "l"(pol) : "memory");
}
// the same box into L2 only (no shared memory, no barrier)
template <int POL>
__device__ __forceinline__ void tma_prefetch_3d(const CUtensorMap *map, int x, int y, int z) {
    const unsigned long long pol = l2_policy<POL>();
    asm volatile("cp.async.bulk.prefetch.tensor.3d.L2.global.tile.L2::cache_hint [%0, {%1, %2, %3}], %4;"
                 ::"l"(map), "r"(x), "r"(y), "r"(z), "l"(pol) : "memory");
}

}  // namespace em
#endif   // EM_EMULATE
