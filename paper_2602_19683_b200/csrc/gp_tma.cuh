// gp_tma.cuh -- thin PTX wrappers for the sm_100a asynchronous machinery the executor uses:
// mbarrier (shared-memory transaction barriers), TMA tiled loads (cp.async.bulk.tensor, SASS
// UTMALDG), proxy fences and named CTA barriers.  No CUTLASS/CuTe dependency.
#pragma once
#include <cuda.h>          // CUtensorMap (type only; the encode entry point is fetched at run time)
#include <cuda_runtime.h>
#include <stdint.h>

#include <cstdio>

namespace gpb {

// Debug aid (build with -DGPB_WATCHDOG): every spin loop of the executor reports where it is stuck
// and traps instead of hanging the device.  Off in the product build.
#ifdef GPB_WATCHDOG
#define GPB_SPIN_GUARD(counter, what, a, b)                                                                         \
    if (++(counter) > (1u << 24)) {                                                                                 \
        printf("[gpb watchdog] cta %d thread %d stuck in %s (%d, %d)\n", (int)blockIdx.x, (int)threadIdx.x, what, \
               (int)(a), (int)(b));                                                                                 \
        __trap();                                                                                                   \
    }
#else
#define GPB_SPIN_GUARD(counter, what, a, b)
#endif

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// ---- mbarrier ---------------------------------------------------------------------------------
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
// make mbarrier.init visible to the async proxy (TMA complete_tx) before first use
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory"); }

// arrive (release.cta): orders the caller's prior memory operations before the phase completion
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("{\n .reg .b64 st;\n mbarrier.arrive.shared::cta.b64 st, [%0];\n}\n" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("{\n .reg .b64 st;\n mbarrier.arrive.expect_tx.shared::cta.b64 st, [%0], %1;\n}\n" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}
// wait (acquire.cta) for the phase with the given parity to complete; try_wait suspends in hardware.
// A parity wait is only meaningful for a thread that cannot lag a whole phase behind the barrier:
// the producer protocol is therefore run by ONE lane (a lane of a diverged warp that reaches a
// wait late finds the barrier one phase further and sleeps for ever -- seen on hardware), and a
// consumer warp re-converges with __syncwarp() before its lane 0 releases a stage.
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity, int tag = 0) {
    const uint32_t a = smem_u32(bar);
    uint32_t done;
    [[maybe_unused]] unsigned spins = 0;
    (void)tag;
    do {
        GPB_SPIN_GUARD(spins, "mbar_wait", tag, parity)
        asm volatile(
            "{\n"
            " .reg .pred p;\n"
            " mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            " selp.u32 %0, 1, 0, p;\n"
            "}\n"
            : "=r"(done)
            : "r"(a), "r"(parity)
            : "memory");
    } while (!done);
}

// ---- TMA ----------------------------------------------------------------------------------------
// 2-D tiled load global -> shared, completion counted in bytes on `bar`.  c0 = inner (contiguous)
// coordinate, c1 = outer coordinate, both in elements of the tensor map.
__device__ __forceinline__ void tma_load_2d(void* smem_dst, const CUtensorMap* map, int c0, int c1, uint64_t* bar) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cta.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];\n" ::"r"(
                     smem_u32(smem_dst)),
                 "l"(reinterpret_cast<uint64_t>(map)), "r"(c0), "r"(c1), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void tma_prefetch_desc(const CUtensorMap* map) {
    asm volatile("prefetch.tensormap [%0];\n" ::"l"(reinterpret_cast<uint64_t>(map)) : "memory");
}
// warm L2 with `bytes` (multiple of 16) starting at a 16-byte aligned global address
__device__ __forceinline__ void l2_prefetch_bulk(const void* gptr, uint32_t bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;\n" ::"l"(gptr), "r"(bytes) : "memory");
}

// Generic-proxy accesses to global memory (LDG/STG, acquire loads) <-> async-proxy accesses (TMA):
// writers fence after their stores and before they signal; readers fence after the acquire and
// before issuing the TMA load.
__device__ __forceinline__ void fence_proxy_async_global() { asm volatile("fence.proxy.async.global;\n" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async_shared() { asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory"); }

// ---- named barrier among a subset of the CTA's warps ---------------------------------------------
// barrier.sync WITHOUT .aligned: the callers reach it out of lane-dependent loops, and the compiler
// does not know that an inline-asm `bar.sync` (= .aligned) needs the warp reconverged first.
template <int ID, int THREADS>
__device__ __forceinline__ void named_bar_sync() {
    asm volatile("barrier.sync %0, %1;\n" ::"n"(ID), "n"(THREADS) : "memory");
}

// ---- register re-balancing between warpgroups (all warps of the warpgroup must execute it) -------
template <int REGS>
__device__ __forceinline__ void reg_alloc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;\n" ::"n"(REGS)); }
template <int REGS>
__device__ __forceinline__ void reg_dealloc() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;\n" ::"n"(REGS)); }

// Publishing a block version: the barrier (warp or CTA) that precedes it orders the other threads' stores
// before this thread, and the release makes everything this thread has observed visible at gpu scope
// before the counter moves -- the pattern of a CUTLASS semaphore release, without the two MEMBAR.SC of
// __threadfence() + atomicAdd on every job.
__device__ __forceinline__ void red_release_add(int* p, int v) {
    asm volatile("red.release.gpu.global.add.s32 [%0], %1;\n" ::"l"(p), "r"(v) : "memory");
}

// "Not yet computed" mark of the triangular solves (gp_kernels.cuh): the pieces of x are published by their VALUES, a
// consumer polls the doubles it needs until none of them carries this bit pattern -- one L2 round trip where a flag plus
// a load of x are two.  The pattern is a SIGNALLING NaN: arithmetic never produces one (NaN results are quiet, and a
// signalling payload that enters through the inputs is quieted by the first operation), so no computed x can equal it.
constexpr long long kSolvePending = (long long)0xFFF4DEADBEEF5EEDull;

__device__ __forceinline__ int ld_acquire(const int* p) {
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];\n" : "=r"(v) : "l"(p) : "memory");
    return v;
}

}  // namespace gpb
