// mc_async.cuh -- sm_100a asynchronous-copy plumbing of the 3-D sweep kernels: TMA tile loads
// (cp.async.bulk.tensor through a CUtensorMap) completing on shared-memory mbarriers ("full" per stage), and the
// "empty" mbarriers on which the consumer warps hand a stage back to the producer lane.  Thin inline-PTX wrappers, no
// arithmetic of the method.
#pragma once

#include <cuda.h>          // CUtensorMap (type only; the encode entry point is fetched at run time in mc_tvd.cu)
#include <stdio.h>

#include "mc_common.cuh"

namespace mc {

MC_DEV unsigned smem_addr(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }

MC_DEV void mbar_init(unsigned bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}

// make freshly initialised barriers visible to the async proxy (the TMA unit) before the first copy
MC_DEV void mbar_init_fence() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }

// one arrival (release at CTA scope: the thread's earlier shared-memory writes are visible to a waiter)
MC_DEV void mbar_arrive(unsigned bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}

// the same, executed by the lanes whose `pred` is true, without a branch
MC_DEV void mbar_arrive_if(unsigned bar, bool pred)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.b32 p, %1, 0;\n"
        "@p mbarrier.arrive.shared::cta.b64 _, [%0];\n"
        "}\n" ::"r"(bar), "r"((unsigned)pred)
        : "memory");
}

// one arrival that also announces `bytes` of asynchronous-copy traffic the phase has to wait for
MC_DEV void mbar_arrive_expect_tx(unsigned bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}

// block until the phase of parity `parity` has completed (acquire at CTA scope); the hardware suspends the
// warp inside try_wait for a bounded time, so the loop rarely spins
MC_DEV void mbar_wait(unsigned bar, unsigned parity)
{
#ifdef MC_DEBUG_HANG
    for (long long spin = 0;; ++spin) {
        unsigned ok;
        asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}\n"
                     : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
        if (ok) return;
        if (spin > 2000000) {
            printf("STUCK block (%d,%d,%d) thread (%d,%d) bar %u parity %u\n", blockIdx.x, blockIdx.y, blockIdx.z,
                   threadIdx.x, threadIdx.y, bar, parity);
            __trap();
        }
    }
#endif
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "MC_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra MC_DONE;\n"
        "bra MC_WAIT;\n"
        "MC_DONE:\n"
        "}\n" ::"r"(bar), "r"(parity)
        : "memory");
}

// 4-D tiled TMA load global -> shared, completing `bytes of the box` on the mbarrier
MC_DEV void tma_load_4d(unsigned dst, const CUtensorMap *map, unsigned bar, int c0, int c1, int c2, int c3)
{
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
        ::"r"(dst), "l"(map), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
        : "memory");
}

// expect_tx + 4-D load, executed by the lanes whose `pred` is true, without a branch
MC_DEV void tma_issue_4d_if(bool pred, unsigned dst, const CUtensorMap *map, unsigned bar, unsigned bytes, int c0, int c1,
                            int c2, int c3)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.b32 p, %8, 0;\n"
        "@p mbarrier.arrive.expect_tx.shared::cta.b64 _, [%2], %7;\n"
        "@p cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];\n"
        "}\n" ::"r"(dst), "l"(map), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(bytes), "r"((unsigned)pred)
        : "memory");
}

MC_DEV void tma_prefetch_descriptor(const CUtensorMap *map)
{
    asm volatile("prefetch.tensormap [%0];" ::"l"(map) : "memory");
}

}  // namespace mc
