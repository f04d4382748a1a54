// Shared-memory mbarrier helpers (PTX mbarrier.*, CTA scope) used by the rings of partial sums in
// transfer.cu and fused.cu.
#pragma once

#include <stdint.h>

namespace gcamb {

__device__ __forceinline__ void mbar_init(uint32_t bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_inval(uint32_t bar)
{
    asm volatile("mbarrier.inval.shared::cta.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, int parity)
{
    uint32_t done;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n" : "=r"(done) : "r"(bar), "r"(parity) : "memory");
    return done != 0;
}
// Wait for the phase with the given parity.  A failed try_wait comes back after ~20 cycles on sm_100a
// whatever suspend-time hint it is given (measured: 6.7e6 loop iterations in one config-1 transfer
// launch, 7 % of all issued instructions, taken from the FP64 instructions of the warps that share the
// scheduler), so a waiting warp sleeps between polls, doubling the nap up to `max_ns`.
__device__ __forceinline__ void mbar_wait(uint32_t bar, int parity, unsigned max_ns = 512)
{
    if (mbar_try_wait(bar, parity)) return;
    unsigned ns = 32;
    do {
        __nanosleep(ns);
        if (ns < max_ns) ns <<= 1;
    } while (!mbar_try_wait(bar, parity));
}

}  // namespace gcamb
