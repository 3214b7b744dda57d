// digest_common.h -- cp.async / mbarrier helpers and tile constants shared by the two digestion kernels
// (ltjk_digest.cu: block panels; ltjk_pdigest.cu: pair lists).
#pragma once
#include <cuda_runtime.h>
#include "ltjk_internal.h"

namespace ltjk {

constexpr int kMT = kDigestRows;   // rows per CTA (128)
constexpr int kMTP = kMT + 2;      // padded row stride of the A tile in shared memory
constexpr int kKC = 16;            // contraction chunk
constexpr int kStages = 5;
constexpr int kTM = 16;            // rows per consumer warp
constexpr int kConsumerWarps = 8;
constexpr int kProducerWarps = 4;
constexpr int kProducerThreads = kProducerWarps * 32;
constexpr int kDigestThreads = (kConsumerWarps + kProducerWarps) * 32;
static_assert(kConsumerWarps * kTM == kMT, "consumer warps must cover the row tile");

__device__ __forceinline__ void cp_async8(void* smem, const void* gmem, bool valid)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    const int sz = valid ? 8 : 0;
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(s), "l"(gmem), "r"(sz));
}
__device__ __forceinline__ void cp_async16(void* smem, const void* gmem, bool valid)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    const int sz = valid ? 16 : 0;
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(gmem), "r"(sz));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }

// ---- mbarrier helpers (producer/consumer pipeline inside one CTA) -------------------------------------------------
__device__ __forceinline__ void mbar_init(unsigned long long* bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(unsigned long long* bar)
{
    asm volatile("{\n.reg .b64 st;\nmbarrier.arrive.shared::cta.b64 st, [%0];\n}\n" ::"r"((unsigned)__cvta_generic_to_shared(bar))
                 : "memory");
}
// arrive on `bar` once all cp.async issued so far by this thread have landed (the count was provisioned at init)
__device__ __forceinline__ void mbar_arrive_on_cp_async(unsigned long long* bar)
{
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];\n" ::"r"((unsigned)__cvta_generic_to_shared(bar))
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity)
{
    const unsigned a = (unsigned)__cvta_generic_to_shared(bar);
    asm volatile(
        "{\n.reg .pred p;\nWAIT_%=:\nmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n@p bra DONE_%=;\nbra WAIT_%=;\nDONE_%=:\n}\n" ::"r"(a),
        "r"(parity)
        : "memory");
}

}  // namespace ltjk
