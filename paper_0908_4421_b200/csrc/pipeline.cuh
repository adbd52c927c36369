// pipeline.cuh -- sm_100a building blocks: mbarrier, 1-D bulk async copy (TMA unit, cp.async.bulk), L2 cache
// policies, warp reductions, a grid-wide barrier.  Inline PTX only; nothing here knows about the optimiser.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace imrt {

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// ---------------------------------------------------------------------------------------------- mbarrier
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// the same on 32-bit shared-window addresses (computed once; keeps address conversion out of the inner loops)
__device__ __forceinline__ void mbar_expect_tx_a(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive_a(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait_a(uint32_t bar, uint32_t parity) {
    uint32_t done;
    do {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(done)
            : "r"(bar), "r"(parity)
            : "memory");
    } while (!done);
}
__device__ __forceinline__ void bulk_g2s_a(uint32_t dst_smem, const void* src_gmem, uint32_t bytes, uint32_t bar, uint64_t policy) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
        ::"r"(dst_smem), "l"(src_gmem), "r"(bytes), "r"(bar), "l"(policy)
        : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity) {
    uint32_t done;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return done != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    while (!mbar_try_wait(bar, parity)) {}
}

// Orders this thread's earlier generic-proxy accesses to shared memory (plain ld / st) before later async-proxy accesses
// (the TMA unit's writes of a bulk copy) to the same bytes.  Issued by every thread that touched the bytes, then a CTA
// barrier, then the producer may issue its bulk copies over them.
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// ---------------------------------------------------------------------------------------------- L2 policies
__device__ __forceinline__ uint64_t policy_evict_first() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ uint64_t policy_evict_last() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
}

// ---------------------------------------------------------------------------------------------- bulk copy
// global -> shared, completion signalled on an mbarrier as transaction bytes.  dst, src 16-byte aligned,
// bytes a positive multiple of 16.  SASS: UBLKCP.
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar, uint64_t policy) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
        ::"r"(smem_u32(dst_smem)), "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)), "l"(policy)
        : "memory");
}

// gather load that is asked to stay in L2 (the vector every transpose row re-reads)
__device__ __forceinline__ float ld_keep(const float* p, uint64_t policy) {
    float v;
    asm volatile("ld.global.L2::cache_hint.f32 %0, [%1], %2;" : "=f"(v) : "l"(p), "l"(policy));
    return v;
}

// ---------------------------------------------------------------------------------------------- warp reductions
template <int V>
__device__ __forceinline__ float vec_sum(float v) {   // sum over aligned groups of V lanes (V = 1,2,4,...,32)
#pragma unroll
    for (int o = V / 2; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double warp_sum(double v) {   // fixed butterfly order: bit-reproducible
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// ---------------------------------------------------------------------------------------------- named barrier
__device__ __forceinline__ void named_bar_sync(int id, int n_threads) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n_threads) : "memory");
}

// ---------------------------------------------------------------------------------------------- grid barrier
__device__ __forceinline__ unsigned long long spin_clock_ns() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}

// Monotone-counter barrier for a cooperative (co-resident) launch over the n_cta CTAs that share `counter` (the whole
// grid, or one rank's CTAs when several plans share a launch).  Every CTA calls it the same number of times;
// `epoch` counts the calls (kept in a register by the caller).  counter must be 0 at kernel start.
// Release / acquire at gpu scope: the arrival is a red.release (the CTA's earlier writes, ordered before it by the
// bar.sync, become visible to whoever acquires the count), the wait an ld.acquire spin (SASS: LDG.STRONG.GPU followed by
// CCTL.IVALL, so the other threads' plain loads after the closing bar.sync cannot hit stale L1 lines).  No full fences.
//
// The wait is BOUNDED: after timeout_ns without the count being reached, the waiter sets BAR_FAULT in the counter --
// which makes every present and future wait on it return at once -- and the call returns true ("the run is faulted") in
// every thread of every CTA that passes the barrier from then on.  Anybody else who detects a fault (a lost peer rank,
// shard_wait) sets the same bit.  The caller leaves its loop without touching another barrier.  *fault_s: one int of
// shared memory, 0 at kernel start.  The counter stays far below 2^31 in a fault-free launch (barriers x CTAs).
constexpr unsigned int BAR_FAULT = 0x80000000u;
__device__ __forceinline__ bool grid_barrier(unsigned int* counter, unsigned int& epoch, int n_cta, unsigned long long timeout_ns,
                                             volatile int* fault_s) {
    __syncthreads();
    ++epoch;
    if (threadIdx.x == 0) {
        asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(counter) : "memory");
        const unsigned int target = epoch * (unsigned int)n_cta;
        unsigned int seen, polls = 0u;
        unsigned long long t0 = 0ull;
        for (;;) {
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(counter) : "memory");
            if (seen >= target) break;                       // also true once BAR_FAULT is set
            if ((++polls & 255u) == 0u) {                    // look at the clock once in a while only
                const unsigned long long now = spin_clock_ns();
                if (t0 == 0ull) t0 = now;
                else if (now - t0 > timeout_ns) { atomicOr(counter, BAR_FAULT); seen = BAR_FAULT; break; }
            }
        }
        if (seen & BAR_FAULT) *fault_s = 1;
    }
    __syncthreads();
    return *fault_s != 0;
}

}  // namespace imrt
