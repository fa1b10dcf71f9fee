// mbarrier, bulk async copy (TMA engine, 1-D) and gpu-scope counter primitives for sm_100a (inline PTX).
//
// Loads:  cp.async.bulk global -> shared, completion counted in bytes on an mbarrier (SASS UBLKCP).
// Stores: cp.async.bulk shared -> global as a bulk async-group of the issuing thread.
// Cross-CTA hand-over: monotone 64-bit counters in global memory, red.release / ld.acquire at gpu scope.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace bege {

#define BEGE_DA __device__ __forceinline__

BEGE_DA uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

BEGE_DA void mbar_init(uint64_t* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(smem_u32(bar)), "r"(count) : "memory");
}
BEGE_DA void mbar_arrive(uint64_t* bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" :: "r"(smem_u32(bar)) : "memory");
}
BEGE_DA void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(smem_u32(bar)), "r"(bytes) : "memory");
}
BEGE_DA bool mbar_try_wait(uint64_t* bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    return ok != 0;
}

// a stuck pipeline must abort, never hang the GPU: every wait gives up after kSpinLimit SM clocks (~0.5 s), raises the
// abort flag (checked by the host after the launch) and lets the caller run on with whatever it has
constexpr long long kSpinLimit = 1000000000ll;

BEGE_DA void mbar_wait(uint64_t* bar, uint32_t parity, int* abort_flag)
{
    if (mbar_try_wait(bar, parity)) return;
    const long long t0 = clock64();
    while (!mbar_try_wait(bar, parity)) {
        if (*(volatile int*)abort_flag) return;
        if (clock64() - t0 > kSpinLimit) { *(volatile int*)abort_flag = 1; return; }
    }
}

BEGE_DA void fence_proxy_async() { asm volatile("fence.proxy.async;" ::: "memory"); }
BEGE_DA void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
BEGE_DA void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }

BEGE_DA uint64_t policy_evict_first()
{
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
BEGE_DA uint64_t policy_evict_last()
{
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}

// global -> shared, `bytes` a multiple of 16, both addresses 16-byte aligned; completes on `bar`
BEGE_DA void bulk_load(void* smem_dst, const void* gmem_src, uint32_t bytes, uint64_t* bar, uint64_t policy)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
                 :: "r"(smem_u32(smem_dst)), "l"(gmem_src), "r"(bytes), "r"(smem_u32(bar)), "l"(policy) : "memory");
}
// shared -> global, joins the issuing thread's current bulk async-group
BEGE_DA void bulk_store(void* gmem_dst, const void* smem_src, uint32_t bytes, uint64_t policy)
{
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group.L2::cache_hint [%0], [%1], %2, %3;"
                 :: "l"(gmem_dst), "r"(smem_u32(smem_src)), "r"(bytes), "l"(policy) : "memory");
}
BEGE_DA void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
BEGE_DA void bulk_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }   // source reusable
BEGE_DA void bulk_wait0() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }             // writes done

BEGE_DA void counter_add_release(unsigned long long* ctr, unsigned long long v)
{
    asm volatile("red.release.gpu.global.add.u64 [%0], %1;" :: "l"(ctr), "l"(v) : "memory");
}
BEGE_DA unsigned long long counter_load_acquire(const unsigned long long* ctr)
{
    unsigned long long v;
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(ctr) : "memory");
    return v;
}
BEGE_DA void counter_add_relaxed(unsigned long long* ctr, unsigned long long v)
{
    asm volatile("red.relaxed.gpu.global.add.u64 [%0], %1;" :: "l"(ctr), "l"(v) : "memory");
}
BEGE_DA unsigned long long counter_load_relaxed(const unsigned long long* ctr)
{
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(ctr) : "memory");
    return v;
}
// whole warp waits until *ctr >= target: lane 0 polls (relaxed, L2), the value is broadcast so that the loop is
// warp-uniform and the warp stays converged.  The data guarded by the counter must be read with ld.global.cg
// (L2 is the point of coherence; the producer publishes with a gpu-scope release after its writes completed).
BEGE_DA void warp_counter_wait_ge(const unsigned long long* ctr, unsigned long long target, int* abort_flag, int lane)
{
    const long long t0 = clock64();
    for (;;) {
        unsigned long long v = 0;
        int bail = 0;
        if (lane == 0) {
            v = counter_load_relaxed(ctr);
            if (v < target) {
                bail = *(volatile int*)abort_flag;
                if (clock64() - t0 > kSpinLimit) { *(volatile int*)abort_flag = 1; bail = 1; }
            }
        }
        v = __shfl_sync(0xffffffffu, v, 0);
        bail = __shfl_sync(0xffffffffu, bail, 0);
        if (v >= target || bail) break;
        __nanosleep(400);
    }
    __syncwarp();
}
// one thread spins until *ctr >= target
BEGE_DA void counter_wait_ge(const unsigned long long* ctr, unsigned long long target, int* abort_flag)
{
    if (counter_load_acquire(ctr) >= target) return;
    const long long t0 = clock64();
    for (;;) {
        if (counter_load_acquire(ctr) >= target) return;
        if (*(volatile int*)abort_flag) return;
        if (clock64() - t0 > kSpinLimit) { *(volatile int*)abort_flag = 1; return; }
        __nanosleep(64);
    }
}

}  // namespace bege
