// mbarrier, bulk async copy (TMA engine, 1-D), shared-memory accessors and gpu-scope counter primitives
// for sm_100a (inline PTX).
//
// Loads:  cp.async.bulk global -> shared, completion counted in bytes on an mbarrier (SASS UBLKCP).
// Cross-CTA hand-over: monotone 64-bit counters in global memory.  The PTX memory-model ordering every arrow
// of the protocol relies on is listed in DESIGN.md section 5 ("hand-over"); in short:
//   producer:  data stores of a warp -> mbarrier.arrive (release, cta scope) on the CTA's per-slot barrier; the thread
//              that sees the phase complete (mbarrier.test_wait, acquire) -> fence.acq_rel.gpu -> red.relaxed.gpu
//              (the fence makes the CTA's stores, observed through the barrier, visible at gpu scope: cumulativity)
//   consumer:  ld.acquire.gpu by one thread sees the count -> fence.proxy.async (the data was written through the
//              generic proxy, the tensor copy reads it through the async proxy) -> cp.async.bulk.tensor of the rows
//              -> mbarrier completion -> shared-memory loads of all threads of the team
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace bege {

#define BEGE_DA __device__ __forceinline__

BEGE_DA uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// ---- shared memory by 32-bit address + immediate byte offset (keeps one base register per access pattern)
template <int OFF> BEGE_DA unsigned long long lds64(uint32_t a)
{
    unsigned long long v;
    asm volatile("ld.shared.b64 %0, [%1+%2];" : "=l"(v) : "r"(a), "n"(OFF));
    return v;
}
template <int OFF> BEGE_DA void lds128(uint32_t a, unsigned long long& v0, unsigned long long& v1)
{
    asm volatile("ld.shared.v2.b64 {%0, %1}, [%2+%3];" : "=l"(v0), "=l"(v1) : "r"(a), "n"(OFF));
}
template <int OFF> BEGE_DA void sts64(uint32_t a, unsigned long long v)
{
    asm volatile("st.shared.b64 [%0+%1], %2;" :: "r"(a), "n"(OFF), "l"(v) : "memory");
}

// ---- mbarrier
BEGE_DA void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(bar), "r"(count) : "memory");
}
BEGE_DA void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(bar), "r"(bytes) : "memory");
}
BEGE_DA void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" :: "r"(bar) : "memory");
}
BEGE_DA bool mbar_test_wait(uint32_t bar, uint32_t parity)      // non-blocking probe
{
    uint32_t ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}
BEGE_DA bool mbar_try_wait(uint32_t bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}

// a stuck pipeline must abort, never hang the GPU: every wait gives up after kSpinLimit SM clocks (~0.5 s), raises the
// abort flag (checked by the host after the launch) and lets the caller run on with whatever it has
constexpr long long kSpinLimit = 1000000000ll;

// The wait loop is kept short (a waiting warp shares its scheduler with working ones): the abort flag and the clock are
// looked at once per 64 probes only.
BEGE_DA void mbar_wait(uint32_t bar, uint32_t parity, int* abort_flag)
{
    if (mbar_try_wait(bar, parity)) return;
    uint32_t spins = 0;
    long long t0 = 0;
    while (!mbar_try_wait(bar, parity)) {
        if ((++spins & 63u) == 0u) {
            if (*(volatile int*)abort_flag) return;
            const long long now = clock64();
            if (t0 == 0) t0 = now;
            if (now - t0 > kSpinLimit) {
                *(volatile int*)abort_flag = 1; return;
            }
        }
    }
}

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
BEGE_DA void bulk_load(uint32_t smem_dst, const void* gmem_src, uint32_t bytes, uint32_t bar, uint64_t policy)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
                 :: "r"(smem_dst), "l"(gmem_src), "r"(bytes), "r"(bar), "l"(policy) : "memory");
}

// 2-D tiled tensor copy global -> shared through a tensor map (kernel parameter), completes on `bar` (SASS UTMALDG)
BEGE_DA void tma_load_2d(uint32_t smem_dst, const void* tmap, int c0, int c1, uint32_t bar, uint64_t policy)
{
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3}], [%4], %5;"
                 :: "r"(smem_dst), "l"(tmap), "r"(c0), "r"(c1), "r"(bar), "l"(policy) : "memory");
}

// generic-proxy writes to shared memory -> visible to the async proxy (TMA) of this CTA
BEGE_DA void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
// generic-proxy accesses (of this thread, and what it has acquired) before async-proxy accesses, all state spaces
BEGE_DA void fence_proxy_async_all() { asm volatile("fence.proxy.async;" ::: "memory"); }

// ---- tensor memory (TMEM, 512 columns x 128 lanes x 32 bit per SM), used here as a second register file for
// loop-invariant per-thread tables: tcgen05.ld/st have their own datapath and take nothing from the L1/LSU data pipe
// that the FFT exchanges saturate.  Shape 32x32b: thread i of a warp reads/writes lane 32 (warp % 4) + i, N columns.
template <int NCOLS> BEGE_DA void tmem_alloc(uint32_t smem_dst)          // one whole warp; address -> shared memory
{
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" :: "r"(smem_dst), "n"(NCOLS) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
template <int NCOLS> BEGE_DA void tmem_dealloc(uint32_t taddr)           // the same warp
{
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(taddr), "n"(NCOLS) : "memory");
}
BEGE_DA void tmem_fence_before_sync() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
BEGE_DA void tmem_fence_after_sync() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
BEGE_DA void tmem_st8(uint32_t taddr, const uint32_t (&r)[8])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};"
                 :: "r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]) : "memory");
}
BEGE_DA void tmem_st4(uint32_t taddr, const uint32_t (&r)[4])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};"
                 :: "r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]) : "memory");
}
BEGE_DA void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
// asynchronous load of 2 complex numbers (4 columns); the values may be used only after tmem_wait_ld on the same array
BEGE_DA void tmem_ld4(uint32_t taddr, unsigned long long (&w)[2])
{
    uint32_t r0, r1, r2, r3;
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(taddr));
    asm("mov.b64 %0, {%1, %2};" : "=l"(w[0]) : "r"(r0), "r"(r1));
    asm("mov.b64 %0, {%1, %2};" : "=l"(w[1]) : "r"(r2), "r"(r3));
}
// waits for all tcgen05.ld of this thread; the array is an in/out operand so that no use can be scheduled above it
BEGE_DA void tmem_wait_ld(unsigned long long (&w)[2])
{
    asm volatile("tcgen05.wait::ld.sync.aligned;" : "+l"(w[0]), "+l"(w[1]) :: "memory");
}

// the wait that covers two staging arrays (dual-stream search: stationary values and the streams' powers)
BEGE_DA void tmem_wait_ld(unsigned long long (&w)[2], unsigned long long (&f)[2])
{
    asm volatile("tcgen05.wait::ld.sync.aligned;" : "+l"(w[0]), "+l"(w[1]), "+l"(f[0]), "+l"(f[1]) :: "memory");
}

// ---- named barrier of `nthreads` threads
BEGE_DA void bar_named(int id, int nthreads) { asm volatile("bar.sync %0, %1;" :: "r"(id), "r"(nthreads) : "memory"); }

// ---- cta-scope monotone counter in shared memory (where a parity wait could be more than one phase away)
BEGE_DA void smem_counter_add_release(uint32_t addr, uint32_t v)
{
    asm volatile("red.release.cta.shared::cta.add.u32 [%0], %1;" :: "r"(addr), "r"(v) : "memory");
}
BEGE_DA uint32_t smem_counter_load_acquire(uint32_t addr)
{
    uint32_t v;
    asm volatile("ld.acquire.cta.shared::cta.u32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
    return v;
}

// ---- gpu-scope counters
BEGE_DA void fence_acq_rel_gpu() { asm volatile("fence.acq_rel.gpu;" ::: "memory"); }
BEGE_DA void counter_add_relaxed(unsigned long long* ctr, unsigned long long v)
{
    asm volatile("red.relaxed.gpu.global.add.u64 [%0], %1;" :: "l"(ctr), "l"(v) : "memory");
}
BEGE_DA unsigned long long counter_load_acquire(const unsigned long long* ctr)
{
    unsigned long long v;
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(ctr) : "memory");
    return v;
}
// ONE thread spins until *ctr >= target; every probe is an acquire load, so whatever the thread (and, after a
// CTA barrier, its team) reads afterwards is ordered after the producers' released writes.
BEGE_DA void counter_wait_ge(const unsigned long long* ctr, unsigned long long target, int* abort_flag)
{
    if (counter_load_acquire(ctr) >= target) return;
    long long t0 = 0;
    for (uint32_t spins = 1;; ++spins) {
        __nanosleep(2000);
        if (counter_load_acquire(ctr) >= target) return;
        if ((spins & 63u) == 0u) {                           // the abort flag and the clock: rarely
            if (*(volatile int*)abort_flag) return;
            const long long now = clock64();
            if (t0 == 0) t0 = now;
            if (now - t0 > kSpinLimit) {
                *(volatile int*)abort_flag = 1; return;
            }
        }
    }
}

}  // namespace bege
