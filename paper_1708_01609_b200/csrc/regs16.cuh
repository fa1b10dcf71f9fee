// Helpers on a thread's 16 complex registers that the search kernel (bege.cu) and the overlap-save probe (ovs_probe.cuh)
// share: unrolled shared-memory exchange and twiddle tables streamed from tensor memory.
#pragma once
#include "cplx.cuh"
#include "async.cuh"

namespace bege {

// 16 values to shared memory at a + p * STRIDE bytes
template <int STRIDE, int P = 0> BEGE_D void sts16(uint32_t a, const c2 (&v)[16])
{
    if constexpr (P < 16) { sts64<P * STRIDE>(a, v[P]); sts16<STRIDE, P + 1>(a, v); }
}
template <int STRIDE, int P = 0> BEGE_D void lds16(uint32_t a, c2 (&v)[16])
{
    if constexpr (P < 16) { v[P] = lds64<P * STRIDE>(a); lds16<STRIDE, P + 1>(a, v); }
}
// v[P0 + 2 j + k] *= table entry (2 j + k), entries streamed from tensor memory two at a time, double buffered;
// the load of chunk 0 into wa was issued by the caller; chunks [0, NCH)
template <int P0, int NCH, int J = 0> BEGE_D void tm_twiddle(uint32_t taddr, c2 (&v)[16], c2 (&wa)[2], c2 (&wb)[2])
{
    if constexpr (J < NCH) {
        c2 (&cur)[2] = (J & 1) ? wb : wa;
        c2 (&nxt)[2] = (J & 1) ? wa : wb;
        tmem_wait_ld(cur);
        if constexpr (J + 1 < NCH) tmem_ld4(taddr + 4 * (J + 1), nxt);
        v[P0 + 2 * J] = cmulw(v[P0 + 2 * J], cur[0]);
        if constexpr (P0 + 2 * J + 1 < 16) v[P0 + 2 * J + 1] = cmulw(v[P0 + 2 * J + 1], cur[1]);
        tm_twiddle<P0, NCH, J + 1>(taddr, v, wa, wb);
    }
}

}  // namespace bege
