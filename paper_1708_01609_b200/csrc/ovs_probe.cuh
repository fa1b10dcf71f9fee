// bake-off probe of the OVERLAP-SAVE variant.  Not on the product path: it exists so
// that the keep-or-kill decision on that variant rests on a measured kernel (profiles/r2_ovs_*).
//
// The templates are L = 4096 samples long, the segment N = 65536: the circular correlation of PAPER.md:74 eq.(3) can be
// assembled from six P = 16384-point correlations of overlapping blocks of the band-limited segment (block i covers the
// samples 12288 i .. 12288 i + 16383 mod N and yields the 12288 lags 12288 i ..; 6 x 12288 >= N).  A P-point transform
// fits one SM's shared memory, so there is no cross-CTA exchange and no ring, and a P-point template spectrum is 4 x
// smaller (every fourth bin of the N-point one: 128 KiB); the price is 6 x 16384 x 14 / (65536 x 16) = 1.31 x the
// butterflies, and 1.5 x the multiplies, exchanges and threshold tests.
//
// One CTA of 1024 threads (64 registers) per SM, persistent over the (template, block) items; per item
//   R[k] = conj(H16_j[k]) X16_i[k]  ->  z = IDFT_P(R) in place in shared memory (16 x 16 x 16 x 4, three exchanges)
//   ->  |z|^2 > thr on the valid lags, hits counted.
// P = 16 x 1024: thread t holds R[t + 1024 i]; 16-point DFTs over i, twiddle w_P^(t p), exchange 1 (CTA barrier): 16
// independent 1024-point problems (outputs n = p + 16 m), each owned by two warps; 1024 = 16 x 64 (exchange 2, the two
// warps meet on an mbarrier), 64 = 16 x 4 (exchange 3, four adjacent lanes).  Each thread overwrites exactly the slots it
// has read (row pitch 68 keeps every access but the last conflict free), so no second buffer is needed.
// sigma is not formed here (it would come from the template's power spectrum and the segment's autocorrelation spectrum,
// a smaller, separate reduction); the probe times the part that dominates.
#pragma once
#include "cplx.cuh"
#include "async.cuh"
#include "regs16.cuh"

namespace bege {

constexpr int kOvsP = 16384;
constexpr int kOvsPitch = 68;                                // elements per row of 64
constexpr int kOvsRegion = 16 * kOvsPitch;                   // elements per 1024-point problem
constexpr int kOvsBufBytes = 16 * kOvsRegion * 8;            // 139,264
constexpr int kOvsSmem = kOvsBufBytes + 4 * 17 * 8 + 16 * 8 + 16 + 128;

__global__ void __launch_bounds__(1024, 1)
k_ovs_probe(const c2* __restrict__ H, const c2* __restrict__ X, uint64_t T, uint32_t n_blocks, float thr2,
            unsigned long long* __restrict__ hits, c2* __restrict__ zdbg, uint64_t dbg_j, int* abort_flag)
{
    extern __shared__ __align__(128) unsigned char ovs_smem[];
    const uint32_t sb = smem_u32(ovs_smem);
    const uint32_t tw3_a = sb + kOvsBufBytes;                 // [4][17] stage-3 twiddles w_64^(v s)
    const uint32_t bar_a = tw3_a + 4 * 17 * 8;                // [16] mbarriers (two warps each)
    const uint32_t tm_a = bar_a + 16 * 8;                     // TMEM base address
    const int t = threadIdx.x, warp = t >> 5, lane = t & 31;
    if (t == 0) { for (int i = 0; i < 16; ++i) mbar_init(bar_a + 8 * i, 2); fence_mbar_init(); }
    if (t < 64) {                                             // w_64^(v s), rounded from fp64
        double sn, cs;
        sincospi(2.0 * (double)(((t >> 4) * (t & 15)) & 63) / 64.0, &sn, &cs);
        reinterpret_cast<float2*>(ovs_smem + kOvsBufBytes)[(t >> 4) * 17 + (t & 15)] = make_float2((float)cs, (float)sn);
    }
    if (t < 32) tmem_alloc<512>(tm_a);
    tmem_fence_before_sync();
    __syncthreads();
    tmem_fence_after_sync();
    const uint32_t tq = *reinterpret_cast<volatile uint32_t*>(ovs_smem + kOvsBufBytes + 4 * 17 * 8 + 16 * 8) +
                        ((uint32_t)(warp & 3) << 21) + 32u * (uint32_t)(warp >> 2);
    {   // loop-invariant twiddles in tensor memory: w_P^(t p) at columns [0, 256), w_1024^(u p) at [256, 512), p = 1 .. 15
        const int u = t & 63;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            uint32_t r1[8], r2[8];
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const int pp = 4 * j + k + 1;
                double sn, cs;
                sincospi(2.0 * (double)((pp * t) & (kOvsP - 1)) / (double)kOvsP, &sn, &cs);
                r1[2 * k] = __float_as_uint((float)cs); r1[2 * k + 1] = __float_as_uint((float)sn);
                sincospi(2.0 * (double)((pp * u) & 1023) / 1024.0, &sn, &cs);
                r2[2 * k] = __float_as_uint((float)cs); r2[2 * k + 1] = __float_as_uint((float)sn);
            }
            tmem_st8(tq + 8 * j, r1);
            tmem_st8(tq + 256 + 8 * j, r2);
        }
        tmem_wait_st();
    }
    tmem_fence_before_sync();
    __syncthreads();
    tmem_fence_after_sync();

    // ---- per-thread addresses (bytes)
    const int i1 = t >> 6, u1 = t & 63;                       // exchange 1, writer: element (p, t = u1 + 64 i1)
    const uint32_t x1w = sb + (uint32_t)(i1 * kOvsPitch + u1) * 8;              // + p * kOvsRegion * 8
    const int p = t >> 6, u = t & 63;                         // stage 2: problem p, column u
    const uint32_t reg_a = sb + (uint32_t)(p * kOvsRegion) * 8;
    const uint32_t x2 = reg_a + (uint32_t)u * 8;              // + i * pitch * 8: element i (read), element q (write)
    const int q = u >> 2, v = u & 3;                          // stage 3: 64-point problem (p, q), thread v of four
    const uint32_t x3r = reg_a + (uint32_t)(q * kOvsPitch + v) * 8;             // + 32 i: E[v + 4 i];  write (s, v): + 32 s
    const uint32_t x4r = reg_a + (uint32_t)(q * kOvsPitch + 4 * v) * 8;         // + (16 j + vv) * 8: element (s = v + 4 j, vv)
    const uint32_t bar_p = bar_a + 8 * p;
    const uint64_t n_items = T * n_blocks;
    uint32_t nit = 0;
    for (uint64_t item = blockIdx.x; item < n_items; item += gridDim.x, ++nit) {
        const uint64_t j = item / n_blocks;
        const uint32_t blk = (uint32_t)(item - j * n_blocks);
        const c2* Hj = H + j * (uint64_t)kOvsP + t;
        const c2* Xb = X + (uint64_t)blk * kOvsP + t;
        {   // next item's template spectrum towards L2 (one 128-byte line per thread)
            const uint64_t nx = item + gridDim.x;
            if (nx < n_items) {
                const c2* nh = H + (nx / n_blocks) * (uint64_t)kOvsP + 16 * t;
                asm volatile("prefetch.global.L2 [%0];" :: "l"(nh));
            }
        }
        c2 a[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) a[i] = cmulc(__ldg(Xb + 1024 * i), __ldcs(Hj + 1024 * i));
        c2 wa[2], wb[2];
        tmem_ld4(tq, wa);
        fft16<+1>(a);
        tm_twiddle<1, 8>(tq, a, wa, wb);                      // a[p] *= w_P^(t p)
        sts16<kOvsRegion * 8>(x1w, a);
        tmem_ld4(tq + 256, wa);
        __syncthreads();
        lds16<kOvsPitch * 8>(x2, a);                          // B_p[u + 64 i]
        fft16<+1>(a);
        tm_twiddle<1, 8>(tq + 256, a, wa, wb);                // a[q] *= w_1024^(u q)
        sts16<kOvsPitch * 8>(x2, a);                          // in place: element (q, u)
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_p);
        mbar_wait(bar_p, nit & 1, abort_flag);
        lds16<32>(x3r, a);                                    // E[v + 4 i] of problem (p, q)
        fft16<+1>(a);
#pragma unroll
        for (int s = 1; s < 16; ++s) {
            const c2 w = lds64<0>(tw3_a + (uint32_t)(v * 17 + s) * 8);
            a[s] = cmulw(a[s], w);
        }
        sts16<32>(x3r, a);                                    // in place: element (s, v) at 4 s + v
        __syncwarp();
#pragma unroll
        for (int jj = 0; jj < 4; ++jj)
#pragma unroll
            for (int vv = 0; vv < 4; ++vv) a[4 * jj + vv] = lds64<0>(x4r + (uint32_t)(16 * jj + vv) * 8);
#pragma unroll
        for (int jj = 0; jj < 4; ++jj) fft4<+1>(a[4 * jj], a[4 * jj + 1], a[4 * jj + 2], a[4 * jj + 3]);
        // a[4 jj + e] = z[n], n = p + 16 q + 256 (v + 4 jj) + 4096 e; lags n < 12288 of the block are valid
        const uint32_t n0 = (uint32_t)(p + 16 * q + 256 * v);
        unsigned cnt = 0;
#pragma unroll
        for (int jj = 0; jj < 4; ++jj)
#pragma unroll
            for (int e = 0; e < 3; ++e) {
                const float zr = re(a[4 * jj + e]), zi = im(a[4 * jj + e]);
                cnt += fmaf(zi, zi, zr * zr) > thr2 ? 1u : 0u;
            }
        if (__any_sync(0xffffffffu, cnt != 0)) {
            for (int d = 16; d >= 1; d >>= 1) cnt += __shfl_xor_sync(0xffffffffu, cnt, d);
            if (lane == 0) atomicAdd(hits, (unsigned long long)cnt);
        }
        if (zdbg && j == dbg_j) {
            const float inv = 1.0f / (float)kOvsP;
#pragma unroll
            for (int jj = 0; jj < 4; ++jj)
#pragma unroll
                for (int e = 0; e < 4; ++e)
                    zdbg[(uint64_t)blk * kOvsP + n0 + 1024u * jj + 4096u * e] = mul2(a[4 * jj + e], bc(inv));
        }
        __syncthreads();                                      // the buffer is free for the next item's exchange 1
    }
    tmem_fence_before_sync();
    __syncthreads();
    if (t < 32) tmem_dealloc<512>(tq - 32u * (uint32_t)(warp >> 2) - ((uint32_t)(warp & 3) << 21));
}

}  // namespace bege
