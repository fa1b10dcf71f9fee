// bege.cu -- sm_100a kernels and C ABI (include/bege.h) of the butterfly-filtering hot path of
// arXiv:1708.01609.  See DESIGN.md for the data layout and the roofline of each kernel.
//
// Index conventions (N = 65536 = 256 x 256, w_M = exp(2 pi i / M)):
//   inverse (search):  k = k1 + 256 k2,  n = 256 n1 + n2
//     z[256 n1 + n2] = 1/N sum_k1 w256^(k1 n1) [ wN^(k1 n2) sum_k2 R[k1 + 256 k2] w256^(k2 n2) ]
//     pass 1 (k_search A teams): 256-point column DFTs over k2 + first twiddle factor -> ring T[n2][k1] (L2)
//     pass 2 (k_search B teams): second twiddle factor, 256-point row DFTs over k1, threshold, compaction
//   forward (bank / segments): n = nl + 256 nh, k = k1 + 256 k2
//     H[k1 + 256 k2] = sum_nl w256^(-nl k2) [ wN^(-nl k1) sum_nh h[nl + 256 nh] w256^(-nh k1) ]
//     step A (k_fwd_rows_*): DFT over nh + twiddle -> scratch G (tile layout), step B (k_fwd_cols): DFT over nl
//   every 256-point DFT is 16 x 16: a half-warp owns one DFT, each lane 16 points in registers.
//
// "Tile layout" of a stored spectrum (bank, segments): see tile_word() in cplx.cuh -- per tile b (columns k1 = 16 b + c)
// only the kept row-blocks i in [I0, I0 + NI) (rows k2 = g + 16 i), two row-blocks per 16-byte word, the words of one
// warp of a pass-1 team contiguous (NI * 256 bytes: one bulk copy per warp and item).  The forward scratch G keeps the
// plain order ((b*16 + i)*16 + c)*16 + g over all 16 row-blocks.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

#include <cuda.h>
#include <cuda_runtime.h>

#include "../../include/bege.h"
#include "cplx.cuh"
#include "async.cuh"
#include "regs16.cuh"
#include "bank64.cuh"

#ifndef BEGE_ABL
// Ablation switches for timing experiments (profiles/r2_search_kernel.md); never set in the product build, results
// are garbage when any is set: 1 no cross-CTA waits, 2 no template tile loads, 4 no ring stores, 8 no ring loads,
// 16 pass-1 teams off, 32 pass-2 teams off.
#define BEGE_ABL 0
#endif

#ifndef BEGE_FUSE
// which passes of k_search use the FMA-fused 16-point DFT (cplx.cuh: 72 instead of 81 packed instructions): bit 0 pass 1,
// bit 1 pass 2.  Measured on one B200, same box, configs[2]: 0: 4.75 / 4.72, 1: 4.66, 2: 4.76 / 4.74,
// 3: 4.67 / 4.68 M correlations/s -- pass 1 at its 64-register budget spills 16 bytes with the fused form and loses
// 1.5 %, pass 2 takes it without spills (18 fewer packed instructions per item, rate unchanged within noise).
#define BEGE_FUSE 2
#endif

namespace bege {

constexpr int kN = 65536;
constexpr int kBatch = 72;                 // segments per launch of the forward transforms (fp32 staging: 38 MB)
constexpr int kMaxGroups = 32;             // search: persistent CTA groups of 16 tiles (9 on a 148-SM B200)
// counter block of a search, each hot word on its own 128-byte line (the record counter takes an atomic per warp with
// tails; a poll of the abort flag on the same line would queue behind them): record counter, abort flag, hit counters,
// done1 / done2 (per group and ring slot: kMaxGroups x kRing x 8 bytes each)
constexpr uint64_t kOffCounter = 0, kOffAbort = 128, kOffHits = 256, kOffDone1 = 1024, kOffDone2 = 8192, kMiscHdr = 16384;
static_assert(kOffDone1 + (uint64_t)kMaxGroups * 16 * 8 <= kOffDone2 && kOffDone2 + (uint64_t)kMaxGroups * 16 * 8 <= kMiscHdr, "counter block");
constexpr int kMaxSlices = 8;              // launches per search whose record copies overlap the next launch
constexpr uint64_t kSliceMinCorr = 32768;  // do not slice below this many correlations per slice

// ------------------------------------------------------------------------------------------------
// private 256-element region of a half-warp: lane a writes its p-th value, lane p reads over a
BEGE_D int pidx(int a, int p) { return (a << 4) + (p ^ a); }

// stage 1 of a 256-point DFT held by a half-warp: 16-point DFT over the register index, then the
// w256^(DIR * lane * p) twiddles (w1[p] = exp(+2 pi i lane p / 256), conjugated for DIR < 0)
template <int DIR>
BEGE_D void stage1(c2 (&v)[16], const float2 (&w1)[16]) {
    fft16<DIR>(v);
#pragma unroll
    for (int p = 1; p < 16; ++p) v[p] = cmulw(v[p], w1[p].x, DIR > 0 ? w1[p].y : -w1[p].y);
}

// full 256-point DFT of a half-warp through its private shared-memory region.
// in: lane a holds x[a + 16 i] in v[i];  out: lane p holds X[p + 16 q] in v[q].
template <int DIR>
BEGE_D void hw_fft256(c2 (&v)[16], const float2 (&w1)[16], c2* priv, int lane16) {
    stage1<DIR>(v, w1);
#pragma unroll
    for (int p = 0; p < 16; ++p) priv[pidx(lane16, p)] = v[p];
    __syncwarp();
#pragma unroll
    for (int a = 0; a < 16; ++a) v[a] = priv[pidx(a, lane16)];
    __syncwarp();
    fft16<DIR>(v);
}

BEGE_D void load_w1(float2 (&w1)[16], const float2* __restrict__ tw256, int lane16) {
#pragma unroll
    for (int p = 0; p < 16; ++p) w1[p] = __ldg(tw256 + p * 16 + lane16);
}

// ------------------------------------------------------------------------------------------------
// a1 (template spectra) lives in bank64.cuh: fp64 arithmetic, one fp32 rounding per stored bin.

// a2, step A: full row DFTs of a data segment.  grid (16, n_segments), 256 thr.
__global__ void __launch_bounds__(256)
k_fwd_rows_data(const c2* __restrict__ x, const float2* __restrict__ tw256, const float2* __restrict__ twN,
                c2* __restrict__ G)
{
    __shared__ c2 sm[16][256];
    const int t = threadIdx.x, ia = blockIdx.x;
    const uint64_t m = blockIdx.y;
    const int ga = t >> 4, a = t & 15;
    const int nl = ga + 16 * ia;
    float2 w1[16];
    load_w1(w1, tw256, a);
    const c2* xin = x + m * (uint64_t)kN;
    c2 v[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) v[i] = xin[nl + 256 * (a + 16 * i)];
    hw_fft256<-1>(v, w1, sm[ga], a);
    c2* out = G + m * (uint64_t)kN;
    const int p = a;
#pragma unroll
    for (int q = 0; q < 16; ++q) {
        const int k1 = p + 16 * q;
        const float2 w = __ldg(twN + nl * 256 + k1);
        out[((q * 16 + ia) * 16 + p) * 16 + ga] = cmulw(v[q], w.x, -w.y);
    }
}

// step B of both forward transforms: column DFTs over nl.  grid (16 tiles, batch), 256 thr.
// Reads G (tile layout, all 16 row-blocks), writes the kept row-blocks [I0, I0+NI) of the spectrum in
// tile layout.  MASK: zero bins outside klo <= min(k, N-k) <= khi (segments).
template <bool MASK>
__global__ void __launch_bounds__(256)
k_fwd_cols(const c2* __restrict__ G, c2* __restrict__ out, uint64_t out_stride, int I0, int NI,
           const float2* __restrict__ tw256, uint32_t klo, uint32_t khi)
{
    __shared__ c2 sm[16][256];
    const int t = threadIdx.x, b = blockIdx.x;
    const uint64_t jl = blockIdx.y;
    const int c = t >> 4, g = t & 15;
    float2 w1[16];
    load_w1(w1, tw256, g);
    const c2* in = G + jl * (uint64_t)kN + (uint64_t)b * 4096;
    c2 v[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) v[i] = in[(i * 16 + c) * 16 + g];
    hw_fft256<-1>(v, w1, sm[c], g);
    // lane p = g holds k2 = p + 16 q; row-blocks are stored in pairs (one 16-byte word per thread and pair)
    ulonglong2* o = reinterpret_cast<ulonglong2*>(out + jl * out_stride) + tile_word(NI, b, 0, t);   // + 32 ip
    const uint32_t k1 = 16 * b + c;
#pragma unroll
    for (int q = 0; q < 16; ++q) {
        if (MASK) {
            const uint32_t k = k1 + 256u * (uint32_t)(g + 16 * q);
            const uint32_t kk = k < (uint32_t)kN / 2 ? k : (uint32_t)kN - k;
            if (kk < klo || kk > khi) v[q] = mk(0.f, 0.f);
        }
    }
#pragma unroll
    for (int ip = 0; ip < 8; ++ip) {
        if (2 * ip < NI) {
            ulonglong2 w;
            // (I0, NI) is (1, 14) or (0, 16): both spelled out so that v is indexed with compile-time constants
            if (I0 == 1) { w.x = v[(2 * ip + 1) & 15]; w.y = v[(2 * ip + 2) & 15]; }
            else         { w.x = v[2 * ip]; w.y = v[(2 * ip + 1) & 15]; }
            o[ip * 32] = w;
        }
    }
}

// ------------------------------------------------------------------------------------------------
// a3 - a7, one persistent warp-specialised kernel for a whole search (PAPER.md:156-162 steps ii-iv; eq.5-9, 13).
// grid (16 tiles, G groups), one CTA of 32 warps (64 registers per thread) per SM, cooperative launch (all CTAs
// co-resident).  The 16 CTAs of a group share the group's (template, segment) items; item `it` of a group is the
// pair (template grp + G (it / nS), segment it % nS).  CTA (b, grp) owns columns k1 = 16 b + c in pass 1 and rows
// n2 = 16 b + r in pass 2.  Four teams of 8 warps, two per pass, team k of a pass taking the items it = k (mod 2).
//
//   A teams (pass 1): every WARP is autonomous -- it owns two columns of the tile (half-warp = column c, lane g holds
//              rows k2 = g + 16 i), and nothing in its item needs another warp: no CTA or team barrier in the loop
//              (the team barriers of the earlier version cost pass 1 a quarter of its time, profiles/r2_search_kernel.md).
//              R = conj(H) X needs one column tile of the template spectrum and one of the segment spectrum.  One of
//              them is STATIONARY -- it sits in tensor memory, 14 complex numbers per thread -- and the other STREAMS
//              through a per-warp shared-memory buffer: the warp's words of a tile are contiguous (tile_word), ONE
//              bulk async copy per warp and item, tracked by the warp's own mbarrier, issued as soon as the warp has
//              read the previous one:
//                single-segment calls (nS = 1): X stationary (loaded once per launch), H streams from HBM;
//                batched calls (nS >= 2):       H stationary (one load per template, it serves all nS segments --
//                                               PAPER.md:156 "loaded once per M inverse FFTs"), X streams from L2.
//              Stage 1: 128-bit loads of the streaming tile, conj(H) X, Parseval partial sum, 16-point DFTs, twiddles
//              theta^p (tensor memory).  The 256-point column DFT is finished inside the half-warp: one exchange
//              through a private padded shared-memory region (__syncwarp only), 16-point DFTs, and lane p holds
//              T[n2 = p + 16 q][k1] in v[q].  The ring keeps an item as T'[k1][n2] (column-major): the 16 lanes of a
//              half-warp store 128 contiguous bytes per q, a warp fills 4 KiB contiguous per item.
//   B teams (pass 2): the 16 rows n2 of T this CTA owns are a 256 x 16 box of T' (256 lines of 128 bytes): ONE tensor
//              copy (TMA, 128-byte swizzle) brings it into a 32 KiB shared-memory tile (3 tiles rotate over the items
//              of both teams, so the next item's copy runs while this one is computed).  The 16 lanes that own row r
//              read its 256 values (conflict free thanks to the swizzle and to the lane map below), apply the four-step
//              factor, run the 256-point row DFT over k1 with their own 256 slots of the tile as the exchange area,
//              threshold against k^2 sum|R|^2 and compact the tails with warp-aggregated atomics.  No warp of pass 2
//              issues a global load of ring data, so none queues behind the store bursts of pass 1 in the LSU.
//              Lane map of a B warp w: row r = 2 w + ((lane >> 3) & 1), a = (lane & 7) | ((lane >> 4) << 3), so that
//              each hardware half-warp covers 8 values of a x 2 rows = 16 distinct 8-byte bank pairs.
//
// Tensor memory holds the loop-invariant per-thread tables (read with tcgen05.ld: no L1/LSU wavefronts -- the LSU
// data pipe was the binding unit of the round-1 kernel at 75 %, see profiles/):
//   columns [0, 32):    pass 2: delta_p = exp(2 pi i a (b + 16 p) / 4096), p < 16 -- the lane-dependent part of the
//                       four-step factor wN^(16 b k1), k1 = a + 16 r, times the inner twiddle w256^(a p); 4 quadrants
//   columns [32, 96):   pass 1, team 0: the stationary tile, 28 columns per thread, 32 per warp of a lane quadrant
//   columns [96, 160):  pass 1: theta^p = exp(2 pi i p (256 g + k1) / N), p = 1 .. 15, same arrangement
//   columns [160, 192): unused
//   columns [192, 256): pass 1, team 1: its copy of the stationary tile (batched calls: the teams change template
//                       at different times)
//   columns [256, 320): dual-stream search only (that variant allocates all 512 columns): per bin of this thread the
//                       pair (|H1~[k]|^2, |L1~[k]|^2) of the segment, 28 columns per thread, 32 per warp of a quadrant
// The CTA-uniform part of the four-step factor, w256^(b r), comes from constant memory (uniform loads, one row per CTA).  All table
// entries are rounded once from fp64 angles.
//
// Hand-over between the passes (PTX memory model): per group and ring slot two monotone counters.
//   done1 (tiles in the ring): each warp of an A team arrives on the CTA's mbarrier amb[slot] after its ring stores.
//              The warp whose arrival completes the phase (it sees so with a test_wait right after) executes ONE
//              fence.acq_rel.gpu and adds 1 to done1[slot] -- pass 1 has the time for the microsecond the gpu-scope
//              fence takes, it is the side that waits for ring slots; a publication cursor in shared memory, claimed by
//              CAS, keeps every tile published exactly once (thread 0 of the B team of the same item parity publishes
//              whatever it finds unpublished in its wait loop and after its last item).
//              That B thread -- the team's service thread -- waits with ld.acquire.gpu until all 16 tiles of its team's
//              item have been added, then issues the tensor copy of the rows.
//   done2 (ring slot read out): as soon as that copy has landed (mbarrier), a thread of the B team adds 1 to
//              done2[slot] under the same kind of fence.  Every A warp acquires 16 of them just before its ring stores
//              (all lanes load the one counter, so the warp stays converged; 2 us between probes while waiting).
// The ring holds kRing items per group (G x kRing x 512 KiB) and lives in L2.
#ifndef BEGE_RING
#define BEGE_RING 16
#endif
constexpr int kRing = BEGE_RING;
constexpr int kSearchThreads = 32 * 32;
#ifndef BEGE_STATS
#define BEGE_STATS 0       // 1: one CTA prints wait statistics of its service threads at the end (experiments only)
#endif
constexpr int kTmemCols = 256;
constexpr int kTmemColsDual = 512;
constexpr uint32_t kTmDelta = 0, kTmStat = 32, kTmTheta = 96, kTmStat1 = 192, kTmAB = 256;
__constant__ float2 c_wb[16][16];          // exp(2 pi i b r / 256): row b = the CTA-uniform part of pass 2's four-step factor;
                                           // rounded from fp64 (host, bege_plan_create)
constexpr int kSigPart = 128;              // Parseval partial sums per pair: 16 tiles x 8 warps (dual-stream search: two sets)

struct SearchArgs {
    CUtensorMap ring_map;                  // T' of all groups and ring slots as a 2-D fp32 tensor: (512, G * kRing * 256)
    const c2* bank; const c2* xseg; const float2* qseg; c2* ring; float* sigpart; bege_tail* rec; c2* zdbg;
    unsigned long long cap; unsigned long long* counter; unsigned long long* done1; unsigned long long* done2;
    int* abort_flag;
    uint64_t j0, nT, sig_pair0;
    uint32_t m0, nS, S;
    float k2, k2hi;
};

// shared-memory map of k_search (byte offsets from the 2048-byte aligned base)
template <int NI> struct SearchSmem {
    static constexpr uint32_t kTile = NI * 256 * 8;              // one column tile of a spectrum
    static constexpr uint32_t kWarpTile = kTile / 8;             // ... the words of one warp
    static constexpr uint32_t kXch = 16 * 17 * 8;                // padded private exchange region of a half-warp, [g][17]
    static constexpr int kNB = NI <= 14 ? 3 : 2;                 // 32 KiB row tiles of pass 2
    static constexpr uint32_t btile = 0;                         // [kNB] row tiles of pass 2 (swizzled: 1024-byte aligned)
    static constexpr uint32_t stream = btile + kNB * 32768;      // [2][8] streaming tile part of each A warp
    static constexpr uint32_t xch = stream + 2 * kTile;          // [2][16] exchange region of each A half-warp
    static constexpr uint32_t abar = xch + 32 * kXch;            // [16] mbarriers: streaming tile part of an A warp has arrived
    static constexpr uint32_t amb = abar + 128;                  // [kRing] mbarriers: tile of ring slot stored (8 A warps)
    static constexpr uint32_t bfull = amb + 8 * kRing;           // [kNB] mbarriers: row tile has arrived
    static constexpr uint32_t bempty = bfull + 24;               // [kNB] u32 counters (8-byte pitch): warps that have read a tile out
    static constexpr uint32_t pubit = bempty + 24;                               // [2] u32: next item of A team k to publish (claimed by atomicCAS)
    static constexpr uint32_t tmem = pubit + 8;                  // TMEM base address
    static constexpr uint32_t total = tmem + 8;
    static_assert(total + 2048 <= 232448, "shared memory of one SM");
};
// the stationary tile has its tensor-memory arrangement written out for bands that need 14 of the 16 row-blocks;
// other bands read it from global memory (L2) -- correct, not tuned
template <int NI> __host__ __device__ constexpr bool search_stat() { return NI == 14; }
template <int NI> constexpr int search_smem() { return (int)SearchSmem<NI>::total + 2048; }

// stage 1 of pass 1: v[I0 + 2 ip], v[I0 + 2 ip + 1] = conj(H) X for the row-block pair ip, acc += |.|^2 (packed);
// q0, q1: the stationary values.  SINGLE: the template streams, the segment is stationary; batched: the other way round
template <int I0, bool SINGLE, int IP> BEGE_D void products1(uint32_t stream_a, c2 q0, c2 q1, c2 (&v)[16], c2& acc)
{
    c2 s0, s1;
    lds128<IP * 512>(stream_a, s0, s1);
    const c2 r0 = SINGLE ? cmulc(q0, s0) : cmulc(s0, q0);
    const c2 r1 = SINGLE ? cmulc(q1, s1) : cmulc(s1, q1);
    v[I0 + 2 * IP] = r0; v[(I0 + 2 * IP + 1) & 15] = r1;
    acc = fma2(r0, r0, acc); acc = fma2(r1, r1, acc);
}
// ... stationary values streamed from tensor memory one pair at a time, double buffered (the load of pair 0 into qa
// was issued by the caller)
template <int I0, bool SINGLE, int IP = 0> BEGE_D void tm_products(uint32_t stream_a, uint32_t taddr, c2 (&v)[16], c2& acc, c2 (&qa)[2], c2 (&qb)[2])
{
    if constexpr (IP < 7) {
        c2 (&cur)[2] = (IP & 1) ? qb : qa;
        c2 (&nxt)[2] = (IP & 1) ? qa : qb;
        tmem_wait_ld(cur);
        if constexpr (IP + 1 < 7) tmem_ld4(taddr + 4 * (IP + 1), nxt);
        products1<I0, SINGLE, IP>(stream_a, cur[0], cur[1], v, acc);
        tm_products<I0, SINGLE, IP + 1>(stream_a, taddr, v, acc, qa, qb);
    }
}
// ... dual-stream search (SINGLE only): R = conj(W) X as above; instead of sum |R|^2 the two streams' own sums
// V1 = sum_k |W[k]|^2 |H1~[k]|^2 and V2 = sum_k |W[k]|^2 |L1~[k]|^2 (see k_search), packed in acc = (V1, V2).  Both are
// sums of non-negative terms: neither stream's variance is a difference of large numbers, however unequal their powers.
// The pairs (|H1~|^2, |L1~|^2) come from tensor memory like the stationary tile.
template <int I0, int IP = 0> BEGE_D void tm_products_dual(uint32_t stream_a, uint32_t tx, uint32_t tab, c2 (&v)[16], c2& acc,
                                                           c2 (&qa)[2], c2 (&qb)[2], c2 (&ra)[2], c2 (&rb)[2])
{
    if constexpr (IP < 7) {
        c2 (&cur)[2] = (IP & 1) ? qb : qa;
        c2 (&nxt)[2] = (IP & 1) ? qa : qb;
        c2 (&rcur)[2] = (IP & 1) ? rb : ra;
        c2 (&rnxt)[2] = (IP & 1) ? ra : rb;
        tmem_wait_ld(cur, rcur);
        if constexpr (IP + 1 < 7) { tmem_ld4(tx + 4 * (IP + 1), nxt); tmem_ld4(tab + 4 * (IP + 1), rnxt); }
        c2 s0, s1;
        lds128<IP * 512>(stream_a, s0, s1);
        const c2 r0 = cmulc(cur[0], s0), r1 = cmulc(cur[1], s1);
        v[I0 + 2 * IP] = r0; v[(I0 + 2 * IP + 1) & 15] = r1;
        acc = fma2(bc(fmaf(im(s0), im(s0), re(s0) * re(s0))), rcur[0], acc);
        acc = fma2(bc(fmaf(im(s1), im(s1), re(s1) * re(s1))), rcur[1], acc);
        tm_products_dual<I0, IP + 1>(stream_a, tx, tab, v, acc, qa, qb, ra, rb);
    }
}
// ... stationary values from global memory (bands that keep all 16 row-blocks)
template <int I0, int NI, bool SINGLE, int IP = 0> BEGE_D void gl_products(uint32_t stream_a, const ulonglong2* __restrict__ statg, c2 (&v)[16], c2& acc)
{
    if constexpr (IP < NI / 2) {
        const ulonglong2 q = __ldg(statg + IP * 32);
        products1<I0, SINGLE, IP>(stream_a, q.x, q.y, v, acc);
        gl_products<I0, NI, SINGLE, IP + 1>(stream_a, statg, v, acc);
    }
}

// DUAL (single-segment calls, 14 row-blocks): the dual-stream search of PAPER.md:155 -- x = H1 + i L1, REAL templates, so
// Re z and Im z are the two detectors' outputs.  Their variances are the Hermitian split of the product spectrum
// (eq.7): with H1~[k] = (X[k] + conj X[N-k])/2 and L1~[k] = (X[k] - conj X[N-k])/2i (the transforms of the
// two real streams) N^2 sigma_1^2 = V1 = sum_k |W[k]|^2 |H1~[k]|^2 and N^2 sigma_2^2 = V2 = sum_k |W[k]|^2 |L1~[k]|^2 --
// two per-tile partial sums of non-negative terms (k_dual_q tabulates |H1~|^2, |L1~|^2 per bin), no pairing of bins
// across tiles in the search and no cancellation when one detector is much louder than the other.  Output: per sample offset and stream the largest |rho|/sigma and its template
// (Table 3), by 64-bit atomicMax as in the max projection.
template <int I0, int NI, bool SINGLE, bool DBG, bool DUAL>
__global__ void __launch_bounds__(kSearchThreads, 1)
k_search(const __grid_constant__ SearchArgs A)
{
    constexpr bool STAT = search_stat<NI>();                 // stationary tile in tensor memory
    static_assert(!DUAL || (SINGLE && STAT && !DBG), "dual-stream search: single-segment calls on 14 row-blocks");
    using SM = SearchSmem<NI>;
    static_assert(NI % 2 == 0, "row-blocks are stored in pairs");
    extern __shared__ __align__(1024) unsigned char smem_dyn[];
    // the row tiles of pass 2 are addressed with xor arithmetic on bits 4 .. 10: 2048-byte aligned base
    const uint32_t sb = (smem_u32(smem_dyn) + 2047u) & ~2047u;
    unsigned char* const smem_raw = smem_dyn + (sb - smem_u32(smem_dyn));
    const int team = threadIdx.x >> 8;                       // 0, 1: A teams; 2, 3: B teams
    const int t = threadIdx.x & 255, warp = t >> 5, lane = t & 31;   // within the team
    const int b = blockIdx.x, grp = blockIdx.y, G = gridDim.y;
    constexpr uint64_t kTile = (uint64_t)NI * 256;           // elements
    int* const abort_flag = A.abort_flag;

    const uint32_t nS = SINGLE ? 1u : A.nS;
    const uint32_t nTg = A.nT > (uint64_t)grp ? (uint32_t)((A.nT - grp + G - 1) / G) : 0u;   // templates of this group
    const uint32_t n_items = nTg * nS;                      // < 2^31: the host splits larger searches
    c2* const myring = A.ring + (uint64_t)grp * kRing * kN;
    unsigned long long* const d1 = A.done1 + grp * kRing;    // one counter pair per ring slot: a count can only
    unsigned long long* const d2 = A.done2 + grp * kRing;    // come from the item that currently owns the slot
    // tile b of template (group-local index tj) / of segment ml
    auto tpl_tile = [&](uint32_t tj) { return A.bank + ((A.j0 + grp + (uint64_t)G * tj) * 16 + b) * kTile; };
    auto seg_tile = [&](uint32_t ml) { return A.xseg + ((uint64_t)(A.m0 + ml) * 16 + b) * kTile; };

    if (threadIdx.x == 0) {
        for (int i = 0; i < 16; ++i) mbar_init(sb + SM::abar + 8 * i, 1);
        for (int i = 0; i < kRing; ++i) mbar_init(sb + SM::amb + 8 * i, 8);
        for (int i = 0; i < SM::kNB; ++i) {
            mbar_init(sb + SM::bfull + 8 * i, 1);
            *reinterpret_cast<volatile uint32_t*>(smem_raw + SM::bempty + 8 * i) = 0;
        }
        reinterpret_cast<volatile uint32_t*>(smem_raw + SM::pubit)[0] = 0;
        reinterpret_cast<volatile uint32_t*>(smem_raw + SM::pubit)[1] = 1;
        fence_mbar_init();
    }
    if (threadIdx.x < 32) tmem_alloc<DUAL ? kTmemColsDual : kTmemCols>(sb + SM::tmem);
    tmem_fence_before_sync();
    __syncthreads();
    tmem_fence_after_sync();
    // this warp's lane quadrant of the tensor memory (lane field = bits 16 and up)
    const uint32_t tq = *reinterpret_cast<volatile uint32_t*>(smem_raw + SM::tmem) + ((uint32_t)(warp & 3) << 21);
    const uint32_t tq_a = tq + 32u * (uint32_t)(warp >> 2);  // pass 1: column block of this warp inside a table
    const uint32_t tq_s = tq_a + (team == 1 ? kTmStat1 : kTmStat);   // pass 1: this team's stationary tile
    // the stationary tile of pass 1 goes from global memory to this thread's TMEM columns (every A warp its own part)
    auto stat_to_tmem = [&](const c2* tile) {
        const ulonglong2* src = reinterpret_cast<const ulonglong2*>(tile) + tile_word(NI, 0, 0, t);
#pragma unroll
        for (int ip = 0; ip < NI / 2; ++ip) {
            const ulonglong2 q = __ldcg(src + ip * 32);
            const uint32_t r[4] = {(uint32_t)q.x, (uint32_t)(q.x >> 32), (uint32_t)q.y, (uint32_t)(q.y >> 32)};
            tmem_st4(tq_s + 4 * ip, r);
        }
        tmem_wait_st();
    };
    if (team == 0) {
        if (warp < 4) {                                      // delta_p, one copy per lane quadrant, B lane map
            const int a = (lane & 7) | ((lane >> 4) << 3);
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                uint32_t r[8];
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    double sn, cs;
                    sincospi(2.0 * (double)((a * (b + 16 * (4 * j + k))) & 4095) / 4096.0, &sn, &cs);
                    r[2 * k] = __float_as_uint((float)cs); r[2 * k + 1] = __float_as_uint((float)sn);
                }
                tmem_st8(tq + kTmDelta + 8 * j, r);
            }
        }
        {                                                    // theta^p, p = 1 .. 15 (+ one unused entry)
            const int c = t >> 4, g = t & 15;
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                uint32_t r[8];
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const int pp = 4 * j + k + 1;
                    double sn, cs;
                    sincospi(2.0 * (double)((pp * (256 * g + 16 * b + c)) & (kN - 1)) / (double)kN, &sn, &cs);
                    r[2 * k] = __float_as_uint((float)cs); r[2 * k + 1] = __float_as_uint((float)sn);
                }
                tmem_st8(tq_a + kTmTheta + 8 * j, r);
            }
        }
        if (DUAL && n_items > 0) {                           // (|H1~|^2, |L1~|^2) of this thread's 14 bins
            const ulonglong2* src = reinterpret_cast<const ulonglong2*>(A.qseg + ((uint64_t)A.m0 * 16 + b) * (uint64_t)(NI * 256)) + tile_word(NI, 0, 0, t);
#pragma unroll
            for (int ip = 0; ip < NI / 2; ++ip) {
                const ulonglong2 q = __ldcg(src + ip * 32);
                const uint32_t r[4] = {(uint32_t)q.x, (uint32_t)(q.x >> 32), (uint32_t)q.y, (uint32_t)(q.y >> 32)};
                tmem_st4(tq + kTmAB + 32u * (uint32_t)(warp >> 2) + 4 * ip, r);
            }
        }
        tmem_wait_st();
    }
    if (team < 2 && STAT && SINGLE && n_items > 0) stat_to_tmem(seg_tile(0));
    tmem_fence_before_sync();
    __syncthreads();
    tmem_fence_after_sync();

    if (team < 2 && !(BEGE_ABL & 16)) {
        // ================================================================ A: pass 1, items it = team (mod 2)
        const int c = t >> 4, g = t & 15;                    // column of the tile, lane of its half-warp (stage 2: g = p)
        const int aw = team * 8 + warp;                      // A warp of the CTA
        const uint32_t bar_w = sb + SM::abar + 8 * aw;
        const uint32_t wbuf = sb + SM::stream + aw * SM::kWarpTile;
        const uint32_t stream_a = wbuf + lane * 16;
        const uint32_t xa = sb + SM::xch + (uint32_t)(aw * 2 + (lane >> 4)) * SM::kXch;
        const uint32_t xw_a = xa + g * 136;                  // + 8 p:    element (g, p) of the half-warp's region
        const uint32_t xr_a = xa + g * 8;                    // + 136 gg: element (gg, p = g)
        constexpr uint32_t kWarpElems = SM::kWarpTile / 8;
        // streaming tile part of this warp: template `it` (single-segment calls) / segment ml (batched calls)
        auto stream_src = [&](uint32_t it, uint32_t ml) { return (SINGLE ? tpl_tile(it) : seg_tile(ml)) + (uint32_t)warp * kWarpElems; };
        const ulonglong2* statg = nullptr;                   // !STAT: the stationary tile in global memory
        if (n_items > 0) {
            if (!STAT && SINGLE) statg = reinterpret_cast<const ulonglong2*>(seg_tile(0)) + tile_word(NI, 0, 0, t);
            if (lane == 0 && (uint32_t)team < n_items && !(BEGE_ABL & 2)) {
                mbar_arrive_expect_tx(bar_w, SM::kWarpTile);
                bulk_load(wbuf, stream_src(team, (uint32_t)team % nS), SM::kWarpTile, bar_w, SINGLE ? policy_evict_first() : policy_evict_last());
            }
        }
        uint32_t nload = 0;                                  // tiles this warp has waited for so far
        uint32_t tj_prev = ~0u;
        // single-segment calls: item it + 2 is template tj + 2 of the group -- the streaming source and the slot of the
        // Parseval partial sums advance by constant strides (running pointers instead of 64-bit index arithmetic per item)
        const c2* src_run = stream_src(team + 2, 0);
        const uint64_t src_step = (uint64_t)G * 2 * 16 * kTile;
        float* sp_run = A.sigpart + ((A.j0 + grp + (uint64_t)G * team) * (uint64_t)A.S + A.m0 - A.sig_pair0) * (DUAL ? 2 * kSigPart : kSigPart) + b * 8 + warp;
        const uint64_t sp_step = (uint64_t)G * 2 * A.S * (DUAL ? 2 * kSigPart : kSigPart);
        // (template, segment) of the item, stepped without a division per item: batched calls have nS >= 2
        uint32_t tj_c = SINGLE ? 0u : (uint32_t)team / nS, ml_c = SINGLE ? 0u : (uint32_t)team % nS;
        for (uint32_t it = team; it < n_items; it += 2) {
            const uint32_t tj = SINGLE ? it : tj_c;
            const uint32_t ml = SINGLE ? 0u : ml_c;
            uint32_t ml_next = ml + 2;                       // segment of the team's next item
            if (!SINGLE && ml_next >= nS) { ml_next -= nS; ++tj_c; }
            ml_c = ml_next;
            const int slot = (int)(it % kRing);
            if (!SINGLE && tj != tj_prev) {                  // batched calls: this warp's part of the next template
                if (STAT) stat_to_tmem(tpl_tile(tj));
                else statg = reinterpret_cast<const ulonglong2*>(tpl_tile(tj)) + tile_word(NI, 0, 0, t);
                tj_prev = tj;
            }
            c2 qa[2], qb[2];                                 // TMEM staging (stationary values, then theta powers)
            c2 ra[2], rb[2];                                 // dual-stream search: staging of (|H1~|^2, |L1~|^2)
            if (STAT) tmem_ld4(tq_s, qa);
            if (DUAL) tmem_ld4(tq + kTmAB + 32u * (uint32_t)(warp >> 2), ra);
#if !(BEGE_ABL & 2)
            mbar_wait(bar_w, nload & 1, abort_flag);
#endif
            ++nload;
            c2 v[16];
            c2 acc = mk(0.f, 0.f);
#pragma unroll
            for (int r = 0; r < 16; ++r) if (r < I0 || r >= I0 + NI) v[r] = mk(0.f, 0.f);
            if constexpr (DUAL) tm_products_dual<I0>(stream_a, tq_s, tq + kTmAB + 32u * (uint32_t)(warp >> 2), v, acc, qa, qb, ra, rb);
            else if constexpr (STAT) tm_products<I0, SINGLE>(stream_a, tq_s, v, acc, qa, qb);
            else gl_products<I0, NI, SINGLE>(stream_a, statg, v, acc);
            tmem_ld4(tq_a + kTmTheta, qa);
            __syncwarp();                                    // the warp has read its part of the streaming tile:
            if (lane == 0 && !(BEGE_ABL & 2)) {              // order the part of this team's next item
                const uint32_t it2 = it + 2;
                if (it2 < n_items) {
                    mbar_arrive_expect_tx(bar_w, SM::kWarpTile);
                    bulk_load(wbuf, SINGLE ? src_run : stream_src(it2, ml_next), SM::kWarpTile, bar_w, SINGLE ? policy_evict_first() : policy_evict_last());
                }
            }
            if (SINGLE) src_run += src_step;
            fft16<+1, (BEGE_FUSE & 1) != 0>(v);
            tm_twiddle<1, 8>(tq_a + kTmTheta, v, qa, qb);    // v[p] *= theta^p, p = 1 .. 15
            sts16<8>(xw_a, v);
            const float sw = warp_sum32(DUAL ? re(acc) : re(acc) + im(acc));  // (includes the __syncwarp the exchange needs)
            const float pw = DUAL ? warp_sum32(im(acc)) : 0.f;               // dual-stream search: sw = V1, pw = V2
            __syncwarp();
            lds16<136>(xr_a, v);
            if (lane == 0) {
                float* sp = sp_run;
                if (!SINGLE) {
                    const uint64_t pr = (A.j0 + grp + (uint64_t)G * tj) * (uint64_t)A.S + (A.m0 + ml) - A.sig_pair0;
                    sp = A.sigpart + pr * (DUAL ? 2 * kSigPart : kSigPart) + b * 8 + warp;
                }
                sp[0] = sw;
                if (DUAL) sp[kSigPart] = pw;
            }
            if (SINGLE) sp_run += sp_step;
            // Ring slot free?  Item it - kRing must have been read out by pass 2 of all 16 CTAs of the group (done2).
            // All lanes load the one counter (a warp-uniform value keeps the warp converged through the wait; a wait
            // taken by lane 0 alone left the warp split in two for the rest of the item, profiles/r2_search_kernel.md); waiting warps
            // sleep 2 us between probes -- the ring is 16 items deep, and frequent probes of one L2 line slow its reds.
            if (!(BEGE_ABL & 1) && it >= (uint32_t)kRing) {
                const unsigned long long need = 16ull * (it / kRing);
                if (counter_load_acquire(d2 + slot) < need) counter_wait_ge(d2 + slot, need, abort_flag);
            }
            __syncwarp();                                    // exchange region free for the next item; ring slot free
            fft16<+1, (BEGE_FUSE & 1) != 0>(v);
            // T'[k1 = 16 b + c][n2 = p + 16 q], p = g: a half-warp stores 128 contiguous bytes per q
            c2* out = myring + (uint64_t)slot * kN + (uint32_t)(16 * b + c) * 256u + g;
#pragma unroll
            for (int q = 0; q < 16; ++q) {
                const c2 o = v[q];
                if (!(BEGE_ABL & 4) || re(o) == 1.2345e-30f) out[q * 16] = o;
            }
            // this warp's part of the tile is on its way: tell the publisher (thread 0 of the B team of the same parity)
            __syncwarp();
            if (lane == 0) {
                mbar_arrive(sb + SM::amb + 8 * slot);
                // the warp that completes the tile publishes it right away (pass 1 has the time: it is the one that waits
                // for ring slots; left to pass 2's service thread the publication sat for microseconds, and the ring's
                // round trip -- not the arithmetic -- set the pace)
                if (!(BEGE_ABL & (1 | 16)) && mbar_test_wait(sb + SM::amb + 8 * slot, (it / kRing) & 1)) {
                    uint32_t* const pub_it = reinterpret_cast<uint32_t*>(smem_raw + SM::pubit) + team;
                    const uint32_t first = *(volatile uint32_t*)pub_it;
                    uint32_t n = 0;
                    while (n < 4 && first + 2 * n < n_items &&
                           mbar_test_wait(sb + SM::amb + 8 * ((first + 2 * n) % kRing), ((first + 2 * n) / kRing) & 1)) ++n;
                    if (n && atomicCAS(pub_it, first, first + 2 * n) == first) {
                        fence_acq_rel_gpu();
                        for (uint32_t i = 0; i < n; ++i) counter_add_relaxed(d1 + (first + 2 * i) % kRing, 1ull);
                    }
                }
            }
        }
    } else if (team >= 2 && !(BEGE_ABL & 32)) {
        // ================================================================ B: pass 2, items ib = team - 2 (mod 2)
        const int kb = team - 2;
        // lane map: 8 values of a x 2 rows per hardware half-warp (conflict-free 64-bit accesses of the swizzled tile)
        const int a = (lane & 7) | ((lane >> 4) << 3);       // lane of the row's 256-point DFT
        const int rbit = (lane >> 3) & 1;
        const int hw = 2 * warp + rbit;                      // row of the row tile
        const int n2 = 16 * b + hw;
        constexpr uint32_t NB = SM::kNB;                     // item i uses tile buffer i % NB (both teams share the buffers)
        // The tile is T'[k1][16 rows] as the tensor copy leaves it: line k1 at 128 k1, its 16-byte chunk j at position
        // j ^ (k1 & 7) (128-byte swizzle).  Row hw owns slot (k1) = 128 k1 + 16 ((hw >> 1) ^ (k1 & 7)) + 8 (hw & 1) of
        // every line; after the loads the same 256 slots are the row's private exchange area.
        const uint32_t base_a = (uint32_t)a * 128u + ((uint32_t)(((hw >> 1) ^ a) & 7) << 4) + 8u * (uint32_t)(hw & 1);
        // ---- service state.  Thread 0 polls done1 (acquire) and issues the tensor copies; the gpu-scope fences -- about a
        // microsecond each while the SM has stores in flight -- are kept off its warp, whose progress paces the team: the
        // warp (1 + item mod 7) of the team takes them at the top of each item (once per seven items and warp).  Thread 0
        // takes them only inside its wait loop, when pass 2 is ahead of pass 1 and the team idles anyway (somebody must
        // publish then, or the group would stall).  The publication cursor lives in shared memory and is claimed by CAS.
        constexpr bool PUB = !(BEGE_ABL & (1 | 16));
        uint32_t* const pub_it = reinterpret_cast<uint32_t*>(smem_raw + SM::pubit) + kb;   // next item of A team kb to publish
        uint32_t ld_it = kb;                                 // next item of this team whose copy is to be issued
        unsigned long long d1v = 0; uint32_t d1v_it = ~0u;   // last acquired tiles-arrived counter and its item
        uint32_t nit = 0;                                    // items this team has started
        long long st_top = 0; unsigned st_ntop = 0, st_nmid = 0, st_spin = 0;
        // whenever all 8 warps of A team kb have stored their part of an item (mbarrier amb[slot]): ONE
        // fence.acq_rel.gpu, then done1[slot] += 1 (and, under the same fence, done2[free_slot] += 1)
        auto publish = [&](int free_slot) {
            uint32_t n = 0;
            const uint32_t first = *(volatile uint32_t*)pub_it;
            if (PUB) {
                while (n < 4 && first + 2 * n < n_items &&
                       mbar_test_wait(sb + SM::amb + 8 * ((first + 2 * n) % kRing), ((first + 2 * n) / kRing) & 1)) ++n;
                if (n && atomicCAS(pub_it, first, first + 2 * n) != first) n = 0;      // another thread of the team has them
            }
            if (n == 0 && free_slot < 0) return;
            fence_acq_rel_gpu();
            for (uint32_t i = 0; i < n; ++i) counter_add_relaxed(d1 + (first + 2 * i) % kRing, 1ull);
            if (free_slot >= 0) counter_add_relaxed(d2 + free_slot, 1ull);
        };
        // copy of item `it` of this team into its tile buffer, if the buffer has been read out (item it - NB, either
        // team) and all 16 tiles of the item are in the ring (d1, acquired: `ready`); non-blocking.  "Read out" is a
        // monotone count of warps (8 per use), not an mbarrier: this thread may look at a buffer whose use before last
        // (by a slow warp of its own team) is still going on, two phases away, where a parity test cannot tell.
        auto try_load = [&](uint32_t it, bool ready) {
            const uint32_t bf = it % NB, us = it / NB;
            if (us > 0 && smem_counter_load_acquire(sb + SM::bempty + 8 * bf) < 8 * us) return;
            if (!ready) return;
            if (!(BEGE_ABL & 8)) {
                fence_proxy_async_all();                     // the tile's generic reads and the acquired ring stores first
                mbar_arrive_expect_tx(sb + SM::bfull + 8 * bf, 32768);
                // box (32 floats = this CTA's 16 rows, 256 lines k1) of item (grp, slot)
                tma_load_2d(sb + SM::btile + bf * 32768, &A.ring_map, 32 * b, (int)(((uint32_t)grp * kRing + it % kRing) * 256u),
                            sb + SM::bfull + 8 * bf, policy_evict_first());
            }
            ld_it = it + 2;
        };
        uint32_t tj_c = SINGLE ? 0u : (uint32_t)kb / nS, ml_c = SINGLE ? 0u : (uint32_t)kb % nS;
        const float* sp_run = A.sigpart + ((A.j0 + grp + (uint64_t)G * kb) * (uint64_t)A.S + A.m0 - A.sig_pair0) * (DUAL ? 2 * kSigPart : kSigPart) + 8 * a;
        const uint64_t sp_step = (uint64_t)G * 2 * A.S * (DUAL ? 2 * kSigPart : kSigPart);
        for (uint32_t ib = kb; ib < n_items; ib += 2) {
            const int slot = (int)(ib % kRing);
            const uint32_t tj = SINGLE ? ib : tj_c;
            const uint32_t ml = SINGLE ? 0u : ml_c;
            if (!SINGLE) { ml_c += 2; if (ml_c >= nS) { ml_c -= nS; ++tj_c; } }
            const uint64_t jl = grp + (uint64_t)G * tj;
            const uint32_t buf = ib % NB, use = ib / NB;
            const uint32_t w0 = sb + SM::btile + buf * 32768 + base_a;   // + 2048 i: T[n2][k1 = a + 16 i]
            //   (w0 ^ cx(p)) + 2048 p:  exchange slot of element (a, p), slot index 16 p + (a ^ p)
            //   (w0 + 2048 a) ^ cx(aa): element (aa, p = a), with cx(j) = 128 j + 16 (j & 7)
            const uint32_t r0 = w0 + 2048u * (uint32_t)a;
            if (t == 0) {
                const unsigned long long target = 16ull * (ib / kRing + 1);
                const long long t0 = clock64();
                if (BEGE_STATS) { if (ld_it == ib) ++st_ntop; else ++st_nmid; }
                for (;;) {
                    if (BEGE_STATS) ++st_spin;
                    if (ld_it == ib) {                       // copy of this item not yet issued
                        publish(-1);
                        try_load(ib, (BEGE_ABL & 1) || counter_load_acquire(d1 + slot) >= target);
                    }
                    if (ld_it > ib && ((BEGE_ABL & 8) || mbar_test_wait(sb + SM::bfull + 8 * buf, use & 1))) break;
                    if (*(volatile int*)abort_flag) break;
                    if (clock64() - t0 > kSpinLimit) {
                        *(volatile int*)abort_flag = 1; break;
                    }
                    __nanosleep(40);
                }
                // The other seven warps wait for this thread at the team's named barrier below: blocked in hardware, they
                // take no issue slots from the working warps (a try_wait loop on the tile's mbarrier cost more
                // instructions per item than the item's arithmetic, profiles/r2_search_kernel.md).
                if (BEGE_STATS) st_top += clock64() - t0;
                // look at the counter of the team's next item now; the answer is used after the exchange
                if (!(BEGE_ABL & 1) && ib + 2 < n_items && ld_it == ib + 2) { d1v = counter_load_acquire(d1 + (ib + 2) % kRing); d1v_it = ib + 2; }
            }
            __syncwarp();
            bar_named(1 + kb, 256);                          // the other seven warps block here in hardware (no spinning)
            // the rows are in shared memory: the ring slot is free.  This item's fence duty: warp 1 + (nit mod 7)
            if (warp == 1 + (int)(nit % 7) && lane == 0) publish(slot);
            ++nit;
            c2 v[16];
            lds16<2048>(w0, v);
            const uint64_t pair = (A.j0 + jl) * (uint64_t)A.S + (A.m0 + ml);
            // Parseval partial sums of tile a: 8 warps, fixed order
            const float4* sp = reinterpret_cast<const float4*>(SINGLE ? sp_run : A.sigpart + (pair - A.sig_pair0) * (DUAL ? 2 * kSigPart : kSigPart) + 8 * a);
            if (SINGLE) sp_run += sp_step;
            const float4 s0 = __ldcg(sp), s1 = __ldcg(sp + 1);
            const float part = ((s0.x + s0.y) + (s0.z + s0.w)) + ((s1.x + s1.y) + (s1.z + s1.w));
            float ppart = 0.f;
            if (DUAL) {
                const float4 p0 = __ldcg(sp + kSigPart / 4), p1 = __ldcg(sp + kSigPart / 4 + 1);
                ppart = ((p0.x + p0.y) + (p0.z + p0.w)) + ((p1.x + p1.y) + (p1.z + p1.w));
            }
            c2 wa[2], wb[2];
            tmem_ld4(tq + kTmDelta, wa);
            // four-step factor wN^(16 b k1), k1 = a + 16 r: its CTA-uniform part w256^(b r) here, the rest in delta_p
#pragma unroll
            for (int r = 1; r < 16; ++r) { const float2 w = c_wb[b][r]; v[r] = cmulw(v[r], w.x, w.y); }
            const float sumR2 = row_sum16(part);
            const float sumP = DUAL ? row_sum16(ppart) : 0.f;
            fft16<+1, (BEGE_FUSE & 2) != 0>(v);
            if (t == 0 && ib + 2 < n_items && ld_it == ib + 2)   // first chance to bring in the team's next item
                try_load(ib + 2, (BEGE_ABL & 1) || (d1v_it == ib + 2 && d1v >= 16ull * ((ib + 2) / kRing + 1)));
            tm_twiddle<0, 8>(tq + kTmDelta, v, wa, wb);      // v[p] *= delta_p = wN^(16 b a) w256^(a p)
            __syncwarp();                                    // every lane of the row has its values in registers
#pragma unroll
            for (int p = 0; p < 16; ++p) sts64<0>((w0 ^ (uint32_t)(128 * p + 16 * (p & 7))) + 2048u * p, v[p]);
            __syncwarp();
#pragma unroll
            for (int aa = 0; aa < 16; ++aa) v[aa] = lds64<0>(r0 ^ (uint32_t)(128 * aa + 16 * (aa & 7)));
            fence_proxy_async_smem();                        // these generic accesses before the next tensor copy into the tile
            __syncwarp();
            if (lane == 0) smem_counter_add_release(sb + SM::bempty + 8 * buf, 1);
            if (t == 0 && ib + 2 < n_items && ld_it == ib + 2)   // bring in the team's next item while this one is finished
                try_load(ib + 2, (BEGE_ABL & 1) || (d1v_it == ib + 2 && d1v >= 16ull * ((ib + 2) / kRing + 1)));
            fft16<+1, (BEGE_FUSE & 2) != 0>(v);
            // lane a holds Z[n1 = a + 16 q]; lag n = 256 n1 + n2
            const float thr = A.k2 * sumR2;
            // dual-stream search: the two sums are N^2 sigma_1^2 = V1 for Re z (H1) and N^2 sigma_2^2 = V2 for Im z (L1)
            const float var1 = sumR2, var2 = sumP;
            const float thr1 = A.k2 * var1, thr2 = A.k2 * var2;
            bool any = false;
#pragma unroll
            for (int q = 0; q < 16; ++q) {
                const float zr = re(v[q]), zi = im(v[q]);
                if (DUAL) any |= (zr * zr > thr1) | (zi * zi > thr2);
                else any |= fmaf(zi, zi, zr * zr) > thr;
            }
            if (DBG) {
                const float invN = 1.0f / (float)kN;
#pragma unroll
                for (int q = 0; q < 16; ++q)
                    A.zdbg[(uint64_t)(a + 16 * q) * 256 + n2] = mul2(v[q], bc(invN));
            }
#if BEGE_ABL
            if (thr == -1.f)                                 // timing experiment only: never emit
#endif
            if (DUAL) {
                if (__any_sync(0xffffffffu, any)) {
                    // PAPER.md:221 Table 3: per sample offset and stream the largest |rho|/sigma and its template
                    unsigned long long* proj1 = reinterpret_cast<unsigned long long*>(A.rec);
                    unsigned long long* proj2 = proj1 + (uint64_t)A.S * kN;
                    const uint32_t lag0 = (uint32_t)(A.m0 + ml) * (uint32_t)kN + (uint32_t)(a * 256 + n2);
                    const unsigned long long idkey = (unsigned long long)(0xffffffffu - (uint32_t)(A.j0 + jl));
#pragma unroll
                    for (int q = 0; q < 16; ++q) {
                        const float zr = re(v[q]), zi = im(v[q]);
                        if (zr * zr > thr1 && var1 > 0.f)
                            atomicMax(proj1 + lag0 + 4096u * q, ((unsigned long long)__float_as_uint(sqrtf(zr * zr / var1)) << 32) | idkey);
                        if (zi * zi > thr2 && var2 > 0.f)
                            atomicMax(proj2 + lag0 + 4096u * q, ((unsigned long long)__float_as_uint(sqrtf(zi * zi / var2)) << 32) | idkey);
                    }
                }
            } else
            if (__any_sync(0xffffffffu, any)) {
                unsigned hits = 0;
                float mag[16];
#pragma unroll
                for (int q = 0; q < 16; ++q) {
                    const float zr = re(v[q]), zi = im(v[q]);
                    mag[q] = fmaf(zi, zi, zr * zr);
                    if (mag[q] > thr) hits |= 1u << q;
                }
                const float inv = 1.0f / sumR2;
                if (A.k2hi < 3.0e38f) {                      // band threshold: drop |z| >= k_hi sigma
                    const float thr_hi = A.k2hi * sumR2;
#pragma unroll
                    for (int q = 0; q < 16; ++q)
                        if (!(mag[q] < thr_hi)) hits &= ~(1u << q);
                }
                const uint32_t lag0 = (uint32_t)(A.m0 + ml) * (uint32_t)kN + (uint32_t)(a * 256 + n2);   // + 4096 q
                if (A.cap == ~0ull) {
                    // max projection: per sample offset the largest |z|/sigma over the bank and
                    // its template, race free: one 64-bit atomicMax on (snr bits, ~template_id); positive floats
                    // order like their bit patterns, equal values go to the smaller template id
                    unsigned long long* proj = reinterpret_cast<unsigned long long*>(A.rec);
#pragma unroll
                    for (int q = 0; q < 16; ++q) {
                        if (hits & (1u << q)) {
                            const float snr = sqrtf(mag[q] * inv);
                            atomicMax(proj + lag0 + 4096u * q, ((unsigned long long)__float_as_uint(snr) << 32) |
                                                                   (unsigned long long)(0xffffffffu - (uint32_t)(A.j0 + jl)));
                        }
                    }
                } else {
                    const int cnt = __popc(hits);
                    int incl = cnt;
#pragma unroll
                    for (int d = 1; d < 32; d <<= 1) {
                        const int o = __shfl_up_sync(0xffffffffu, incl, d);
                        if (lane >= d) incl += o;
                    }
                    const int total = __shfl_sync(0xffffffffu, incl, 31);
                    unsigned long long base = 0;
                    if (lane == 31) base = atomicAdd(A.counter, (unsigned long long)total);
                    base = __shfl_sync(0xffffffffu, base, 31);
                    unsigned long long slot_r = base + (unsigned long long)(incl - cnt);
#pragma unroll
                    for (int q = 0; q < 16; ++q) {
                        if (hits & (1u << q)) {
                            if (slot_r < A.cap) {
                                bege_tail r;
                                r.template_id = (uint32_t)(A.j0 + jl);
                                r.lag = lag0 + 4096u * q;
                                r.snr = sqrtf(mag[q] * inv);
                                A.rec[slot_r] = r;
                            }
                            ++slot_r;
                        }
                    }
                }
            }
        }
        if (BEGE_STATS && b == 3 && grp == 1 && t == 0)
            printf("B team %d: items %u, copies issued at the item top %u / ahead %u, top-loop cycles/item %lld, spins/item %u\n", kb, nit,
                   st_ntop, st_nmid, st_top / (long long)max(nit, 1u), st_spin / max(nit, 1u));
        if (t == 0) {                                        // tiles A team kb stores after this team's last copy
            publish(-1);
            for (;;) {
                const uint32_t nx = *(volatile uint32_t*)pub_it;
                if (!PUB || nx >= n_items) break;
                mbar_wait(sb + SM::amb + 8 * (nx % kRing), (nx / kRing) & 1, abort_flag);
                if (*(volatile int*)abort_flag) break;
                publish(-1);
            }
        }
    }
    // every warp is done with the tensor memory: give it back
    tmem_fence_before_sync();
    __syncthreads();
    if (threadIdx.x < 32) tmem_dealloc<DUAL ? kTmemColsDual : kTmemCols>(tq);
}

// sum of the 8 warp partial sums of a tile, in the order pass 2 uses
__host__ __device__ inline float tile_sum8(const float* w)
{
    return ((w[0] + w[1]) + (w[2] + w[3])) + ((w[4] + w[5]) + (w[6] + w[7]));
}

// sigma_jm = sqrt(sum of the 16 x 8 partial sums) / N
__global__ void k_sigma(const float* __restrict__ sigpart, float* __restrict__ sigma, uint64_t n)
{
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    // same order as pass 2 (tile_sum8, then row_sum16: xor 8, 4, 2, 1) so that sigma matches the search bit for bit
    float v[16];
    for (int a = 0; a < 16; ++a) v[a] = tile_sum8(sigpart + i * kSigPart + 8 * a);
    for (int d = 8; d >= 1; d >>= 1)
        for (int a = 0; a < d; ++a) v[a] = v[a] + v[a + d];
    sigma[i] = sqrtf(v[0]) / (float)kN;
}

// dual-stream search: per stored bin k of a segment spectrum X (x = H1 + i L1) the powers of the two real streams,
// Q[k] = (|H1~[k]|^2, |L1~[k]|^2) = (|X[k] + conj X[N-k]|^2, |X[k] - conj X[N-k]|^2) / 4, same tile layout as X.
// grid (16 tiles, segments), 256 threads.
__global__ void __launch_bounds__(256)
k_dual_q(const c2* __restrict__ xs, float2* __restrict__ q, int I0, int NI)
{
    const int t = threadIdx.x, b = blockIdx.x;
    const uint64_t m = blockIdx.y;
    const int c = t >> 4, g = t & 15;
    const c2* X = xs + m * (uint64_t)(16 * NI * 256);
    float2* Q = q + m * (uint64_t)(16 * NI * 256);
    for (int ii = 0; ii < NI; ++ii) {
        const uint32_t k = (uint32_t)(16 * b + c) + 256u * (uint32_t)(g + 16 * (ii + I0));
        const uint32_t km = ((uint32_t)kN - k) & (uint32_t)(kN - 1);
        const int bm = (int)((km & 255u) >> 4), cm = (int)(km & 15u), gm = (int)((km >> 8) & 15u), im_ = (int)(km >> 12) - I0;
        const size_t idx = (size_t)tile_word(NI, b, ii / 2, t) * 2 + (ii & 1);
        float2 val = make_float2(0.f, 0.f);
        if (im_ >= 0 && im_ < NI) {                          // (a mirror bin outside the stored row-blocks is out of band, as is k)
            const c2 a = X[idx], d = X[(size_t)tile_word(NI, bm, im_ / 2, 16 * cm + gm) * 2 + (im_ & 1)];
            const float sr = re(a) + re(d), si = im(a) - im(d);      // X[k] + conj X[N-k]
            const float dr = re(a) - re(d), di = im(a) + im(d);      // X[k] - conj X[N-k]
            val = make_float2(0.25f * (sr * sr + si * si), 0.25f * (dr * dr + di * di));
        }
        Q[idx] = val;
    }
}

// dual-stream search: sigma_1 = sqrt(V1)/N, sigma_2 = sqrt(V2)/N from the 2 x 128 partial sums of a pair
__global__ void k_sigma_dual(const float* __restrict__ sigpart, float* __restrict__ s1, float* __restrict__ s2, uint64_t n)
{
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float v[16], w[16];
    for (int a = 0; a < 16; ++a) { v[a] = tile_sum8(sigpart + i * 2 * kSigPart + 8 * a); w[a] = tile_sum8(sigpart + i * 2 * kSigPart + kSigPart + 8 * a); }
    for (int d = 8; d >= 1; d >>= 1)
        for (int a = 0; a < d; ++a) { v[a] = v[a] + v[a + d]; w[a] = w[a] + w[a + d]; }     // the order of row_sum16
    s1[i] = sqrtf(v[0]) / (float)kN;
    s2[i] = sqrtf(w[0]) / (float)kN;
}

// dual-stream search: offsets with a hit in both streams, and those whose templates' start frequencies differ by less
// than delta
__global__ void k_dual_coinc(const uint32_t* __restrict__ id1, const uint32_t* __restrict__ id2, const double* __restrict__ f0,
                             double delta, uint64_t n, unsigned long long* __restrict__ out)
{
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    bool sim = false, coi = false;
    if (i < n) {
        const uint32_t a = id1[i], b = id2[i];
        sim = a != 0xffffffffu && b != 0xffffffffu;
        coi = sim && fabs(f0[a] - f0[b]) < delta;
    }
    const unsigned ms = __ballot_sync(0xffffffffu, sim), mc = __ballot_sync(0xffffffffu, coi);
    if ((threadIdx.x & 31) == 0) {
        if (ms) atomicAdd(out, (unsigned long long)__popc(ms));
        if (mc) atomicAdd(out + 1, (unsigned long long)__popc(mc));
    }
}

}  // namespace bege

// =================================================================================================
// host side
// =================================================================================================
using namespace bege;

struct Slot { uint64_t off = 0, bytes = 0; void* own = nullptr; };

struct bege_plan {
    int device = 0;
    cudaStream_t stream = nullptr, side = nullptr;
    bool own_stream = false;
    uint32_t N = 0;
    double fs = 0, lo = 0, hi = 0;
    uint32_t klo = 0, khi = 0;
    int I0 = 0, NI = 16;
    int G = 0;                      // search groups (16 CTAs each), all co-resident
    int n_sm = 0;
    float2 *tw256 = nullptr, *twN = nullptr;
    d2* tw256d = nullptr;           // exp(2 pi i m / 256) in fp64 (bank generation)
    // workspace
    unsigned char* ws = nullptr; uint64_t ws_bytes = 0, bump = 0; bool user_ws = false;
    Slot s_bank, s_x, s_q, s_scratch, s_sig, s_rec, s_misc, s_par, s_tmp;
    bool bank_real = false, have_sigma_dual = false;
    std::vector<cudaEvent_t> ev_slice;
    uint64_t T = 0; uint32_t S = 0; double tau = 0; uint32_t L = 0;
    bool have_sigma = false;
    // pinned staging
    unsigned long long* h_count = nullptr;
    cudaEvent_t ev_a = nullptr, ev_b = nullptr, ev_done = nullptr;
    bool profiling = false;
    CUtensorMap ring_map{};          // the ring as a 2-D tensor (pass 2 fetches its row tiles with one tensor copy)
    void* ring_map_for = nullptr;   // ring address the map was encoded for
    void* l2_window = nullptr;      // ring region currently marked persisting in L2 (access policy window of the stream)
    size_t l2_limit_prev = 0; bool l2_limit_raised = false;  // device limit found before this plan raised it (first search)
    uint64_t max_items = ((1ull << 31) - 1) / 2;   // per group and launch (the kernel counts items in 32 bits)
    bege_stats stats{};
    std::string err;
};

// take the ring's persisting-L2 window off the plan's stream again (the stream may be the caller's).  Per search this
// touches the stream attribute only: no context-wide reset (it would evict other users' persisting lines and
// synchronise), no change of the device limit.
static void drop_l2_window(bege_plan* p)
{
    if (!p->l2_window || !p->stream) return;
    cudaStreamAttrValue av{};
    av.accessPolicyWindow.base_ptr = nullptr;
    av.accessPolicyWindow.num_bytes = 0;
    av.accessPolicyWindow.hitRatio = 0.f;
    av.accessPolicyWindow.hitProp = cudaAccessPropertyNormal;
    av.accessPolicyWindow.missProp = cudaAccessPropertyNormal;
    cudaStreamSetAttribute(p->stream, cudaStreamAttributeAccessPolicyWindow, &av);
    cudaGetLastError();
    p->l2_window = nullptr;
}
// every return path of a search, error returns included, leaves the caller's stream without the window
struct L2WindowGuard { bege_plan* p; ~L2WindowGuard() { drop_l2_window(p); } };

// the ring goes away (plan destroyed / workspace replaced): give its lines back to normal caching and put the device's
// persisting-L2 limit back to what it was before this plan raised it
static void release_l2(bege_plan* p)
{
    drop_l2_window(p);
    if (!p->l2_limit_raised) return;
    cudaCtxResetPersistingL2Cache();
    cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, p->l2_limit_prev);
    cudaGetLastError();
    p->l2_limit_raised = false;
}

static int fail(bege_plan* p, int code, const char* fmt, ...)
{
    if (p) {
        char buf[512];
        va_list ap; va_start(ap, fmt); vsnprintf(buf, sizeof buf, fmt, ap); va_end(ap);
        p->err = buf;
    }
    return code;
}
#define CU(p, call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return fail((p), BEGE_ECUDA, "%s: %s", #call, cudaGetErrorString(e_)); } while (0)

static uint64_t align_up(uint64_t v, uint64_t a) { return (v + a - 1) / a * a; }

// (re)size a slot: reuse if big enough; own memory if no user workspace, else bump-allocate from it
static int slot_get(bege_plan* p, Slot& s, uint64_t need, void** out)
{
    need = align_up(need ? need : 256, 256);
    if (!p->user_ws) {
        if (s.bytes < need) {
            if (s.own) { cudaFree(s.own); s.own = nullptr; s.bytes = 0; }
            cudaError_t e = cudaMalloc(&s.own, need);
            if (e != cudaSuccess) { cudaGetLastError(); return fail(p, BEGE_ENOMEM, "cudaMalloc(%llu) failed: %s", (unsigned long long)need, cudaGetErrorString(e)); }
            s.bytes = need;
        }
        *out = s.own;
        return BEGE_OK;
    }
    if (s.bytes < need) {
        const bool last = s.bytes && s.off + s.bytes == p->bump;
        if (last) p->bump = s.off;                       // grow the most recent slot in place
        else if (s.bytes) return fail(p, BEGE_ENOMEM, "workspace slot cannot grow (%llu -> %llu bytes); call bege_plan_set_workspace again",
                                      (unsigned long long)s.bytes, (unsigned long long)need);
        if (p->bump + need > p->ws_bytes)
            return fail(p, BEGE_ENOMEM, "workspace too small: need %llu more bytes, %llu of %llu used",
                        (unsigned long long)need, (unsigned long long)p->bump, (unsigned long long)p->ws_bytes);
        s.off = p->bump; s.bytes = need; p->bump += need;
    }
    *out = p->ws + s.off;
    return BEGE_OK;
}
static void slot_free(Slot& s) { if (s.own) cudaFree(s.own); s = Slot(); }

// Parseval partial sums of all pairs: one set of kSigPart per pair, two for the dual-stream search (which needs a bank
// of real templates).  Inside a caller's workspace the slot cannot grow later, so it takes the larger size at once
// (bege_plan_workspace_bytes counts that).
static uint64_t sig_bytes(const bege_plan* p)
{
    return p->T * p->S * (uint64_t)((p->bank_real || p->user_ws) ? 2 * kSigPart : kSigPart) * sizeof(float);
}

static uint64_t tpl_bytes(const bege_plan* p) { return (uint64_t)p->NI * 16 * 256 * sizeof(c2); }

static void count_launch(bege_plan* p, uint64_t n = 1) { p->stats.kernel_launches += n; }

// the instantiations of the search kernel: row-blocks kept (14 / 16), single-segment or batched, debug z output;
// plus the dual-stream variant (single-segment, 14 row-blocks)
static const void* search_variant(int NI, bool single, bool dbg, bool dual = false)
{
    if (dual) return (const void*)k_search<1, 14, true, false, true>;
    if (NI == 14) {
        if (single) return dbg ? (const void*)k_search<1, 14, true, true, false> : (const void*)k_search<1, 14, true, false, false>;
        return dbg ? (const void*)k_search<1, 14, false, true, false> : (const void*)k_search<1, 14, false, false, false>;
    }
    if (single) return dbg ? (const void*)k_search<0, 16, true, true, false> : (const void*)k_search<0, 16, true, false, false>;
    return dbg ? (const void*)k_search<0, 16, false, true, false> : (const void*)k_search<0, 16, false, false, false>;
}

extern "C" const char* bege_version(void) { return "bege 0.2 (sm_100a)"; }

extern "C" const char* bege_last_error(const bege_plan* p) { return p ? p->err.c_str() : "null plan"; }

extern "C" int bege_plan_create(bege_plan** out, uint32_t N, double fs, double lo, double hi, int device, void* stream)
{
    if (!out) return BEGE_EINVAL;
    if (N != (uint32_t)kN || !(fs > 0) || !(lo > 0) || !(hi > lo) || !(hi < 0.5 * fs)) return BEGE_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) { cudaGetLastError(); return BEGE_ECUDA; }
    bege_plan* p = new bege_plan();
    p->device = device; p->N = N; p->fs = fs; p->lo = lo; p->hi = hi;
    auto bail = [&](int code) { bege_plan_destroy(p); return code; };
    if (cudaSetDevice(device) != cudaSuccess) return bail(BEGE_ECUDA);
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return bail(BEGE_ECUDA);
    if (prop.major < 10) return bail(BEGE_ECUDA);              // sm_100a code only
    p->n_sm = prop.multiProcessorCount;
    // a caller on the legacy default stream passes cudaStreamLegacy (handle 0 would be indistinguishable from NULL)
    if (stream) p->stream = (cudaStream_t)stream;
    else { if (cudaStreamCreateWithFlags(&p->stream, cudaStreamNonBlocking) != cudaSuccess) return bail(BEGE_ECUDA); p->own_stream = true; }
    if (cudaStreamCreateWithFlags(&p->side, cudaStreamNonBlocking) != cudaSuccess) return bail(BEGE_ECUDA);
    if (cudaEventCreate(&p->ev_a) != cudaSuccess || cudaEventCreate(&p->ev_b) != cudaSuccess ||
        cudaEventCreateWithFlags(&p->ev_done, cudaEventDisableTiming) != cudaSuccess) return bail(BEGE_ECUDA);
    if (cudaMallocHost(&p->h_count, 8 * (2 + kMaxSlices)) != cudaSuccess) return bail(BEGE_ECUDA);

    // band in bins, inclusive edges: klo = ceil(lo N/fs), khi = floor(hi N/fs)
    const double df = fs / N;
    p->klo = (uint32_t)ceil(lo / df - 1e-9);
    p->khi = (uint32_t)floor(hi / df + 1e-9);
    // kept row-blocks: block i holds rows k2 = g + 16 i, g < 16, i.e. bins [4096 i, 4096 i + 4095]; a block is
    // kept when it (or its mirror at N - k) contains an in-band bin
    bool keep[16];
    int first = 16, last = -1;
    for (int i = 0; i < 16; ++i) {
        const uint32_t a = 4096u * i, b = a + 4095u;
        auto hit = [&](uint32_t l, uint32_t h) { return !(b < l || a > h); };
        keep[i] = hit(p->klo, p->khi) || hit(N - p->khi, N - p->klo);
        if (keep[i]) { if (i < first) first = i; last = i; }
    }
    if (first == 1 && last == 14) { p->I0 = 1; p->NI = 14; } else { p->I0 = 0; p->NI = 16; }

    std::vector<float2> w256(256), wN((size_t)256 * 256);
    for (int pp = 0; pp < 16; ++pp)
        for (int g = 0; g < 16; ++g) {
            const double a = 2.0 * M_PI * (double)(g * pp) / 256.0;
            w256[pp * 16 + g] = make_float2((float)cos(a), (float)sin(a));
        }
    for (int n2 = 0; n2 < 256; ++n2)
        for (int k1 = 0; k1 < 256; ++k1) {
            const double a = 2.0 * M_PI * (double)(n2 * k1) / (double)N;
            wN[(size_t)n2 * 256 + k1] = make_float2((float)cos(a), (float)sin(a));
        }
    {
        std::vector<d2> t256(256);
        for (int m = 0; m < 256; ++m) { t256[m].x = cos(2.0 * M_PI * m / 256.0); t256[m].y = sin(2.0 * M_PI * m / 256.0); }
        if (cudaMalloc(&p->tw256d, 256 * sizeof(d2)) != cudaSuccess) return bail(BEGE_ENOMEM);
        if (cudaMemcpy(p->tw256d, t256.data(), 256 * sizeof(d2), cudaMemcpyHostToDevice) != cudaSuccess) return bail(BEGE_ECUDA);
        if (cudaFuncSetAttribute(k_bank_gen64, cudaFuncAttributeMaxDynamicSharedMemorySize, kBankSmem) != cudaSuccess) return bail(BEGE_ECUDA);
    }
    {   // exp(2 pi i b r / 256) for the search kernel's CTA-uniform twiddles (constant memory of this device's context)
        std::vector<float2> tb(256);
        for (int bb = 0; bb < 16; ++bb)
            for (int r = 0; r < 16; ++r) {
                const double a = 2.0 * M_PI * (double)((bb * r) & 255) / 256.0;
                tb[bb * 16 + r] = make_float2((float)cos(a), (float)sin(a));
            }
        if (cudaMemcpyToSymbol(c_wb, tb.data(), sizeof(float2) * 256) != cudaSuccess) return bail(BEGE_ECUDA);
    }
    if (cudaMalloc(&p->tw256, w256.size() * sizeof(float2)) != cudaSuccess ||
        cudaMalloc(&p->twN, wN.size() * sizeof(float2)) != cudaSuccess) return bail(BEGE_ENOMEM);
    if (cudaMemcpy(p->tw256, w256.data(), w256.size() * sizeof(float2), cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMemcpy(p->twN, wN.data(), wN.size() * sizeof(float2), cudaMemcpyHostToDevice) != cudaSuccess) return bail(BEGE_ECUDA);

    // the search kernel needs all its CTAs co-resident (groups hand over through global counters)
    int occ = 0;
    for (int i = 0; i < 9; ++i) {
        const void* f = i == 8 ? search_variant(14, true, false, true) : search_variant(i >> 2 ? 16 : 14, (i >> 1) & 1, i & 1);
        const int sm = (i < 8 && (i >> 2)) ? search_smem<16>() : search_smem<14>();
        if (cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, sm) != cudaSuccess) return bail(BEGE_ECUDA);
        int o = 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o, f, kSearchThreads, sm) != cudaSuccess) return bail(BEGE_ECUDA);
        occ = i ? std::min(occ, o) : o;
    }
    int coop = 0;
    cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, device);
    p->G = std::min(kMaxGroups, occ * prop.multiProcessorCount / 16);
    if (!coop || p->G < 1) return bail(BEGE_ECUDA);
    p->stats.hbm_bytes_per_template = tpl_bytes(p);
    *out = p;
    return BEGE_OK;
}

extern "C" void bege_plan_destroy(bege_plan* p)
{
    if (!p) return;
    cudaSetDevice(p->device);
    if (p->stream) cudaStreamSynchronize(p->stream);
    release_l2(p);
    if (p->side) { cudaStreamSynchronize(p->side); cudaStreamDestroy(p->side); }
    if (p->own_stream && p->stream) cudaStreamDestroy(p->stream);
    for (Slot* s : {&p->s_bank, &p->s_x, &p->s_q, &p->s_scratch, &p->s_sig, &p->s_rec, &p->s_misc, &p->s_par, &p->s_tmp}) slot_free(*s);
    if (p->tw256) cudaFree(p->tw256);
    if (p->twN) cudaFree(p->twN);
    if (p->tw256d) cudaFree(p->tw256d);
    if (p->h_count) cudaFreeHost(p->h_count);
    if (p->ev_a) cudaEventDestroy(p->ev_a);
    if (p->ev_b) cudaEventDestroy(p->ev_b);
    if (p->ev_done) cudaEventDestroy(p->ev_done);
    for (cudaEvent_t e : p->ev_slice) cudaEventDestroy(e);
    delete p;
}

// one region serves the fp32 staging of the segment transform (kBatch segments), the window table of the bank
// generation and the search ring (G groups x kRing items)
static uint64_t scratch_bytes(const bege_plan* p)
{
    return std::max<uint64_t>((uint64_t)kBatch * kN * sizeof(c2), (uint64_t)p->G * kRing * kN * sizeof(c2));
}

extern "C" int bege_plan_workspace_bytes(const bege_plan* p, uint64_t T, uint32_t S, uint64_t cap, uint64_t* bytes)
{
    if (!p || !bytes) return BEGE_EINVAL;
    auto al = [](uint64_t v) { return align_up(v ? v : 256, 256); };
    uint64_t b = 0;
    b += al(T * tpl_bytes(p));                         // bank
    b += al(T * 16);                                   // template parameters (f0, fdot)
    b += al((uint64_t)S * tpl_bytes(p));               // segment spectra
    b += al((uint64_t)S * tpl_bytes(p));               // (|H1~|^2, |L1~|^2) per stored bin (dual-stream search)
    b += al(scratch_bytes(p));                          // four-step staging (stays in L2)
    b += al(T * S * 2 * kSigPart * sizeof(float));     // Parseval partial sums (two sets in the dual-stream search)
    b += al(std::max<uint64_t>(cap * sizeof(bege_tail), (uint64_t)S * kN * 16));  // records / max-projection array(s)
    b += al(kMiscHdr + (uint64_t)S * kN * sizeof(c2)); // counters + raw segment staging
    b += al(std::max<uint64_t>(std::max<uint64_t>(2 * T * S * sizeof(float), (uint64_t)S * kN * 16), kN * sizeof(c2) + 512));   // sigma / projection / debug output
    *bytes = b + 4096;
    return BEGE_OK;
}

extern "C" int bege_plan_set_workspace(bege_plan* p, void* dev_ptr, uint64_t bytes)
{
    if (!p) return BEGE_EINVAL;
    if (dev_ptr && ((uintptr_t)dev_ptr & 255)) return fail(p, BEGE_EINVAL, "workspace must be 256-byte aligned");
    CU(p, cudaSetDevice(p->device));
    CU(p, cudaStreamSynchronize(p->stream));
    release_l2(p);
    for (Slot* s : {&p->s_bank, &p->s_x, &p->s_q, &p->s_scratch, &p->s_sig, &p->s_rec, &p->s_misc, &p->s_par, &p->s_tmp}) slot_free(*s);
    p->ws = (unsigned char*)dev_ptr; p->ws_bytes = dev_ptr ? bytes : 0; p->bump = 0; p->user_ws = dev_ptr != nullptr;
    p->T = 0; p->S = 0; p->have_sigma = false; p->have_sigma_dual = false; p->bank_real = false;
    return BEGE_OK;
}

static int bank_generate_impl(bege_plan* p, const double* f0, const double* fdot, uint64_t T, double tau, int real_tpl);

extern "C" int bege_bank_generate(bege_plan* p, const double* f0, const double* fdot, uint64_t T, double tau)
{
    return bank_generate_impl(p, f0, fdot, T, tau, 0);
}

extern "C" int bege_bank_generate_real(bege_plan* p, const double* f0, const double* fdot, uint64_t T, double tau)
{
    return bank_generate_impl(p, f0, fdot, T, tau, 1);
}

extern "C" int bege_bank_generate_real_symmetric(bege_plan* p, const double* f0, const double* fdot, uint64_t T, double tau)
{
    return bank_generate_impl(p, f0, fdot, T, tau, 2);
}

// real_tpl: 0 complex chirp, 1 its real part, 2 the time-symmetric real template (see k_bank_gen64)
static int bank_generate_impl(bege_plan* p, const double* f0, const double* fdot, uint64_t T, double tau, int real_tpl)
{
    if (!p) return BEGE_EINVAL;
    if (!f0 || !fdot || T == 0 || T > 0xffffffffull) return fail(p, BEGE_EINVAL, "bad bank arguments");
    const long Ll = lround(tau * p->fs);
    if (Ll < 2 || Ll > kN / 16) return fail(p, BEGE_EINVAL, "tau*fs = %ld outside [2, %d]", Ll, kN / 16);
    CU(p, cudaSetDevice(p->device));
    void *bank, *par, *scr;
    int rc;
    if ((rc = slot_get(p, p->s_bank, T * tpl_bytes(p), &bank))) return rc;
    if ((rc = slot_get(p, p->s_par, T * 16, &par))) return rc;
    if ((rc = slot_get(p, p->s_scratch, scratch_bytes(p), &scr))) return rc;
    p->T = 0; p->have_sigma = false; p->have_sigma_dual = false;
    double* d_f0 = (double*)par; double* d_fd = d_f0 + T;
    CU(p, cudaMemcpyAsync(d_f0, f0, T * sizeof(double), cudaMemcpyHostToDevice, p->stream));
    CU(p, cudaMemcpyAsync(d_fd, fdot, T * sizeof(double), cudaMemcpyHostToDevice, p->stream));
    // unit L2 norm: ||h||^2 = sum_n hann_L[n]^2 (the phase factor has modulus 1); the window goes to the device
    // already divided by the norm
    const uint32_t L = (uint32_t)Ll;
    std::vector<double> hann(L);
    double n2 = 0;
    for (uint32_t n = 0; n < L; ++n) { hann[n] = 0.5 - 0.5 * cos(2.0 * M_PI * n / (double)(L - 1)); n2 += hann[n] * hann[n]; }
    const double inv_norm = 1.0 / sqrt(n2);
    for (uint32_t n = 0; n < L; ++n) hann[n] *= inv_norm;
    double* d_hann = (double*)scr;                           // the scratch region is free outside a search
    CU(p, cudaMemcpyAsync(d_hann, hann.data(), L * sizeof(double), cudaMemcpyHostToDevice, p->stream));
    const uint64_t stride = tpl_bytes(p) / sizeof(c2);
    const unsigned ctas = (unsigned)std::min<uint64_t>(T, (uint64_t)p->n_sm);
    k_bank_gen64<<<ctas, 256, kBankSmem, p->stream>>>(d_f0, d_fd, T, p->fs, L, d_hann, p->tw256d, (float2*)bank, stride, p->I0, p->NI, real_tpl);
    count_launch(p);
    CU(p, cudaStreamSynchronize(p->stream));                 // `hann` (pageable) must outlive its copy
    CU(p, cudaGetLastError());
    CU(p, cudaStreamSynchronize(p->stream));
    p->T = T; p->tau = tau; p->L = L; p->bank_real = real_tpl != 0;
    return BEGE_OK;
}

extern "C" int bege_segment_load(bege_plan* p, const float* x, uint32_t S)
{
    if (!p) return BEGE_EINVAL;
    if (!x || S == 0 || (uint64_t)S * kN > 0xffffffffull) return fail(p, BEGE_EINVAL, "bad segment arguments");
    CU(p, cudaSetDevice(p->device));
    void *xs, *misc, *scr;
    int rc;
    if ((rc = slot_get(p, p->s_x, (uint64_t)S * tpl_bytes(p), &xs))) return rc;
    if ((rc = slot_get(p, p->s_misc, kMiscHdr + (uint64_t)S * kN * sizeof(c2), &misc))) return rc;
    if ((rc = slot_get(p, p->s_scratch, scratch_bytes(p), &scr))) return rc;
    p->S = 0; p->have_sigma = false; p->have_sigma_dual = false;
    c2* raw = (c2*)((unsigned char*)misc + kMiscHdr);
    cudaPointerAttributes at;
    cudaError_t e = cudaPointerGetAttributes(&at, x);
    if (e != cudaSuccess) { cudaGetLastError(); at.type = cudaMemoryTypeUnregistered; }
    const bool on_dev = at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
    CU(p, cudaMemcpyAsync(raw, x, (uint64_t)S * kN * sizeof(c2), on_dev ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, p->stream));
    const uint64_t stride = tpl_bytes(p) / sizeof(c2);
    for (uint32_t m0 = 0; m0 < S; m0 += kBatch) {
        const unsigned nb = std::min<uint32_t>(kBatch, S - m0);
        k_fwd_rows_data<<<dim3(16, nb), 256, 0, p->stream>>>(raw + (uint64_t)m0 * kN, p->tw256, p->twN, (c2*)scr);
        k_fwd_cols<true><<<dim3(16, nb), 256, 0, p->stream>>>((const c2*)scr, (c2*)xs + m0 * stride, stride, p->I0, p->NI, p->tw256, p->klo, p->khi);
        count_launch(p, 2);
    }
    {   // powers of the two real streams for the dual-stream search: two floats per stored bin, same layout
        void* q;
        if ((rc = slot_get(p, p->s_q, (uint64_t)S * tpl_bytes(p), &q))) return rc;
        k_dual_q<<<dim3(16, S), 256, 0, p->stream>>>((const c2*)xs, (float2*)q, p->I0, p->NI);
        count_launch(p);
    }
    CU(p, cudaGetLastError());
    CU(p, cudaStreamSynchronize(p->stream));
    p->S = S;
    return BEGE_OK;
}

// keep the ring's lines resident in L2 for the duration of a search: they are rewritten every few microseconds and
// must not be written back to HBM in between (ncu: 31 KB of write-back per correlation without this).  Best effort,
// errors ignored.  The window is taken off the stream again when the search returns (the stream may be the caller's).
static void set_l2_window(bege_plan* p, void* ring)
{
    if (p->l2_window == ring) return;
    const size_t bytes = (size_t)p->G * kRing * kN * sizeof(c2);
    if (!p->l2_limit_raised) {                               // once per plan, and only if the limit has to grow
        size_t cur = 0;
        if (cudaDeviceGetLimit(&cur, cudaLimitPersistingL2CacheSize) == cudaSuccess && cur < bytes &&
            cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, bytes) == cudaSuccess) { p->l2_limit_prev = cur; p->l2_limit_raised = true; }
    }
    cudaStreamAttrValue av{};
    av.accessPolicyWindow.base_ptr = ring;
    av.accessPolicyWindow.num_bytes = bytes;
    av.accessPolicyWindow.hitRatio = 1.0f;
    av.accessPolicyWindow.hitProp = cudaAccessPropertyPersisting;
    av.accessPolicyWindow.missProp = cudaAccessPropertyStreaming;
    cudaStreamSetAttribute(p->stream, cudaStreamAttributeAccessPolicyWindow, &av);
    cudaGetLastError();
    p->l2_window = ring;
}

// The ring as pass 2 sees it: a 2-D fp32 tensor, inner dimension the 256 complex n2 of a line (512 floats), outer
// dimension the lines k1 of all groups and ring slots; box = this CTA's 16 rows (32 floats = 128 bytes) x 256 lines,
// 128-byte swizzle.  Encoded by the driver (cuTensorMapEncodeTiled, looked up at run time: no link to libcuda).
static int make_ring_map(bege_plan* p, void* ring)
{
    if (p->ring_map_for == ring) return BEGE_OK;
    typedef CUresult (*encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static encode_fn encode = nullptr;
    if (!encode) {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult qr;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr) != cudaSuccess || !fn ||
            qr != cudaDriverEntryPointSuccess) { cudaGetLastError(); return fail(p, BEGE_ECUDA, "cuTensorMapEncodeTiled not available"); }
        encode = (encode_fn)fn;
    }
    const cuuint64_t gdim[2] = {512, (cuuint64_t)p->G * kRing * 256};
    const cuuint64_t gstride[1] = {2048};                    // bytes between lines
    const cuuint32_t box[2] = {32, 256};
    const cuuint32_t estride[2] = {1, 1};
    const CUresult r = encode(&p->ring_map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, ring, gdim, gstride, box, estride,
                              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(p, BEGE_ECUDA, "cuTensorMapEncodeTiled failed (%d)", (int)r);
    p->ring_map_for = ring;
    return BEGE_OK;
}

// one cooperative launch of the persistent search kernel over templates [j0, j0 + nT) x segments [m0, m0 + nS)
static int launch_search(bege_plan* p, const c2* bank, const c2* xs, c2* ring, float* sig, uint64_t sig_pair0, float k2, float k2hi,
                         bege_tail* rec, uint64_t cap, unsigned char* misc, c2* zdbg, uint64_t j0, uint64_t nT, uint32_t m0,
                         uint32_t nS, bool first = true, const float2* qseg = nullptr)
{
    const bool dual = qseg != nullptr;
    // the first launch of a search also clears the record counter, the abort flag and the hit counters
    CU(p, cudaMemsetAsync(misc + (first ? 0 : kOffDone1), 0, kMiscHdr - (first ? 0 : kOffDone1), p->stream));
    const int G = (int)std::min<uint64_t>((uint64_t)p->G, nT);
    const dim3 grid(16, G);
    set_l2_window(p, (void*)ring);
    { const int rc = make_ring_map(p, (void*)ring); if (rc) return rc; }
    SearchArgs a{};
    a.ring_map = p->ring_map;
    a.bank = bank; a.xseg = xs; a.qseg = qseg; a.ring = ring; a.sigpart = sig; a.rec = rec; a.zdbg = zdbg;
    a.cap = cap; a.counter = (unsigned long long*)(misc + kOffCounter); a.abort_flag = (int*)(misc + kOffAbort);
    a.done1 = (unsigned long long*)(misc + kOffDone1); a.done2 = (unsigned long long*)(misc + kOffDone2);
    a.j0 = j0; a.nT = nT; a.sig_pair0 = sig_pair0; a.m0 = m0; a.nS = nS; a.S = p->S; a.k2 = k2; a.k2hi = k2hi;
    void* args[] = {&a};
    const void* f = search_variant(p->NI, nS == 1, zdbg != nullptr, dual);
    const int smem = p->NI == 14 ? search_smem<14>() : search_smem<16>();
    if (p->profiling) cudaEventRecord(p->ev_a, p->stream);
    CU(p, cudaLaunchCooperativeKernel(f, grid, dim3(kSearchThreads), args, smem, p->stream));
    count_launch(p);
    if (p->profiling) {
        cudaEventRecord(p->ev_b, p->stream);
        CU(p, cudaEventSynchronize(p->ev_b));
        float ms = 0; cudaEventElapsedTime(&ms, p->ev_a, p->ev_b);
        p->stats.fused_kernel_ms += ms; p->stats.fused_kernel_launches += 1;
    }
    return BEGE_OK;
}

static int check_abort(bege_plan* p, unsigned char* misc)
{
    int flag = 0;
    CU(p, cudaMemcpyAsync(&flag, misc + kOffAbort, sizeof flag, cudaMemcpyDeviceToHost, p->stream));
    CU(p, cudaStreamSynchronize(p->stream));
    if (flag) return fail(p, BEGE_ECUDA, "search pipeline timed out waiting on a group counter");
    return BEGE_OK;
}

// template slices of one search: each slice is one launch of the persistent kernel.  Several slices let the copy of
// slice i's records to the host (side stream) run while slice i + 1 is searched (only the tails cross
// the bus, and they must not hold up the search); one slice never exceeds the kernel's 32-bit item count per group.
static uint64_t slice_templates(const bege_plan* p, bool want_overlap)
{
    const uint64_t maxT = std::max<uint64_t>(1, p->max_items / p->S) * (uint64_t)p->G;
    uint64_t n = 1;
    if (want_overlap) n = std::min<uint64_t>(kMaxSlices, std::max<uint64_t>(1, p->T * p->S / kSliceMinCorr));
    uint64_t per = (p->T + n - 1) / n;
    per = (per + p->G - 1) / p->G * p->G;            // whole rounds of the groups
    return std::min(per, maxT);
}

static int search_impl(bege_plan* p, float k_sigma, float k_hi, bege_tail* tails_out, uint64_t cap, uint64_t* n_tails)
{
    if (!p) return BEGE_EINVAL;
    if (!n_tails || (cap && !tails_out) || !(k_sigma >= 0.f) || !(k_hi >= k_sigma) || cap == ~0ull)
        return fail(p, BEGE_EINVAL, "bad search arguments");
    if (!p->T || !p->S) return fail(p, BEGE_ESTATE, "bege_search needs a generated bank and loaded segments");
    CU(p, cudaSetDevice(p->device));
    L2WindowGuard l2_guard{p};
    void *sig, *rec, *misc, *scr, *bank, *xs;
    int rc;
    if ((rc = slot_get(p, p->s_sig, sig_bytes(p), &sig))) return rc;
    if ((rc = slot_get(p, p->s_rec, cap * sizeof(bege_tail), &rec))) return rc;
    if ((rc = slot_get(p, p->s_misc, kMiscHdr, &misc))) return rc;
    if ((rc = slot_get(p, p->s_scratch, scratch_bytes(p), &scr))) return rc;
    if ((rc = slot_get(p, p->s_bank, 0, &bank))) return rc;
    if ((rc = slot_get(p, p->s_x, 0, &xs))) return rc;
    unsigned long long* counter = (unsigned long long*)misc;
    const uint64_t per = slice_templates(p, cap > 0);
    const uint64_t nsl = (p->T + per - 1) / per;
    // all slices are enqueued at once; after each one its running record count goes to pinned host memory
    std::vector<cudaEvent_t>& ev = p->ev_slice;
    while (ev.size() < std::min<uint64_t>(nsl, kMaxSlices)) {
        cudaEvent_t e; CU(p, cudaEventCreateWithFlags(&e, cudaEventDisableTiming)); ev.push_back(e);
    }
    const bool overlap = nsl <= (uint64_t)kMaxSlices;      // more slices only for > 2^31-item searches: no overlap then
    for (uint64_t i = 0; i < nsl; ++i) {
        const uint64_t jj = i * per;
        if ((rc = launch_search(p, (const c2*)bank, (const c2*)xs, (c2*)scr, (float*)sig, 0, k_sigma * k_sigma, k_hi * k_hi,
                                (bege_tail*)rec, cap, (unsigned char*)misc, nullptr, jj, std::min(per, p->T - jj), 0, p->S,
                                i == 0))) return rc;
        if (overlap) {
            CU(p, cudaMemcpyAsync(p->h_count + 2 + i, counter, sizeof(unsigned long long), cudaMemcpyDeviceToHost, p->stream));
            CU(p, cudaEventRecord(ev[i], p->stream));
        }
    }
    CU(p, cudaGetLastError());
    CU(p, cudaMemcpyAsync(p->h_count, counter, sizeof(unsigned long long), cudaMemcpyDeviceToHost, p->stream));
    CU(p, cudaMemcpyAsync(p->h_count + 1, (unsigned char*)misc + kOffAbort, sizeof(int), cudaMemcpyDeviceToHost, p->stream));
    // only the tails cross PCIe: the records of slice i are complete once slice i has finished, and are
    // copied on the side stream while the main stream searches slice i + 1
    uint64_t copied = 0;
    if (overlap && cap) {
        for (uint64_t i = 0; i < nsl; ++i) {
            CU(p, cudaEventSynchronize(ev[i]));
            const uint64_t upto = std::min<uint64_t>(p->h_count[2 + i], cap);
            if (upto > copied) {
                CU(p, cudaMemcpyAsync(tails_out + copied, (bege_tail*)rec + copied, (upto - copied) * sizeof(bege_tail),
                                      cudaMemcpyDeviceToHost, p->side));
                copied = upto;
            }
        }
    }
    CU(p, cudaStreamSynchronize(p->stream));
    drop_l2_window(p);
    if (*(volatile int*)(p->h_count + 1)) return fail(p, BEGE_ECUDA, "search pipeline timed out waiting on a group counter");
    const uint64_t total = *p->h_count;
    const uint64_t ncopy = std::min<uint64_t>(total, cap);
    if (ncopy > copied)
        CU(p, cudaMemcpyAsync(tails_out + copied, (bege_tail*)rec + copied, (ncopy - copied) * sizeof(bege_tail),
                              cudaMemcpyDeviceToHost, p->side));
    CU(p, cudaStreamSynchronize(p->side));
    p->stats.correlations += p->T * p->S;
    p->have_sigma = true; p->have_sigma_dual = false;
    *n_tails = total;
    if (total > cap) return fail(p, BEGE_EOVERFLOW, "%llu tails exceed cap %llu", (unsigned long long)total, (unsigned long long)cap);
    return BEGE_OK;
}


extern "C" int bege_search(bege_plan* p, float k_sigma, bege_tail* tails_out, uint64_t cap, uint64_t* n_tails)
{
    return search_impl(p, k_sigma, INFINITY, tails_out, cap, n_tails);
}

extern "C" int bege_search_band(bege_plan* p, float k_lo, float k_hi, bege_tail* tails_out, uint64_t cap, uint64_t* n_tails)
{
    return search_impl(p, k_lo, k_hi, tails_out, cap, n_tails);
}

// max projection: unpack (snr bits, ~template_id) keys into the two output arrays and count the offsets that hold a tail
__global__ void k_proj_decode(const unsigned long long* __restrict__ proj, float* __restrict__ snr, uint32_t* __restrict__ id,
                              unsigned long long* __restrict__ hits, uint64_t n)
{
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    bool hit = false;
    if (i < n) {
        const unsigned long long key = proj[i];
        hit = key != 0ull;
        snr[i] = hit ? __uint_as_float((uint32_t)(key >> 32)) : 0.f;
        id[i] = hit ? 0xffffffffu - (uint32_t)key : 0xffffffffu;
    }
    const unsigned m = __ballot_sync(0xffffffffu, hit);
    if ((threadIdx.x & 31) == 0 && m) atomicAdd(hits, (unsigned long long)__popc(m));
}

extern "C" int bege_search_maxproj(bege_plan* p, float k_sigma, float* snr_out, uint32_t* id_out, uint64_t* n_hits)
{
    if (!p) return BEGE_EINVAL;
    if (!snr_out || !id_out || !(k_sigma >= 0.f)) return fail(p, BEGE_EINVAL, "bad search arguments");
    if (!p->T || !p->S) return fail(p, BEGE_ESTATE, "bege_search_maxproj needs a generated bank and loaded segments");
    CU(p, cudaSetDevice(p->device));
    L2WindowGuard l2_guard{p};
    void *sig, *proj, *misc, *scr, *bank, *xs, *tmp;
    int rc;
    const uint64_t n = (uint64_t)p->S * kN;
    if ((rc = slot_get(p, p->s_sig, sig_bytes(p), &sig))) return rc;
    if ((rc = slot_get(p, p->s_rec, n * sizeof(unsigned long long), &proj))) return rc;
    if ((rc = slot_get(p, p->s_misc, kMiscHdr, &misc))) return rc;
    if ((rc = slot_get(p, p->s_scratch, scratch_bytes(p), &scr))) return rc;
    if ((rc = slot_get(p, p->s_tmp, n * 8, &tmp))) return rc;
    if ((rc = slot_get(p, p->s_bank, 0, &bank))) return rc;
    if ((rc = slot_get(p, p->s_x, 0, &xs))) return rc;
    CU(p, cudaMemsetAsync(proj, 0, n * sizeof(unsigned long long), p->stream));
    const uint64_t per = slice_templates(p, false);
    for (uint64_t jj = 0; jj < p->T; jj += per) {
        // cap = ~0 switches the kernel's epilogue from appending records to the projection array passed as `rec`
        if ((rc = launch_search(p, (const c2*)bank, (const c2*)xs, (c2*)scr, (float*)sig, 0, k_sigma * k_sigma, INFINITY,
                                (bege_tail*)proj, ~0ull, (unsigned char*)misc, nullptr, jj, std::min(per, p->T - jj), 0, p->S,
                                jj == 0))) return rc;
    }
    CU(p, cudaGetLastError());
    float* d_snr = (float*)tmp; uint32_t* d_id = (uint32_t*)(d_snr + n);
    unsigned long long* d_hits = (unsigned long long*)((unsigned char*)misc + kOffHits);      // cleared by the first launch
    k_proj_decode<<<(unsigned)((n + 255) / 256), 256, 0, p->stream>>>((const unsigned long long*)proj, d_snr, d_id, d_hits, n);
    count_launch(p);
    CU(p, cudaMemcpyAsync(snr_out, d_snr, n * sizeof(float), cudaMemcpyDeviceToHost, p->stream));
    CU(p, cudaMemcpyAsync(id_out, d_id, n * sizeof(uint32_t), cudaMemcpyDeviceToHost, p->stream));
    CU(p, cudaMemcpyAsync(p->h_count, d_hits, sizeof(unsigned long long), cudaMemcpyDeviceToHost, p->stream));
    rc = check_abort(p, (unsigned char*)misc);      // synchronises the stream
    drop_l2_window(p);
    if (rc) return rc;
    p->stats.correlations += p->T * p->S;
    p->have_sigma = true; p->have_sigma_dual = false;
    if (n_hits) *n_hits = *p->h_count;
    return BEGE_OK;
}

extern "C" int bege_search_dual(bege_plan* p, float k_sigma, float* snr1, uint32_t* id1, float* snr2, uint32_t* id2,
                                double delta_hz, uint64_t* n_simultaneous, uint64_t* n_coincident)
{
    if (!p) return BEGE_EINVAL;
    if (!snr1 || !id1 || !snr2 || !id2 || !(k_sigma >= 0.f)) return fail(p, BEGE_EINVAL, "bad search arguments");
    if (!p->T || !p->S) return fail(p, BEGE_ESTATE, "bege_search_dual needs a generated bank and loaded segments");
    if (!p->bank_real) return fail(p, BEGE_ESTATE, "bege_search_dual needs a bank of real templates (bege_bank_generate_real)");
    if (p->NI != 14) return fail(p, BEGE_EINVAL, "bege_search_dual supports bands inside bins [4096, 61440) only");
    CU(p, cudaSetDevice(p->device));
    L2WindowGuard l2_guard{p};
    void *sig, *proj, *misc, *scr, *bank, *xs, *q, *tmp, *par;
    int rc;
    const uint64_t n = (uint64_t)p->S * kN;
    if ((rc = slot_get(p, p->s_sig, sig_bytes(p), &sig))) return rc;
    if ((rc = slot_get(p, p->s_rec, 2 * n * sizeof(unsigned long long), &proj))) return rc;
    if ((rc = slot_get(p, p->s_misc, kMiscHdr, &misc))) return rc;
    if ((rc = slot_get(p, p->s_scratch, scratch_bytes(p), &scr))) return rc;
    if ((rc = slot_get(p, p->s_tmp, 2 * n * 8, &tmp))) return rc;
    if ((rc = slot_get(p, p->s_bank, 0, &bank))) return rc;
    if ((rc = slot_get(p, p->s_x, 0, &xs))) return rc;
    if ((rc = slot_get(p, p->s_q, 0, &q))) return rc;
    if ((rc = slot_get(p, p->s_par, 0, &par))) return rc;
    p->have_sigma = false; p->have_sigma_dual = false;
    CU(p, cudaMemsetAsync(proj, 0, 2 * n * sizeof(unsigned long long), p->stream));
    const uint64_t maxT = std::max<uint64_t>(1, p->max_items) * (uint64_t)p->G;
    bool first = true;
    // the stationary operand of a single-segment launch is the segment (and its Q): one launch (group) per segment
    for (uint32_t m = 0; m < p->S; ++m)
        for (uint64_t jj = 0; jj < p->T; jj += maxT) {
            if ((rc = launch_search(p, (const c2*)bank, (const c2*)xs, (c2*)scr, (float*)sig, 0, k_sigma * k_sigma, INFINITY,
                                    (bege_tail*)proj, ~0ull, (unsigned char*)misc, nullptr, jj, std::min(maxT, p->T - jj), m, 1,
                                    first, (const float2*)q))) return rc;
            first = false;
        }
    CU(p, cudaGetLastError());
    float* d_snr1 = (float*)tmp; uint32_t* d_id1 = (uint32_t*)(d_snr1 + n);
    float* d_snr2 = (float*)(d_id1 + n); uint32_t* d_id2 = (uint32_t*)(d_snr2 + n);
    unsigned long long* d_cnt = (unsigned long long*)((unsigned char*)misc + kOffHits);      // hits1, hits2, simultaneous, coincident
    CU(p, cudaMemsetAsync(d_cnt, 0, 4 * sizeof(unsigned long long), p->stream));
    const unsigned nb = (unsigned)((n + 255) / 256);
    k_proj_decode<<<nb, 256, 0, p->stream>>>((const unsigned long long*)proj, d_snr1, d_id1, d_cnt, n);
    k_proj_decode<<<nb, 256, 0, p->stream>>>((const unsigned long long*)proj + n, d_snr2, d_id2, d_cnt + 1, n);
    k_dual_coinc<<<nb, 256, 0, p->stream>>>(d_id1, d_id2, (const double*)par, delta_hz, n, d_cnt + 2);
    count_launch(p, 3);
    CU(p, cudaMemcpyAsync(snr1, d_snr1, n * sizeof(float), cudaMemcpyDeviceToHost, p->stream));
    CU(p, cudaMemcpyAsync(id1, d_id1, n * sizeof(uint32_t), cudaMemcpyDeviceToHost, p->stream));
    CU(p, cudaMemcpyAsync(snr2, d_snr2, n * sizeof(float), cudaMemcpyDeviceToHost, p->stream));
    CU(p, cudaMemcpyAsync(id2, d_id2, n * sizeof(uint32_t), cudaMemcpyDeviceToHost, p->stream));
    CU(p, cudaMemcpyAsync(p->h_count + 2, d_cnt, 4 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, p->stream));
    rc = check_abort(p, (unsigned char*)misc);      // synchronises the stream
    drop_l2_window(p);
    if (rc) return rc;
    p->stats.correlations += p->T * p->S;
    p->have_sigma_dual = true;
    if (n_simultaneous) *n_simultaneous = p->h_count[4];
    if (n_coincident) *n_coincident = p->h_count[5];
    return BEGE_OK;
}

extern "C" int bege_get_sigma_dual(bege_plan* p, float* sigma1_out, float* sigma2_out)
{
    if (!p || !sigma1_out || !sigma2_out) return BEGE_EINVAL;
    if (!p->have_sigma_dual) return fail(p, BEGE_ESTATE, "bege_get_sigma_dual needs a completed bege_search_dual");
    CU(p, cudaSetDevice(p->device));
    const uint64_t n = p->T * p->S;
    if (n == 0) return fail(p, BEGE_ESTATE, "no bank / segments loaded");
    void *sig, *tmp;
    int rc;
    if ((rc = slot_get(p, p->s_sig, 0, &sig))) return rc;
    if ((rc = slot_get(p, p->s_tmp, 2 * n * sizeof(float), &tmp))) return rc;
    k_sigma_dual<<<(unsigned)((n + 255) / 256), 256, 0, p->stream>>>((const float*)sig, (float*)tmp, (float*)tmp + n, n);
    count_launch(p);
    CU(p, cudaMemcpyAsync(sigma1_out, tmp, n * sizeof(float), cudaMemcpyDeviceToHost, p->stream));
    CU(p, cudaMemcpyAsync(sigma2_out, (float*)tmp + n, n * sizeof(float), cudaMemcpyDeviceToHost, p->stream));
    CU(p, cudaStreamSynchronize(p->stream));
    return BEGE_OK;
}

extern "C" int bege_get_sigma(bege_plan* p, float* sigma_out)
{
    if (!p || !sigma_out) return BEGE_EINVAL;
    if (!p->have_sigma) return fail(p, BEGE_ESTATE, "bege_get_sigma needs a completed bege_search");
    CU(p, cudaSetDevice(p->device));
    const uint64_t n = p->T * p->S;
    if (n == 0) return fail(p, BEGE_ESTATE, "no bank / segments loaded");
    void *sig, *tmp;
    int rc;
    if ((rc = slot_get(p, p->s_sig, 0, &sig))) return rc;
    if ((rc = slot_get(p, p->s_tmp, n * sizeof(float), &tmp))) return rc;
    k_sigma<<<(unsigned)((n + 255) / 256), 256, 0, p->stream>>>((const float*)sig, (float*)tmp, n);
    count_launch(p);
    CU(p, cudaMemcpyAsync(sigma_out, tmp, n * sizeof(float), cudaMemcpyDeviceToHost, p->stream));
    CU(p, cudaStreamSynchronize(p->stream));
    return BEGE_OK;
}

extern "C" int bege_debug_correlate(bege_plan* p, uint64_t j, uint32_t m, float* z_out, float* sigma_out)
{
    if (!p || !z_out) return BEGE_EINVAL;
    if (!p->T || !p->S) return fail(p, BEGE_ESTATE, "needs a bank and segments");
    if (j >= p->T || m >= p->S) return fail(p, BEGE_EINVAL, "pair (%llu, %u) out of range", (unsigned long long)j, m);
    CU(p, cudaSetDevice(p->device));
    L2WindowGuard l2_guard{p};
    void *scr, *bank, *xs, *misc, *tmp;
    int rc;
    if ((rc = slot_get(p, p->s_scratch, scratch_bytes(p), &scr))) return rc;
    if ((rc = slot_get(p, p->s_misc, kMiscHdr, &misc))) return rc;
    if ((rc = slot_get(p, p->s_tmp, kN * sizeof(c2) + 512, &tmp))) return rc;
    if ((rc = slot_get(p, p->s_bank, 0, &bank))) return rc;
    if ((rc = slot_get(p, p->s_x, 0, &xs))) return rc;
    c2* zd = (c2*)tmp;
    float* sg = (float*)((unsigned char*)tmp + kN * sizeof(c2));     // private partial sums of this one pair
    const bool prof = p->profiling; p->profiling = false;
    // sig_pair0 = this pair's index, so that its partial sums land on sg[0..127]
    rc = launch_search(p, (const c2*)bank, (const c2*)xs, (c2*)scr, sg, j * p->S + m, 1e30f, INFINITY, nullptr, 0,
                       (unsigned char*)misc, zd, j, 1, m, 1);
    p->profiling = prof;
    if (!rc) rc = check_abort(p, (unsigned char*)misc);
    drop_l2_window(p);
    if (rc) return rc;
    float part[kSigPart];
    CU(p, cudaMemcpyAsync(z_out, zd, kN * sizeof(c2), cudaMemcpyDeviceToHost, p->stream));
    CU(p, cudaMemcpyAsync(part, sg, sizeof part, cudaMemcpyDeviceToHost, p->stream));
    CU(p, cudaStreamSynchronize(p->stream));
    if (sigma_out) {
        float v[16];
        for (int a = 0; a < 16; ++a) v[a] = tile_sum8(part + 8 * a);
        for (int d = 8; d >= 1; d >>= 1) for (int a = 0; a < d; ++a) v[a] = v[a] + v[a + d];
        *sigma_out = sqrtf(v[0]) / (float)kN;
    }
    return BEGE_OK;
}

extern "C" int bege_debug_set_max_items(bege_plan* p, uint64_t max_items)
{
    if (!p) return BEGE_EINVAL;
    if (max_items == 0 || max_items > ((1ull << 31) - 1) / 2) return fail(p, BEGE_EINVAL, "max_items outside [1, 2^30)");
    p->max_items = max_items;
    return BEGE_OK;
}

// tile layout -> natural order, on the host (debug only)
static void untile(const bege_plan* p, const std::vector<float2>& tile, float* out)
{
    memset(out, 0, sizeof(float) * 2 * kN);
    for (int b = 0; b < 16; ++b)
        for (int ii = 0; ii < p->NI; ++ii)
            for (int c = 0; c < 16; ++c)
                for (int g = 0; g < 16; ++g) {
                    const float2 v = tile[(size_t)tile_word(p->NI, b, ii / 2, 16 * c + g) * 2 + (ii & 1)];
                    const size_t k = (size_t)(16 * b + c) + 256 * (size_t)(g + 16 * (ii + p->I0));
                    out[2 * k] = v.x; out[2 * k + 1] = v.y;
                }
}

extern "C" int bege_debug_template_spectrum(bege_plan* p, uint64_t j, float* H_out)
{
    if (!p || !H_out) return BEGE_EINVAL;
    if (j >= p->T) return fail(p, BEGE_EINVAL, "template %llu out of range", (unsigned long long)j);
    CU(p, cudaSetDevice(p->device));
    void* bank; slot_get(p, p->s_bank, 0, &bank);
    std::vector<float2> tile(tpl_bytes(p) / sizeof(float2));
    CU(p, cudaMemcpyAsync(tile.data(), (unsigned char*)bank + j * tpl_bytes(p), tpl_bytes(p), cudaMemcpyDeviceToHost, p->stream));
    CU(p, cudaStreamSynchronize(p->stream));
    untile(p, tile, H_out);
    return BEGE_OK;
}

extern "C" int bege_debug_segment_spectrum(bege_plan* p, uint32_t m, float* X_out)
{
    if (!p || !X_out) return BEGE_EINVAL;
    if (m >= p->S) return fail(p, BEGE_EINVAL, "segment %u out of range", m);
    CU(p, cudaSetDevice(p->device));
    void* xs; slot_get(p, p->s_x, 0, &xs);
    std::vector<float2> tile(tpl_bytes(p) / sizeof(float2));
    CU(p, cudaMemcpyAsync(tile.data(), (unsigned char*)xs + (uint64_t)m * tpl_bytes(p), tpl_bytes(p), cudaMemcpyDeviceToHost, p->stream));
    CU(p, cudaStreamSynchronize(p->stream));
    untile(p, tile, X_out);
    return BEGE_OK;
}

extern "C" int bege_plan_set_profiling(bege_plan* p, int on) { if (!p) return BEGE_EINVAL; p->profiling = on != 0; return BEGE_OK; }
extern "C" int bege_plan_get_stats(const bege_plan* p, bege_stats* out) { if (!p || !out) return BEGE_EINVAL; *out = p->stats; return BEGE_OK; }
extern "C" int bege_plan_reset_stats(bege_plan* p)
{
    if (!p) return BEGE_EINVAL;
    const uint64_t keep = p->stats.hbm_bytes_per_template;
    p->stats = bege_stats{}; p->stats.hbm_bytes_per_template = keep;
    return BEGE_OK;
}

// ------------------------------------------------------------------------------------------------
// bege_segment_spectrum_static: the band-limited forward transform of a few segments (a2, PAPER.md:155 step i) for
// callers that must not allocate device memory -- no plan, no workspace, no cudaMalloc / cudaFree anywhere below.
//
// The four-step transform needs somewhere to keep the row transforms G between its two kernels, and its twiddle
// tables.  bege_segment_load takes both from the plan's (allocated) memory; here they live in the three file-scope
// __device__ arrays that follow.  They are part of the library image, so every GPU on which the library is used
// carries them (2.5 MiB) from the moment the module is loaded there until the process exits.
//
// In host code the NAMES of these arrays are host-side shadow symbols, not device addresses, and must never be handed
// to a kernel.  static_setup() asks the runtime for the real addresses (cudaGetSymbolAddress, once per device, with that
// device current) and only those go into launches.
constexpr uint32_t kStaticMaxSeg = BEGE_STATIC_MAX_SEGMENTS;
static __device__ __align__(256) c2     g_static_G[(size_t)kStaticMaxSeg * kN];   // step A -> step B staging, 2 MiB
static __device__ __align__(256) float2 g_static_tw256[256];                      // exp(2 pi i g p / 256) at [16 p + g]
static __device__ __align__(256) float2 g_static_twN[kN];                         // exp(2 pi i nl k1 / N) at [256 nl + k1]

// fills the two twiddle tables in place (fp64 angles in units of pi, one rounding to fp32 -- the plan's tables are made
// the same way on the host).  Device code may name the arrays directly.  grid 256, 256 thr.
__global__ void __launch_bounds__(256) k_static_tables()
{
    const int t = threadIdx.x, r = blockIdx.x;
    double s, c;
    sincospi(2.0 * (double)(r * t) / (double)kN, &s, &c);
    g_static_twN[r * 256 + t] = make_float2((float)c, (float)s);
    if (r == 0) {
        sincospi(2.0 * (double)((t >> 4) * (t & 15)) / 256.0, &s, &c);
        g_static_tw256[t] = make_float2((float)c, (float)s);
    }
}

// step B of the forward transform as in k_fwd_cols<true>, but the masked spectrum leaves in NATURAL order
// (out[m N + k], all 16 row-blocks) so that the caller needs to know nothing of the tile layout.  The 16 columns of a
// tile are 16 consecutive bins of every row k2: the results go through shared memory once more so that each half-warp
// stores one full 128-byte line.  grid (16 tiles, n_segments), 256 thr.
__global__ void __launch_bounds__(256)
k_fwd_cols_natural(const c2* __restrict__ G, c2* __restrict__ out, const float2* __restrict__ tw256, uint32_t klo, uint32_t khi)
{
    __shared__ c2 sm[256 * 17];                    // first the 16 private 256-word exchange regions, then [k2][c] padded to 17
    const int t = threadIdx.x, b = blockIdx.x;
    const uint64_t m = blockIdx.y;
    const int c = t >> 4, g = t & 15;
    float2 w1[16];
    load_w1(w1, tw256, g);
    const c2* in = G + m * (uint64_t)kN + (uint64_t)b * 4096;
    c2 v[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) v[i] = in[(i * 16 + c) * 16 + g];
    hw_fft256<-1>(v, w1, sm + c * 256, g);         // lane g now holds X[k1 + 256 k2], k1 = 16 b + c, k2 = g + 16 q, in v[q]
    __syncthreads();                               // every half-warp is done with its exchange region
    const uint32_t k1 = 16 * b + c;
#pragma unroll
    for (int q = 0; q < 16; ++q) {
        const uint32_t k = k1 + 256u * (uint32_t)(g + 16 * q);
        const uint32_t kk = k < (uint32_t)kN / 2 ? k : (uint32_t)kN - k;
        sm[(g + 16 * q) * 17 + c] = (kk < klo || kk > khi) ? mk(0.f, 0.f) : v[q];
    }
    __syncthreads();
    c2* o = out + m * (uint64_t)kN + 16 * b;
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        const int k2 = 16 * i + c;                 // here the half-warp index picks the row and the lane the column
        o[256 * k2 + g] = sm[k2 * 17 + g];
    }
}

namespace {
struct StaticDev { bool ready = false; c2* G = nullptr; float2 *tw256 = nullptr, *twN = nullptr; };
constexpr int kStaticMaxDev = 64;
StaticDev g_static_dev[kStaticMaxDev];
std::mutex g_static_mu;

int static_fail(char* errbuf, uint64_t errbuf_len, int code, const char* fmt, ...)
{
    if (errbuf && errbuf_len) {
        va_list ap; va_start(ap, fmt); vsnprintf(errbuf, (size_t)errbuf_len, fmt, ap); va_end(ap);
    }
    return code;
}

// One-time set-up of `device` (already current): resolve the device addresses of the static arrays, fill the tables,
// wait for that to finish.  Returns a cudaError_t and the name of the step that failed.
cudaError_t static_setup(StaticDev& d, cudaStream_t st, const char** what)
{
    cudaError_t e;
    *what = "cudaGetSymbolAddress(g_static_G)";
    if ((e = cudaGetSymbolAddress((void**)&d.G, g_static_G)) != cudaSuccess) return e;
    *what = "cudaGetSymbolAddress(g_static_tw256)";
    if ((e = cudaGetSymbolAddress((void**)&d.tw256, g_static_tw256)) != cudaSuccess) return e;
    *what = "cudaGetSymbolAddress(g_static_twN)";
    if ((e = cudaGetSymbolAddress((void**)&d.twN, g_static_twN)) != cudaSuccess) return e;
    *what = "k_static_tables";
    k_static_tables<<<256, 256, 0, st>>>();
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    *what = "cudaStreamSynchronize (set-up)";
    if ((e = cudaStreamSynchronize(st)) != cudaSuccess) return e;   // later calls may come on other streams
    d.ready = true;
    return cudaSuccess;
}
}  // namespace

extern "C" int bege_segment_spectrum_static(int device, void* cuda_stream, double fs, double lo, double hi, const float* x_dev,
                                            uint32_t n_segments, float* X_out_dev, char* errbuf, uint64_t errbuf_len)
{
    if (errbuf && errbuf_len) errbuf[0] = 0;
    // argument checks first: none of them needs a device
    if (!(fs > 0) || !(lo > 0) || !(hi > lo) || !(hi < 0.5 * fs))
        return static_fail(errbuf, errbuf_len, BEGE_EINVAL, "band must satisfy 0 < band_lo_hz < band_hi_hz < fs/2");
    if (n_segments == 0) return static_fail(errbuf, errbuf_len, BEGE_EINVAL, "n_segments is 0");
    if (n_segments > kStaticMaxSeg)
        return static_fail(errbuf, errbuf_len, BEGE_EINVAL,
                           "n_segments = %u exceeds BEGE_STATIC_MAX_SEGMENTS = %u: the built-in staging array holds no more; "
                           "split the call or use a plan (bege_segment_load)", n_segments, kStaticMaxSeg);
    if (!x_dev || !X_out_dev) return static_fail(errbuf, errbuf_len, BEGE_EINVAL, "x_dev_c64 / X_out_dev_c64 is NULL");
    if (x_dev == X_out_dev) return static_fail(errbuf, errbuf_len, BEGE_EINVAL, "in-place transform is not supported");
    if (device < 0 || device >= kStaticMaxDev) return static_fail(errbuf, errbuf_len, BEGE_EINVAL, "device %d outside [0, %d)", device, kStaticMaxDev);
#define CUS(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { cudaGetLastError(); \
        return static_fail(errbuf, errbuf_len, BEGE_ECUDA, "%s: %s", #call, cudaGetErrorString(e_)); } } while (0)
    CUS(cudaSetDevice(device));
    for (const void* ptr : {(const void*)x_dev, (const void*)X_out_dev}) {
        cudaPointerAttributes at;
        if (cudaPointerGetAttributes(&at, ptr) != cudaSuccess || !(at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged)) {
            cudaGetLastError();
            return static_fail(errbuf, errbuf_len, BEGE_EINVAL, "%s must be device memory", ptr == (const void*)x_dev ? "x_dev_c64" : "X_out_dev_c64");
        }
    }
    cudaStream_t st = cuda_stream ? (cudaStream_t)cuda_stream : cudaStreamLegacy;
    StaticDev d;
    {
        std::lock_guard<std::mutex> lk(g_static_mu);
        StaticDev& slot = g_static_dev[device];
        if (!slot.ready) {
            int major = 0;
            CUS(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, device));
            if (major < 10) return static_fail(errbuf, errbuf_len, BEGE_ECUDA, "device %d is sm_%d0; the library holds sm_100a code only", device, major);
            const char* what = "";
            const cudaError_t e = static_setup(slot, st, &what);
            if (e != cudaSuccess) { cudaGetLastError(); return static_fail(errbuf, errbuf_len, BEGE_ECUDA, "set-up of device %d, %s: %s", device, what, cudaGetErrorString(e)); }
        }
        d = slot;
    }
    // band in bins exactly as bege_plan_create computes it (inclusive edges)
    const double df = fs / kN;
    const uint32_t klo = (uint32_t)ceil(lo / df - 1e-9), khi = (uint32_t)floor(hi / df + 1e-9);
    // Nothing in G has to start at zero: step A writes all N words of each of the n_segments slots it is given before
    // step B (same stream) reads them, and slots beyond n_segments are not read.
    k_fwd_rows_data<<<dim3(16, n_segments), 256, 0, st>>>((const c2*)x_dev, d.tw256, d.twN, d.G);
    k_fwd_cols_natural<<<dim3(16, n_segments), 256, 0, st>>>(d.G, (c2*)X_out_dev, d.tw256, klo, khi);
    CUS(cudaGetLastError());
#undef CUS
    return BEGE_OK;
}
