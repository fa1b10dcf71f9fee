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
// "Tile layout" of a spectrum (bank, segments, forward scratch): for tile b (columns k1 = 16 b + c),
// kept row-block i (rows k2 = g + 16 i), element index ((b*NI + (i - I0))*16 + c)*16 + g, so that the 16
// lanes g of a half-warp (and the two half-warps c, c+1 of a warp) read contiguous memory.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

#include <cuda_runtime.h>

#include "../../include/bege.h"
#include "cplx.cuh"
#include "async.cuh"
#include "bank64.cuh"

#ifndef BEGE_ABL
// Ablation switches for timing experiments (profiles/r1e_search_kernel.md); never set in the product build, results
// are garbage when any is set: 1 no cross-CTA waits, 2 no template tile loads, 4 no ring stores, 8 no ring loads,
// 16 pass-1 teams off, 32 pass-2 teams off.
#define BEGE_ABL 0
#endif

namespace bege {

constexpr int kN = 65536;
constexpr int kBatch = 72;                 // spectra per launch of the forward transforms (fp64 bank staging: 75 MB)
constexpr int kMaxGroups = 32;             // search: persistent CTA groups of 16 tiles (9 on a 148-SM B200)
constexpr uint64_t kMiscHdr = 4096;        // counter @0, abort flag @8, done1 @256, done2 @2048 (per group and ring slot)

// ------------------------------------------------------------------------------------------------
// shared-memory exchange index for the column passes: stage-1 thread (c, g) writes its p-th value,
// stage-2 thread (c, p) reads over g.  XOR swizzle keeps both sides bank-conflict free (8-byte words).
BEGE_D int xidx(int c, int g, int p) { return ((p << 4) + g) * 16 + (c ^ g); }
// private 256-element region of a half-warp: lane a writes its p-th value, lane p reads over a
BEGE_D int pidx(int a, int p) { return (a << 4) + (p ^ a); }

// stage 1 of a 256-point DFT held by a half-warp: 16-point DFT over the register index, then the
// w256^(DIR * lane * p) twiddles (w1[p] = exp(+2 pi i lane p / 256), conjugated for DIR < 0)
template <int DIR>
BEGE_D void stage1(c2 (&v)[16], const float2 (&w1)[16]) {
    fft16<DIR>(v);
#pragma unroll
    for (int p = 1; p < 16; ++p) v[p] = cmul(v[p], w1[p].x, DIR > 0 ? w1[p].y : -w1[p].y);
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
        out[((q * 16 + ia) * 16 + p) * 16 + ga] = cmul(v[q], w.x, -w.y);
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
    // lane p = g holds k2 = p + 16 q
    c2* o = out + jl * out_stride + (uint64_t)b * NI * 256;
    const uint32_t k1 = 16 * b + c;
#pragma unroll
    for (int q = 0; q < 16; ++q) {
        if (q < I0 || q >= I0 + NI) continue;
        c2 val = v[q];
        if (MASK) {
            const uint32_t k = k1 + 256u * (uint32_t)(g + 16 * q);
            const uint32_t kk = k < (uint32_t)kN / 2 ? k : (uint32_t)kN - k;
            if (kk < klo || kk > khi) val = mk(0.f, 0.f);
        }
        o[((q - I0) * 16 + c) * 16 + g] = val;
    }
}

// ------------------------------------------------------------------------------------------------
// a3 - a7, one persistent warp-specialised kernel for a whole search (PAPER.md:156-162 steps ii-iv; eq.5-9, 13).
// grid (16 tiles, G groups), one CTA of 32 warps (64 registers per thread) per SM, cooperative launch (all CTAs
// co-resident).  The 16 CTAs of a group share the group's (template, segment) items; item `it` of a group is the
// pair (template grp + G (it / nS), segment it % nS).  CTA (b, grp) owns columns k1 = 16 b + c in pass 1 and rows
// n2 = 16 b + r in pass 2.  The path is latency bound, not pipe bound (profiles/), so the kernel is built for
// warps in flight: four teams of 8 warps, two per pass, team k of a pass taking the items it = k (mod 2).
//   A teams (pass 1): the template's column tile arrives in shared memory by bulk async copy from HBM (one
//              buffer per team, refilled as soon as the team has read it, mbarrier-tracked).  Stage 1: half-warp
//              c, lane g holds rows k2 = g + 16 i of column c: conj(H) X against the segment tile (shared
//              memory), Parseval partial sum, 16-point DFTs, twiddles theta^p generated from one complex number
//              per thread.  One exchange through shared memory (two named barriers of the team per item).
//              Stage 2: lane c, p = warp-pair index: 16-point DFTs, and
//              T[n2 = p + 16 q][16 b + c] goes straight from registers to the ring in L2 (128 B per half-warp
//              and store).  The tile is published (done1) with a release issued one item later.
//   B teams (pass 2): half-warp r waits for all 16 tiles of an item (done1), loads its row of T from the ring,
//              runs the 256-point row DFT over k1 through a private shared-memory region, thresholds against
//              k^2 sum|R|^2, compacts the tails with warp-aggregated atomics, and releases its share of the
//              ring slot (done2) as soon as the row is in registers.
// The ring holds kRing items per group (G x kRing x 512 KiB) and lives in L2.  Four-step twiddle wN^(k1 n2) with
// n2 = p + 16 q is split into wN^(k1 p), folded into theta = exp(2 pi i (256 g + k1) / N) of pass 1, and
// wN^(16 k1 q), applied by pass 2 to its inputs (q = n2 >> 4 is the CTA's tile index there: a 16 x 16 table in
// shared memory); theta and the tables are rounded once from fp64 angles.
constexpr int kRing = 8;
constexpr int kSearchThreads = 32 * 32;
constexpr int kPriv = 16 * 17;                              // padded private region of a half-warp (c2 elements)
constexpr int kXch = 16 * 16 * 17;                          // padded exchange buffer of pass 1 (c2 elements)

template <int NI, bool XS> struct SearchSmem {
    c2 hbuf[2][NI * 256];                                   // template column tile of each A team
    c2 xs[XS ? NI * 256 : 2];                               // segment column tile (single-segment searches)
    c2 xch[2][kXch];                                        // pass 1 of each A team: stage 1 -> stage 2, [p][g][c]
    c2 bpriv[32][kPriv];                                    // pass 2: private exchange regions
    float2 tbl[256];                                        // wN^(16 b k1), k1 = a + 16 r, [r][a] (pass 2)
    float2 w1t[256];                                        // w256^(a p), [p][a]
    float ssig[2][8];                                       // Parseval partial sums of the 8 warps of an A team
    uint64_t hfull[2];
};
template <int NI, bool SINGLE> __host__ __device__ constexpr bool search_xs() { return SINGLE && NI <= 14; }
template <int NI, bool SINGLE> constexpr int search_smem() { return (int)sizeof(SearchSmem<NI, search_xs<NI, SINGLE>()>) + 128; }

BEGE_D void bar_team(int id) { asm volatile("bar.sync %0, 256;" :: "r"(id) : "memory"); }   // the 8 warps of a team
BEGE_D c2 cmul2(c2 x, c2 w) { return cmul(x, re(w), im(w)); }                               // x * w

template <int I0, int NI, bool SINGLE>
__global__ void __launch_bounds__(kSearchThreads, 1)
k_search(const c2* __restrict__ bank, const c2* __restrict__ xseg, c2* __restrict__ ring,
         float* __restrict__ sigpart, float k2, float k2hi, bege_tail* __restrict__ rec, unsigned long long cap,
         unsigned long long* __restrict__ counter, c2* __restrict__ zdbg, uint64_t j0, uint64_t nT,
         uint32_t m0, uint32_t nS, uint32_t S, unsigned long long* done1, unsigned long long* done2,
         int* abort_flag)
{
    constexpr bool XS = search_xs<NI, SINGLE>();
    extern __shared__ __align__(128) unsigned char smem_raw[];
    SearchSmem<NI, XS>& sm = *reinterpret_cast<SearchSmem<NI, XS>*>(smem_raw);
    const int team = threadIdx.x >> 8;                       // 0, 1: A teams; 2, 3: B teams
    const int t = threadIdx.x & 255, warp = t >> 5, lane = t & 31;   // within the team
    const int b = blockIdx.x, grp = blockIdx.y, G = gridDim.y;
    constexpr uint32_t kTileBytes = NI * 256 * sizeof(c2);
    constexpr uint64_t kTile = (uint64_t)NI * 256;

    if (threadIdx.x == 0) {
        mbar_init(&sm.hfull[0], 1); mbar_init(&sm.hfull[1], 1);
        fence_mbar_init();
    }
    if (team == 0) {                                         // tbl[r][a] = exp(2 pi i 16 b (a + 16 r) / N)
        const int r = t >> 4, a = t & 15;
        double sn, cs;
        sincospi(2.0 * (double)((16 * b * (a + 16 * r)) & (kN - 1)) / (double)kN, &sn, &cs);
        sm.tbl[t] = make_float2((float)cs, (float)sn);
    } else if (team == 1) {                                  // w1t[p][a] = exp(2 pi i a p / 256)
        const int p = t >> 4, a = t & 15;
        double sn, cs;
        sincospi(2.0 * (double)((a * p) & 255) / 256.0, &sn, &cs);
        sm.w1t[t] = make_float2((float)cs, (float)sn);
    } else if (XS && team == 2) {
        const c2* xb = xseg + ((uint64_t)m0 * 16 + b) * kTile;
        for (int ii = 0; ii < NI; ++ii) sm.xs[XS ? ii * 256 + t : 0] = xb[ii * 256 + t];
    }
    __syncthreads();

    const uint32_t nTg = nT > (uint64_t)grp ? (uint32_t)((nT - grp + G - 1) / G) : 0u;   // templates of this group
    const uint32_t n_items = nTg * nS;                      // < 2^31: the host splits larger searches
    c2* myring = ring + (uint64_t)grp * kRing * kN;
    unsigned long long* d1 = done1 + grp * kRing;            // one counter pair per ring slot: a count can only
    unsigned long long* d2 = done2 + grp * kRing;            // come from the item that currently owns the slot

    if ((BEGE_ABL & 16) && team < 2) return;
    if ((BEGE_ABL & 32) && team >= 2) return;
    if (team < 2) {
        // ================================================================ A: pass 1, items it = team (mod 2)
        const int c = t >> 4, g = t & 15;                    // stage 1: column of the tile, lane of its half-warp
        const int c2i = t & 15, p2 = t >> 4;                 // stage 2: column, index p of n2 = p + 16 q
        c2 theta;                                            // exp(2 pi i (256 g + k1) / N), k1 = 16 b + c
        {
            double sn, cs;
            sincospi(2.0 * (double)(256 * g + 16 * b + c) / (double)kN, &sn, &cs);
            theta = mk((float)cs, (float)sn);
        }
        uint64_t* hfull = &sm.hfull[team];
        c2* hb = sm.hbuf[team];
        if (t == 0 && (uint32_t)team < n_items && !(BEGE_ABL & 2)) {
            mbar_arrive_expect_tx(hfull, kTileBytes);
            bulk_load(hb, bank + ((j0 + grp + (uint64_t)G * (SINGLE ? (uint32_t)team : team / nS)) * 16 + b) * kTile,
                      kTileBytes, hfull, policy_evict_first());
        }
        c2* xw = sm.xch[team] + g * 17 + c;                  // + p * 272: element [p][g][c] of the exchange buffer
        const c2* xrd = sm.xch[team] + p2 * 272 + c2i;       // + gg * 17
        const int bar_id = 1 + team;
        int pending = -1;                                    // ring slot whose tile this warp has yet to publish
        uint32_t nload = 0;                                  // tiles this team has waited for so far
        uint32_t tj_prev = ~0u;
        for (uint32_t it = team; it < n_items; it += 2) {
            const uint32_t tj = SINGLE ? it : it / nS;
            const uint32_t ml = SINGLE ? 0u : (uint32_t)(it - tj * nS);
            const int slot = (int)(it % kRing);
            if (tj != tj_prev) {                             // a new template tile was ordered for this item
#if !(BEGE_ABL & 2)
                mbar_wait(hfull, nload & 1, abort_flag);
#endif
                ++nload;
                tj_prev = tj;
            }
            c2 v[16];
            c2 acc = mk(0.f, 0.f);
            {
                const c2* xb = xseg + ((uint64_t)(m0 + ml) * 16 + b) * kTile;
#pragma unroll
                for (int r = 0; r < 16; ++r) {
                    if (r >= I0 && r < I0 + NI) {
                        const c2 xv = XS ? sm.xs[XS ? (r - I0) * 256 + t : 0] : __ldg(xb + (r - I0) * 256 + t);
                        v[r] = cmulc(xv, hb[(r - I0) * 256 + t]);
                        acc = fma2(v[r], v[r], acc);
                    } else {
                        v[r] = mk(0.f, 0.f);
                    }
                }
            }
            fft16<+1>(v);
            {   // v[p] *= theta^p, powers by a depth-4 product tree
                const c2 t2 = cmul2(theta, theta), t4 = cmul2(t2, t2), t8 = cmul2(t4, t4);
                const c2 t3 = cmul2(t2, theta), t5 = cmul2(t4, theta), t6 = cmul2(t4, t2), t7 = cmul2(t4, t3);
                v[1] = cmul2(v[1], theta); v[2] = cmul2(v[2], t2); v[3] = cmul2(v[3], t3); v[4] = cmul2(v[4], t4);
                v[5] = cmul2(v[5], t5); v[6] = cmul2(v[6], t6); v[7] = cmul2(v[7], t7); v[8] = cmul2(v[8], t8);
                v[9] = cmul2(v[9], cmul2(t8, theta)); v[10] = cmul2(v[10], cmul2(t8, t2));
                v[11] = cmul2(v[11], cmul2(t8, t3)); v[12] = cmul2(v[12], cmul2(t8, t4));
                v[13] = cmul2(v[13], cmul2(t8, t5)); v[14] = cmul2(v[14], cmul2(t8, t6));
                v[15] = cmul2(v[15], cmul2(t8, t7));
            }
#pragma unroll
            for (int p = 0; p < 16; ++p) xw[p * 272] = v[p];
            const float sw = warp_sum32(re(acc) + im(acc));
            if (lane == 0) sm.ssig[team][warp] = sw;
            bar_team(bar_id);                                // exchange buffer complete, template tile read out
            if (t == 0 && !(BEGE_ABL & 2)) {                 // order the tile of this team's next item
                const uint32_t it2 = it + 2;
                if (it2 < n_items) {
                    const uint32_t tj2 = SINGLE ? it2 : it2 / nS;
                    if (tj2 != tj) {
                        mbar_arrive_expect_tx(hfull, kTileBytes);
                        bulk_load(hb, bank + ((j0 + grp + (uint64_t)G * tj2) * 16 + b) * kTile, kTileBytes, hfull,
                                  policy_evict_first());
                    }
                }
            }
            unsigned long long d2v = ~0ull;                  // slot-free counter, polled early: the load is in flight
            if (it >= kRing && lane == 0 && !(BEGE_ABL & 1)) d2v = counter_load_relaxed(d2 + slot);   // during stage 2
#pragma unroll
            for (int gg = 0; gg < 16; ++gg) v[gg] = xrd[gg * 17];
            float tot = 0.f;
            if (t == 0) {
#pragma unroll
                for (int w = 0; w < 8; ++w) tot += sm.ssig[team][w];
            }
            bar_team(bar_id);                                // exchange buffer free for the team's next item
            if (pending >= 0 && t == 0)                      // the team's stores of its previous item were all issued
                counter_add_release(d1 + pending, 1ull);     // before this barrier and have long landed
            fft16<+1>(v);
#if !(BEGE_ABL & 1)
            if (it >= kRing) {                               // ring slot read out by pass 2 of item it - kRing
                d2v = __shfl_sync(0xffffffffu, d2v, 0);
                if (d2v < 128ull * (it / kRing)) warp_counter_wait_ge(d2 + slot, 128ull * (it / kRing), abort_flag, lane);
            }
#endif
            c2* out = myring + (uint64_t)slot * kN + 16 * b + c2i + p2 * 256;
#pragma unroll
            for (int q = 0; q < 16; ++q) {
                const c2 o = v[q];
                if (!(BEGE_ABL & 4) || re(o) == 1.2345e-30f) out[q * 4096] = o;
            }
            if (t == 0) sigpart[((j0 + grp + (uint64_t)G * tj) * (uint64_t)S + (m0 + ml)) * 16 + b] = tot;
            pending = slot;
        }
        bar_team(bar_id);
        if (pending >= 0 && t == 0) counter_add_release(d1 + pending, 1ull);
    } else {
        // ================================================================ B: pass 2, items ib = team - 2 (mod 2)
        const int kb = team - 2;
        const int hw = t >> 4, a = t & 15;                   // row of the row tile, lane of its half-warp
        const int n2 = 16 * b + hw;
        c2* priv = sm.bpriv[kb * 16 + hw];
        c2* pwr = priv + a * 17;                             // + p:      stage-1 output p of lane a
        const c2* prd = priv + a;                            // + 17 aa:  stage-2 input from lane aa
        const float2* w1 = sm.w1t + a;                       // + 16 p:   exp(2 pi i a p / 256)
        const uint64_t row_off = (uint64_t)n2 * 256 + (uint64_t)a;           // T[n2][k1 = a + 16 r]
        for (uint32_t ib = kb; ib < n_items; ib += 2) {
            const int slot = (int)(ib % kRing);
            const uint32_t use = ib / kRing;
            const uint32_t tj = SINGLE ? ib : ib / nS;
            const uint32_t ml = SINGLE ? 0u : (uint32_t)(ib - tj * nS);
            const uint64_t jl = grp + (uint64_t)G * tj;
#if !(BEGE_ABL & 1)
            warp_counter_wait_ge(d1 + slot, 16ull * (use + 1), abort_flag, lane);     // all 16 tiles are in the ring
#endif
            const c2* src = myring + (uint64_t)slot * kN + row_off;
            c2 v[16];
#pragma unroll
            for (int r = 0; r < 16; ++r) v[r] = (BEGE_ABL & 8) ? mk((float)(r + a), (float)ib) : __ldcg(src + 16 * r);
#pragma unroll
            for (int r = 0; r < 16; ++r) v[r] = cmul(v[r], sm.tbl[16 * r + a]);          // wN^(16 k1 q), q = b
            const uint64_t pair = (j0 + jl) * (uint64_t)S + (m0 + ml);
            const float sumR2 = hw_sum16(__ldcg(sigpart + pair * 16 + a));
            fft16<+1>(v);
            __syncwarp();
            if (lane == 0) counter_add_relaxed(d2 + slot, 1ull);             // this warp's rows are in registers (the
                                                                             // loads have returned: fft16 consumed them)
#pragma unroll
            for (int p = 1; p < 16; ++p) v[p] = cmul(v[p], w1[16 * p]);
#pragma unroll
            for (int p = 0; p < 16; ++p) pwr[p] = v[p];
            __syncwarp();
#pragma unroll
            for (int aa = 0; aa < 16; ++aa) v[aa] = prd[aa * 17];
            __syncwarp();
            fft16<+1>(v);
            // lane a holds Z[n1 = a + 16 q]; lag n = 256 n1 + n2
            const float thr = k2 * sumR2;
            unsigned hits = 0;
#pragma unroll
            for (int q = 0; q < 16; ++q) {
                const c2 sq = mul2(v[q], v[q]);
                if (re(sq) + im(sq) > thr) hits |= 1u << q;
            }
            if (zdbg != nullptr) {
                const float invN = 1.0f / (float)kN;
#pragma unroll
                for (int q = 0; q < 16; ++q)
                    zdbg[(uint64_t)(a + 16 * q) * 256 + n2] = mul2(v[q], bc(invN));
            }
#if BEGE_ABL
            if (thr == -1.f)                                 // timing experiment only: never emit
#endif
            if (__any_sync(0xffffffffu, hits != 0)) {
                const float inv = 1.0f / sumR2;
                if (k2hi < 3.0e38f) {                        // band threshold: drop |z| >= k_hi sigma
                    const float thr_hi = k2hi * sumR2;
#pragma unroll
                    for (int q = 0; q < 16; ++q) {
                        const c2 sq = mul2(v[q], v[q]);
                        if (!(re(sq) + im(sq) < thr_hi)) hits &= ~(1u << q);
                    }
                }
                if (cap == ~0ull) {
                    // max projection: per sample offset the largest |z|/sigma over the bank and
                    // its template, race free: one 64-bit atomicMax on (snr bits, ~template_id); positive floats
                    // order like their bit patterns, equal values go to the smaller template id
                    unsigned long long* proj = reinterpret_cast<unsigned long long*>(rec);
#pragma unroll
                    for (int q = 0; q < 16; ++q) {
                        if (hits & (1u << q)) {
                            const c2 sq = mul2(v[q], v[q]);
                            const float snr = sqrtf((re(sq) + im(sq)) * inv);
                            const uint32_t lag = (uint32_t)(m0 + ml) * (uint32_t)kN + (uint32_t)((a + 16 * q) * 256 + n2);
                            atomicMax(proj + lag, ((unsigned long long)__float_as_uint(snr) << 32) |
                                                      (unsigned long long)(0xffffffffu - (uint32_t)(j0 + jl)));
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
                    if (lane == 31) base = atomicAdd(counter, (unsigned long long)total);
                    base = __shfl_sync(0xffffffffu, base, 31);
                    unsigned long long slot_r = base + (unsigned long long)(incl - cnt);
#pragma unroll
                    for (int q = 0; q < 16; ++q) {
                        if (hits & (1u << q)) {
                            if (slot_r < cap) {
                                const c2 sq = mul2(v[q], v[q]);
                                bege_tail r;
                                r.template_id = (uint32_t)(j0 + jl);
                                r.lag = (uint32_t)(m0 + ml) * (uint32_t)kN + (uint32_t)((a + 16 * q) * 256 + n2);
                                r.snr = sqrtf((re(sq) + im(sq)) * inv);
                                rec[slot_r] = r;
                            }
                            ++slot_r;
                        }
                    }
                }
            }
        }
    }
}

// sigma_jm = sqrt(sum of the 16 tile partial sums) / N
__global__ void k_sigma(const float* __restrict__ sigpart, float* __restrict__ sigma, uint64_t n)
{
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float s = 0.f;
    // same pairwise order as hw_sum16 (xor 8, 4, 2, 1) so that sigma matches the search bit for bit
    float v[16];
    for (int a = 0; a < 16; ++a) v[a] = sigpart[i * 16 + a];
    for (int d = 8; d >= 1; d >>= 1)
        for (int a = 0; a < d; ++a) v[a] = v[a] + v[a + d];
    s = v[0];
    sigma[i] = sqrtf(s) / (float)kN;
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
    float2 *tw256 = nullptr, *twN = nullptr;
    d2 *tw256d = nullptr, *twNd = nullptr;   // exp(2 pi i m / 256), exp(2 pi i m / N) in fp64 (bank generation)
    // workspace
    unsigned char* ws = nullptr; uint64_t ws_bytes = 0, bump = 0; bool user_ws = false;
    Slot s_bank, s_x, s_scratch, s_sig, s_rec, s_misc, s_par, s_proj;
    uint64_t T = 0; uint32_t S = 0; double tau = 0; uint32_t L = 0;
    bool have_sigma = false;
    // pinned staging
    unsigned long long* h_count = nullptr;
    cudaEvent_t ev_a = nullptr, ev_b = nullptr, ev_done = nullptr;
    bool profiling = false;
    void* l2_window = nullptr;      // ring region currently marked persisting in L2 (access policy window of the stream)
    bege_stats stats{};
    std::string err;
};

// take the ring's persisting-L2 window off the plan's stream again (the stream may be the caller's)
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
    cudaCtxResetPersistingL2Cache();
    cudaGetLastError();
    p->l2_window = nullptr;
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

static uint64_t tpl_bytes(const bege_plan* p) { return (uint64_t)p->NI * 16 * 256 * sizeof(c2); }

static void count_launch(bege_plan* p, uint64_t n = 1) { p->stats.kernel_launches += n; }

extern "C" const char* bege_version(void) { return "bege 0.1 (sm_100a)"; }

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
    if (stream) p->stream = (cudaStream_t)stream;
    else { if (cudaStreamCreateWithFlags(&p->stream, cudaStreamNonBlocking) != cudaSuccess) return bail(BEGE_ECUDA); p->own_stream = true; }
    if (cudaStreamCreateWithFlags(&p->side, cudaStreamNonBlocking) != cudaSuccess) return bail(BEGE_ECUDA);
    if (cudaEventCreate(&p->ev_a) != cudaSuccess || cudaEventCreate(&p->ev_b) != cudaSuccess ||
        cudaEventCreateWithFlags(&p->ev_done, cudaEventDisableTiming) != cudaSuccess) return bail(BEGE_ECUDA);
    if (cudaMallocHost(&p->h_count, 64) != cudaSuccess) return bail(BEGE_ECUDA);

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
        std::vector<d2> t256(256), tN(N);
        for (int m = 0; m < 256; ++m) { t256[m].x = cos(2.0 * M_PI * m / 256.0); t256[m].y = sin(2.0 * M_PI * m / 256.0); }
        for (uint32_t m = 0; m < N; ++m) { tN[m].x = cos(2.0 * M_PI * m / (double)N); tN[m].y = sin(2.0 * M_PI * m / (double)N); }
        if (cudaMalloc(&p->tw256d, 256 * sizeof(d2)) != cudaSuccess || cudaMalloc(&p->twNd, N * sizeof(d2)) != cudaSuccess) return bail(BEGE_ENOMEM);
        if (cudaMemcpy(p->tw256d, t256.data(), 256 * sizeof(d2), cudaMemcpyHostToDevice) != cudaSuccess ||
            cudaMemcpy(p->twNd, tN.data(), N * sizeof(d2), cudaMemcpyHostToDevice) != cudaSuccess) return bail(BEGE_ECUDA);
        if (cudaFuncSetAttribute(k_bank_cols64, cudaFuncAttributeMaxDynamicSharedMemorySize, 16 * 256 * (int)sizeof(d2)) != cudaSuccess) return bail(BEGE_ECUDA);
    }
    if (cudaMalloc(&p->tw256, w256.size() * sizeof(float2)) != cudaSuccess ||
        cudaMalloc(&p->twN, wN.size() * sizeof(float2)) != cudaSuccess) return bail(BEGE_ENOMEM);
    if (cudaMemcpy(p->tw256, w256.data(), w256.size() * sizeof(float2), cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMemcpy(p->twN, wN.data(), wN.size() * sizeof(float2), cudaMemcpyHostToDevice) != cudaSuccess) return bail(BEGE_ECUDA);

    // the search kernel needs all its CTAs co-resident (groups hand over through global counters)
    int occ = 0;
    {
        const void* fs[4] = {(const void*)k_search<1, 14, true>, (const void*)k_search<1, 14, false>,
                             (const void*)k_search<0, 16, true>, (const void*)k_search<0, 16, false>};
        const int sms[4] = {search_smem<14, true>(), search_smem<14, false>(), search_smem<16, true>(), search_smem<16, false>()};
        for (int i = 0; i < 4; ++i) {
            if (cudaFuncSetAttribute(fs[i], cudaFuncAttributeMaxDynamicSharedMemorySize, sms[i]) != cudaSuccess) return bail(BEGE_ECUDA);
            int o = 0;
            if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o, fs[i], kSearchThreads, sms[i]) != cudaSuccess) return bail(BEGE_ECUDA);
            occ = i ? std::min(occ, o) : o;
        }
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
    drop_l2_window(p);
    if (p->side) { cudaStreamSynchronize(p->side); cudaStreamDestroy(p->side); }
    if (p->own_stream && p->stream) cudaStreamDestroy(p->stream);
    for (Slot* s : {&p->s_bank, &p->s_x, &p->s_scratch, &p->s_sig, &p->s_rec, &p->s_misc, &p->s_par, &p->s_proj}) slot_free(*s);
    if (p->tw256) cudaFree(p->tw256);
    if (p->twN) cudaFree(p->twN);
    if (p->tw256d) cudaFree(p->tw256d);
    if (p->twNd) cudaFree(p->twNd);
    if (p->h_count) cudaFreeHost(p->h_count);
    if (p->ev_a) cudaEventDestroy(p->ev_a);
    if (p->ev_b) cudaEventDestroy(p->ev_b);
    if (p->ev_done) cudaEventDestroy(p->ev_done);
    delete p;
}

// one region serves the fp64 staging of the bank generation (kBatch spectra of 16-byte elements), the fp32 staging of
// the segment transform and the search ring (G groups x kRing items)
static uint64_t scratch_bytes(const bege_plan* p)
{
    return std::max<uint64_t>((uint64_t)kBatch * kN * sizeof(d2), (uint64_t)p->G * kRing * kN * sizeof(c2));
}

extern "C" int bege_plan_workspace_bytes(const bege_plan* p, uint64_t T, uint32_t S, uint64_t cap, uint64_t* bytes)
{
    if (!p || !bytes) return BEGE_EINVAL;
    auto al = [](uint64_t v) { return align_up(v ? v : 256, 256); };
    uint64_t b = 0;
    b += al(T * tpl_bytes(p));                         // bank
    b += al(T * 16);                                   // template parameters (f0, fdot)
    b += al((uint64_t)S * tpl_bytes(p));               // segment spectra
    b += al(scratch_bytes(p));                          // four-step staging (stays in L2)
    b += al(T * S * 16 * sizeof(float));               // Parseval partial sums
    b += al(std::max<uint64_t>(cap * sizeof(bege_tail), (uint64_t)S * kN * 8));   // records / max-projection array
    b += al(kMiscHdr + (uint64_t)S * kN * sizeof(c2)); // counters + raw segment staging
    *bytes = b + 4096;
    return BEGE_OK;
}

extern "C" int bege_plan_set_workspace(bege_plan* p, void* dev_ptr, uint64_t bytes)
{
    if (!p) return BEGE_EINVAL;
    if (dev_ptr && ((uintptr_t)dev_ptr & 255)) return fail(p, BEGE_EINVAL, "workspace must be 256-byte aligned");
    CU(p, cudaSetDevice(p->device));
    CU(p, cudaStreamSynchronize(p->stream));
    drop_l2_window(p);
    for (Slot* s : {&p->s_bank, &p->s_x, &p->s_scratch, &p->s_sig, &p->s_rec, &p->s_misc, &p->s_par, &p->s_proj}) slot_free(*s);
    p->ws = (unsigned char*)dev_ptr; p->ws_bytes = dev_ptr ? bytes : 0; p->bump = 0; p->user_ws = dev_ptr != nullptr;
    p->T = 0; p->S = 0; p->have_sigma = false;
    return BEGE_OK;
}

extern "C" int bege_bank_generate(bege_plan* p, const double* f0, const double* fdot, uint64_t T, double tau)
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
    p->T = 0; p->have_sigma = false;
    double* d_f0 = (double*)par; double* d_fd = d_f0 + T;
    CU(p, cudaMemcpyAsync(d_f0, f0, T * sizeof(double), cudaMemcpyHostToDevice, p->stream));
    CU(p, cudaMemcpyAsync(d_fd, fdot, T * sizeof(double), cudaMemcpyHostToDevice, p->stream));
    // unit L2 norm: ||h||^2 = sum_n hann_L[n]^2 (the phase factor has modulus 1)
    const uint32_t L = (uint32_t)Ll;
    double n2 = 0;
    for (uint32_t n = 0; n < L; ++n) { const double w = 0.5 - 0.5 * cos(2.0 * M_PI * n / (double)(L - 1)); n2 += w * w; }
    const double inv_norm = 1.0 / sqrt(n2);
    const uint64_t stride = tpl_bytes(p) / sizeof(c2);
    for (uint64_t j0 = 0; j0 < T; j0 += kBatch) {
        const unsigned nb = (unsigned)std::min<uint64_t>(kBatch, T - j0);
        k_bank_rows64<<<dim3(16, nb), 256, 0, p->stream>>>(d_f0, d_fd, j0, p->fs, L, inv_norm, p->tw256d, p->twNd, (d2*)scr);
        k_bank_cols64<<<dim3(16, nb), 256, 16 * 256 * sizeof(d2), p->stream>>>((const d2*)scr, (float2*)bank + j0 * stride, stride,
                                                                            p->I0, p->NI, p->tw256d);
        count_launch(p, 2);
    }
    CU(p, cudaGetLastError());
    CU(p, cudaStreamSynchronize(p->stream));
    p->T = T; p->tau = tau; p->L = L;
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
    p->S = 0; p->have_sigma = false;
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
    CU(p, cudaGetLastError());
    CU(p, cudaStreamSynchronize(p->stream));
    p->S = S;
    return BEGE_OK;
}

// one cooperative launch of the persistent search kernel over templates [j0, j0 + nT) x segments [m0, m0 + nS)
static int launch_search(bege_plan* p, const c2* bank, const c2* xs, c2* ring, float* sig, float k2, float k2hi, bege_tail* rec,
                         uint64_t cap, unsigned char* misc, c2* zdbg, uint64_t j0, uint64_t nT, uint32_t m0, uint32_t nS,
                         bool first = true)
{
    unsigned long long* counter = (unsigned long long*)misc;
    int* abort_flag = (int*)(misc + 8);
    unsigned long long* done1 = (unsigned long long*)(misc + 256);
    unsigned long long* done2 = (unsigned long long*)(misc + 2048);
    // the first launch of a search also clears the record counter and the abort flag (first 16 bytes)
    CU(p, cudaMemsetAsync(misc + (first ? 0 : 16), 0, kMiscHdr - (first ? 0 : 16), p->stream));
    const int G = (int)std::min<uint64_t>((uint64_t)p->G, nT);
    const dim3 grid(16, G);
    if (p->l2_window != (void*)ring) {
        // keep the ring's lines resident: they are rewritten every few microseconds and must not be written back
        // to HBM in between (ncu: 31 KB of write-back per correlation without this); best effort, errors ignored
        const size_t bytes = (size_t)p->G * kRing * kN * sizeof(c2);
        cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, bytes);
        cudaStreamAttrValue av{};
        av.accessPolicyWindow.base_ptr = (void*)ring;
        av.accessPolicyWindow.num_bytes = bytes;
        av.accessPolicyWindow.hitRatio = 1.0f;
        av.accessPolicyWindow.hitProp = cudaAccessPropertyPersisting;
        av.accessPolicyWindow.missProp = cudaAccessPropertyStreaming;
        cudaStreamSetAttribute(p->stream, cudaStreamAttributeAccessPolicyWindow, &av);
        cudaGetLastError();
        p->l2_window = (void*)ring;
    }
    const bool single = (p->S == 1);
    unsigned long long capll = cap;
    uint32_t S = p->S;
    void* args[] = {&bank, &xs, &ring, &sig, &k2, &k2hi, &rec, &capll, &counter, &zdbg, &j0, &nT, &m0, &nS, &S,
                    &done1, &done2, &abort_flag};
    const void* f = p->NI == 14 ? (single ? (const void*)k_search<1, 14, true> : (const void*)k_search<1, 14, false>)
                                : (single ? (const void*)k_search<0, 16, true> : (const void*)k_search<0, 16, false>);
    const int kSearchSmem = p->NI == 14 ? (single ? search_smem<14, true>() : search_smem<14, false>())
                                        : (single ? search_smem<16, true>() : search_smem<16, false>());
    if (p->profiling) cudaEventRecord(p->ev_a, p->stream);
    CU(p, cudaLaunchCooperativeKernel(f, grid, dim3(kSearchThreads), args, kSearchSmem, p->stream));
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
    CU(p, cudaMemcpyAsync(&flag, misc + 8, sizeof flag, cudaMemcpyDeviceToHost, p->stream));
    CU(p, cudaStreamSynchronize(p->stream));
    if (flag) return fail(p, BEGE_ECUDA, "search pipeline timed out waiting on a group counter");
    return BEGE_OK;
}

static int search_impl(bege_plan* p, float k_sigma, float k_hi, bege_tail* tails_out, uint64_t cap, uint64_t* n_tails)
{
    if (!p) return BEGE_EINVAL;
    if (!n_tails || (cap && !tails_out) || !(k_sigma >= 0.f) || !(k_hi >= k_sigma) || cap == ~0ull)
        return fail(p, BEGE_EINVAL, "bad search arguments");
    if (!p->T || !p->S) return fail(p, BEGE_ESTATE, "bege_search needs a generated bank and loaded segments");
    CU(p, cudaSetDevice(p->device));
    void *sig, *rec, *misc, *scr, *bank, *xs;
    int rc;
    if ((rc = slot_get(p, p->s_sig, p->T * p->S * 16 * sizeof(float), &sig))) return rc;
    if ((rc = slot_get(p, p->s_rec, cap * sizeof(bege_tail), &rec))) return rc;
    if ((rc = slot_get(p, p->s_misc, kMiscHdr, &misc))) return rc;
    if ((rc = slot_get(p, p->s_scratch, scratch_bytes(p), &scr))) return rc;
    if ((rc = slot_get(p, p->s_bank, 0, &bank))) return rc;
    if ((rc = slot_get(p, p->s_x, 0, &xs))) return rc;
    unsigned long long* counter = (unsigned long long*)misc;
    // the kernel counts a group's (template, segment) items in 32 bits: split longer searches
    const uint64_t maxT = std::max<uint64_t>(1, ((1ull << 31) - 1) / p->S / 2) * (uint64_t)p->G;
    for (uint64_t jj = 0; jj < p->T; jj += maxT) {
        if ((rc = launch_search(p, (const c2*)bank, (const c2*)xs, (c2*)scr, (float*)sig, k_sigma * k_sigma, k_hi * k_hi,
                                (bege_tail*)rec, cap, (unsigned char*)misc, nullptr, jj, std::min(maxT, p->T - jj), 0, p->S,
                                jj == 0))) return rc;
    }
    CU(p, cudaGetLastError());
    // only the tails cross PCIe: count first, then exactly the records, on the side stream
    CU(p, cudaMemcpyAsync(p->h_count, counter, sizeof(unsigned long long), cudaMemcpyDeviceToHost, p->stream));
    CU(p, cudaEventRecord(p->ev_done, p->stream));
    CU(p, cudaStreamWaitEvent(p->side, p->ev_done, 0));
    CU(p, cudaMemcpyAsync(p->h_count + 1, (unsigned char*)misc + 8, sizeof(int), cudaMemcpyDeviceToHost, p->stream));
    CU(p, cudaStreamSynchronize(p->stream));
    if (*(volatile int*)(p->h_count + 1)) return fail(p, BEGE_ECUDA, "search pipeline timed out waiting on a group counter");
    const uint64_t total = *p->h_count;
    const uint64_t ncopy = std::min<uint64_t>(total, cap);
    if (ncopy) {
        CU(p, cudaMemcpyAsync(tails_out, rec, ncopy * sizeof(bege_tail), cudaMemcpyDeviceToHost, p->side));
        CU(p, cudaStreamSynchronize(p->side));
    }
    p->stats.correlations += p->T * p->S;
    p->have_sigma = true;
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

extern "C" int bege_search_maxproj(bege_plan* p, float k_sigma, float* snr_out, uint32_t* id_out, uint64_t* n_hits)
{
    if (!p) return BEGE_EINVAL;
    if (!snr_out || !id_out || !(k_sigma >= 0.f)) return fail(p, BEGE_EINVAL, "bad search arguments");
    if (!p->T || !p->S) return fail(p, BEGE_ESTATE, "bege_search_maxproj needs a generated bank and loaded segments");
    CU(p, cudaSetDevice(p->device));
    void *sig, *proj, *misc, *scr, *bank, *xs;
    int rc;
    const uint64_t n = (uint64_t)p->S * kN;
    if ((rc = slot_get(p, p->s_sig, p->T * p->S * 16 * sizeof(float), &sig))) return rc;
    if ((rc = slot_get(p, p->s_rec, n * sizeof(unsigned long long), &proj))) return rc;
    if ((rc = slot_get(p, p->s_misc, kMiscHdr, &misc))) return rc;
    if ((rc = slot_get(p, p->s_scratch, scratch_bytes(p), &scr))) return rc;
    if ((rc = slot_get(p, p->s_bank, 0, &bank))) return rc;
    if ((rc = slot_get(p, p->s_x, 0, &xs))) return rc;
    CU(p, cudaMemsetAsync(proj, 0, n * sizeof(unsigned long long), p->stream));
    const uint64_t maxT = std::max<uint64_t>(1, ((1ull << 31) - 1) / p->S / 2) * (uint64_t)p->G;
    for (uint64_t jj = 0; jj < p->T; jj += maxT) {
        // cap = ~0 switches the kernel's epilogue from appending records to the projection array passed as `rec`
        if ((rc = launch_search(p, (const c2*)bank, (const c2*)xs, (c2*)scr, (float*)sig, k_sigma * k_sigma, INFINITY,
                                (bege_tail*)proj, ~0ull, (unsigned char*)misc, nullptr, jj, std::min(maxT, p->T - jj), 0, p->S,
                                jj == 0))) return rc;
    }
    CU(p, cudaGetLastError());
    std::vector<unsigned long long> host(n);
    CU(p, cudaMemcpyAsync(host.data(), proj, n * sizeof(unsigned long long), cudaMemcpyDeviceToHost, p->stream));
    if ((rc = check_abort(p, (unsigned char*)misc))) return rc;      // synchronises the stream
    uint64_t hits = 0;
    for (uint64_t i = 0; i < n; ++i) {
        const unsigned long long key = host[i];
        if (key) {
            const uint32_t bits = (uint32_t)(key >> 32);
            memcpy(&snr_out[i], &bits, sizeof(float));
            id_out[i] = 0xffffffffu - (uint32_t)key;
            ++hits;
        } else {
            snr_out[i] = 0.f;
            id_out[i] = 0xffffffffu;
        }
    }
    p->stats.correlations += p->T * p->S;
    p->have_sigma = true;
    if (n_hits) *n_hits = hits;
    return BEGE_OK;
}

extern "C" int bege_get_sigma(bege_plan* p, float* sigma_out)
{
    if (!p || !sigma_out) return BEGE_EINVAL;
    if (!p->have_sigma) return fail(p, BEGE_ESTATE, "bege_get_sigma needs a completed bege_search");
    CU(p, cudaSetDevice(p->device));
    const uint64_t n = p->T * p->S;
    float* d = nullptr;
    CU(p, cudaMalloc(&d, n * sizeof(float)));
    void* sig; slot_get(p, p->s_sig, 0, &sig);
    k_sigma<<<(unsigned)((n + 255) / 256), 256, 0, p->stream>>>((const float*)sig, d, n);
    count_launch(p);
    cudaError_t e = cudaMemcpyAsync(sigma_out, d, n * sizeof(float), cudaMemcpyDeviceToHost, p->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(p->stream);
    cudaFree(d);
    CU(p, e);
    return BEGE_OK;
}

extern "C" int bege_debug_correlate(bege_plan* p, uint64_t j, uint32_t m, float* z_out, float* sigma_out)
{
    if (!p || !z_out) return BEGE_EINVAL;
    if (!p->T || !p->S) return fail(p, BEGE_ESTATE, "needs a bank and segments");
    if (j >= p->T || m >= p->S) return fail(p, BEGE_EINVAL, "pair (%llu, %u) out of range", (unsigned long long)j, m);
    CU(p, cudaSetDevice(p->device));
    void *scr, *bank, *xs, *misc;
    int rc;
    if ((rc = slot_get(p, p->s_scratch, scratch_bytes(p), &scr))) return rc;
    if ((rc = slot_get(p, p->s_misc, kMiscHdr, &misc))) return rc;
    slot_get(p, p->s_bank, 0, &bank); slot_get(p, p->s_x, 0, &xs);
    c2* zd = nullptr; float* sg = nullptr;
    CU(p, cudaMalloc(&zd, kN * sizeof(c2)));
    CU(p, cudaMalloc(&sg, 16 * sizeof(float)));         // private partial sums of this one pair
    const bool prof = p->profiling; p->profiling = false;
    // the kernel indexes the partial sums by (j*S + m)*16: bias the base so that this pair lands on sg[0..15]
    float* sg_biased = sg - (j * p->S + m) * 16;
    rc = launch_search(p, (const c2*)bank, (const c2*)xs, (c2*)scr, sg_biased, 1e30f, INFINITY, nullptr, 0, (unsigned char*)misc, zd, j, 1, m, 1);
    p->profiling = prof;
    if (!rc) rc = check_abort(p, (unsigned char*)misc);
    if (rc) { cudaFree(zd); cudaFree(sg); return rc; }
    float part[16];
    cudaError_t e = cudaMemcpyAsync(z_out, zd, kN * sizeof(c2), cudaMemcpyDeviceToHost, p->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(part, sg, sizeof part, cudaMemcpyDeviceToHost, p->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(p->stream);
    if (e == cudaSuccess) e = cudaGetLastError();
    cudaFree(zd); cudaFree(sg);
    CU(p, e);
    if (sigma_out) {
        float v[16];
        for (int a = 0; a < 16; ++a) v[a] = part[a];
        for (int d = 8; d >= 1; d >>= 1) for (int a = 0; a < d; ++a) v[a] = v[a] + v[a + d];
        *sigma_out = sqrtf(v[0]) / (float)kN;
    }
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
                    const float2 v = tile[(((size_t)b * p->NI + ii) * 16 + c) * 16 + g];
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
