// Packed complex fp32 arithmetic for sm_100a.
//
// A complex number lives in one 64-bit register pair as (re, im) and is processed with Blackwell's
// packed fp32x2 instructions (PTX add/sub/mul/fma.rn.f32x2 -> SASS FADD2/FMUL2/FFMA2).  ptxas folds
// the half swap (mk(im, re)) and the scalar broadcast (mk(s, s)) written below into operand
// modifiers (.F32x2.LO_HI, .F32), so a complex add is 1 issue slot and a twiddle multiply 2.
// Measured on B200: FFMA2 issues at half the rate of FFMA, i.e. the same flops in half the issue
// slots, which is what leaves room for the load / shared-memory / integer instructions of the FFT.
//
// The packed instructions have no per-half sign, so the cross terms of a multiplication by a RUN-TIME complex
// number w = (c, d) are two scalar FFMAs (free operand negation, same FMA-pipe time as one FFMA2): 3 issue slots
// and no sign/pack moves.  Compile-time twiddles (fft16) are folded into the butterflies' FMAs and cost one slot.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace bege {

typedef unsigned long long c2;   // packed (re, im), fp32 each

#define BEGE_D __device__ __forceinline__

BEGE_D c2 mk(float re, float im) { c2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(re), "f"(im)); return r; }
BEGE_D float re(c2 v) { float a, b; asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); (void)b; return a; }
BEGE_D float im(c2 v) { float a, b; asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); (void)a; return b; }

BEGE_D c2 add2(c2 a, c2 b) { c2 d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
BEGE_D c2 sub2(c2 a, c2 b) { c2 d; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
BEGE_D c2 mul2(c2 a, c2 b) { c2 d; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
BEGE_D c2 fma2(c2 a, c2 b, c2 c) { c2 d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d; }

BEGE_D c2 swp(c2 a) { return mk(im(a), re(a)); }
BEGE_D c2 bc(float s) { return mk(s, s); }

// a + i*b and a - i*b
BEGE_D c2 add_i(c2 a, c2 b) { return fma2(swp(b), mk(-1.f, 1.f), a); }
BEGE_D c2 sub_i(c2 a, c2 b) { return fma2(swp(b), mk(1.f, -1.f), a); }

// x * (c + i d), c and d compile-time constants (the pair is an immediate)
BEGE_D c2 cmul(c2 x, float c, float d) { return fma2(swp(x), mk(-d, d), mul2(x, bc(c))); }
// x * w, w a run-time number:  (xr c, xi c) + (-xi d, xr d)
BEGE_D c2 cmulw(c2 x, float c, float d) {
    const c2 t = mul2(x, bc(c));
    return mk(fmaf(-im(x), d, re(t)), fmaf(re(x), d, im(t)));
}
BEGE_D c2 cmulw(c2 x, c2 w) { return cmulw(x, re(w), im(w)); }
// conj(h) * x = x * conj(h):  (xr hr, xi hr) + (xi hi, -xr hi)
BEGE_D c2 cmulc(c2 x, c2 h) {
    const c2 t = mul2(x, bc(re(h)));
    return mk(fmaf(im(x), im(h), re(t)), fmaf(-re(x), im(h), im(t)));
}

// 4-point DFT, DIR = +1: exp(+2 pi i jk/4) (inverse), DIR = -1: forward.  In place, natural order.
template <int DIR>
BEGE_D void fft4(c2& a0, c2& a1, c2& a2, c2& a3) {
    const c2 s02 = add2(a0, a2), d02 = sub2(a0, a2);
    const c2 s13 = add2(a1, a3), d13 = sub2(a1, a3);
    a0 = add2(s02, s13);
    a2 = sub2(s02, s13);
    if (DIR > 0) { a1 = add_i(d02, d13); a3 = sub_i(d02, d13); }
    else         { a1 = sub_i(d02, d13); a3 = add_i(d02, d13); }
}

// x * exp(DIR * 2 pi i m / 16), m a compile-time constant
template <int DIR, int M>
BEGE_D c2 tw16(c2 x) {
    constexpr int m = ((M % 16) + 16) % 16;
    constexpr float C1 = 0.92387953251128675613f, S1 = 0.38268343236508977173f, H = 0.70710678118654752440f;
    if (m == 0) return x;
    if (m == 4) return DIR > 0 ? mul2(swp(x), mk(-1.f, 1.f)) : mul2(swp(x), mk(1.f, -1.f));     // * (+-i)
    if (m == 8) return mul2(x, bc(-1.f));
    if (m == 12) return DIR > 0 ? mul2(swp(x), mk(1.f, -1.f)) : mul2(swp(x), mk(-1.f, 1.f));
    // cos / sin of 2 pi m / 16
    constexpr float c = (m == 1 || m == 15) ? C1 : (m == 2 || m == 14) ? H : (m == 3 || m == 13) ? S1
                      : (m == 5 || m == 11) ? -S1 : (m == 6 || m == 10) ? -H : /* 7, 9 */ -C1;
    constexpr float s0 = (m == 1 || m == 7) ? S1 : (m == 2 || m == 6) ? H : (m == 3 || m == 5) ? C1
                       : (m == 9 || m == 15) ? -S1 : (m == 10 || m == 14) ? -H : /* 11, 13 */ -C1;
    constexpr float s = DIR > 0 ? s0 : -s0;
    return cmul(x, c, s);
}

// 16-point DFT in registers: A[k] = sum_i a[i] exp(DIR 2 pi i ik/16); in place, natural order in and out.
// i = i0 + 4 i1, k = k0 + 4 k1:  radix-4 over i1, twiddle w16^(i0 k0), radix-4 over i0.
template <int DIR>
BEGE_D void fft16_plain(c2 (&a)[16]) {
#pragma unroll
    for (int i0 = 0; i0 < 4; ++i0) fft4<DIR>(a[i0], a[i0 + 4], a[i0 + 8], a[i0 + 12]);
    // now a[i0 + 4 k0] holds B[i0][k0]
    a[1 + 4 * 1] = tw16<DIR, 1>(a[1 + 4 * 1]);
    a[1 + 4 * 2] = tw16<DIR, 2>(a[1 + 4 * 2]);
    a[1 + 4 * 3] = tw16<DIR, 3>(a[1 + 4 * 3]);
    a[2 + 4 * 1] = tw16<DIR, 2>(a[2 + 4 * 1]);
    a[2 + 4 * 2] = tw16<DIR, 4>(a[2 + 4 * 2]);
    a[2 + 4 * 3] = tw16<DIR, 6>(a[2 + 4 * 3]);
    a[3 + 4 * 1] = tw16<DIR, 3>(a[3 + 4 * 1]);
    a[3 + 4 * 2] = tw16<DIR, 6>(a[3 + 4 * 2]);
    a[3 + 4 * 3] = tw16<DIR, 9>(a[3 + 4 * 3]);
    // radix-4 over i0 for each k0: inputs a[0 + 4k0], a[1 + 4k0], a[2 + 4k0], a[3 + 4k0] -> outputs k = k0 + 4 k1
#pragma unroll
    for (int k0 = 0; k0 < 4; ++k0) fft4<DIR>(a[4 * k0], a[4 * k0 + 1], a[4 * k0 + 2], a[4 * k0 + 3]);
    // a[4 k0 + k1] now holds A[k0 + 4 k1]: transpose the 4x4 index (register renaming, free when unrolled)
#pragma unroll
    for (int k0 = 0; k0 < 4; ++k0)
#pragma unroll
        for (int k1 = k0 + 1; k1 < 4; ++k1) { const c2 t = a[4 * k0 + k1]; a[4 * k0 + k1] = a[4 * k1 + k0]; a[4 * k1 + k0] = t; }
}

// y + k * (i x): one packed FMA (the half swap and the (-k, k) pair are operand forms, see the header comment)
BEGE_D c2 fma_i(c2 x, float k, c2 y) { return fma2(swp(x), mk(-k, k), y); }

// 16-point DFT in registers: A[k] = sum_i a[i] exp(DIR 2 pi i ik/16); in place, natural order in and out.
// i = i0 + 4 i1, k = k0 + 4 k1:  radix-4 over i1, twiddle w16^(i0 k0), radix-4 over i0.
//
// The twiddles of the middle step are never applied as multiplications of their own.  With s = DIR, T = tan(pi/8),
// C = cos(pi/8), H = cos(pi/4):
//   w16^1 = C (1 + i s T)      w16^2 = H (1 + i s)        w16^3 = i s C (1 - i s T)
//   w16^4 = i s                w16^6 = i s H (1 + i s)    w16^9 = -C (1 + i s T)
// so each twiddled input first becomes u = x + (i s t) x (ONE packed FMA, |t| <= 1), and the real scale C or H and
// the factor i s that remain ride on the FMAs of the radix-4 butterfly that follows (its sums and differences are
// formed up to the common scale of the odd pair, which the four output FMAs then carry).  Per quartet 11 (10 for
// k0 = 2) packed instructions instead of 14 (13): 72 per transform instead of 81, all single-rounded FMAs.
template <int DIR>
BEGE_D void fft16_fused(c2 (&a)[16]) {
    constexpr float s = DIR > 0 ? 1.f : -1.f;
    constexpr float C = 0.92387953251128675613f, H = 0.70710678118654752440f, T = 0.41421356237309504880f;
#pragma unroll
    for (int i0 = 0; i0 < 4; ++i0) fft4<DIR>(a[i0], a[i0 + 4], a[i0 + 8], a[i0 + 12]);
    // now a[i0 + 4 k0] holds B[i0][k0]; radix-4 over i0 for each k0, outputs k = k0 + 4 k1 left in a[4 k0 + k1]
    fft4<DIR>(a[0], a[1], a[2], a[3]);                       // k0 = 0: no twiddles
    {   // k0 = 1: twiddles w16^1, w16^2, w16^3
        const c2 x0 = a[4];
        const c2 u1 = fma_i(a[5], s * T, a[5]), u2 = fma_i(a[6], s, a[6]), u3 = fma_i(a[7], -s * T, a[7]);
        const c2 s02 = fma2(bc(H), u2, x0), d02 = fma2(bc(-H), u2, x0);
        const c2 s13 = fma_i(u3, s, u1), d13 = fma_i(u3, -s, u1);              // (y1 +- y3) / C
        a[4] = fma2(bc(C), s13, s02); a[6] = fma2(bc(-C), s13, s02);
        a[5] = fma_i(d13, s * C, d02); a[7] = fma_i(d13, -s * C, d02);
    }
    {   // k0 = 2: twiddles w16^2, w16^4, w16^6
        const c2 x0 = a[8];
        const c2 u1 = fma_i(a[9], s, a[9]), u3 = fma_i(a[11], s, a[11]);
        const c2 s02 = fma_i(a[10], s, x0), d02 = fma_i(a[10], -s, x0);
        const c2 s13 = fma_i(u3, s, u1), d13 = fma_i(u3, -s, u1);              // (y1 +- y3) / H
        a[8] = fma2(bc(H), s13, s02); a[10] = fma2(bc(-H), s13, s02);
        a[9] = fma_i(d13, s * H, d02); a[11] = fma_i(d13, -s * H, d02);
    }
    {   // k0 = 3: twiddles w16^3, w16^6, w16^9
        const c2 x0 = a[12];
        const c2 u1 = fma_i(a[13], -s * T, a[13]), u2 = fma_i(a[14], s, a[14]), u3 = fma_i(a[15], s * T, a[15]);
        const c2 s02 = fma_i(u2, s * H, x0), d02 = fma_i(u2, -s * H, x0);
        const c2 m13 = fma_i(u1, -s, u3), d13 = fma_i(u1, s, u3);              // -(y1 + y3) / C, (y1 - y3) / C
        a[12] = fma2(bc(-C), m13, s02); a[14] = fma2(bc(C), m13, s02);
        a[13] = fma_i(d13, s * C, d02); a[15] = fma_i(d13, -s * C, d02);
    }
    // a[4 k0 + k1] now holds A[k0 + 4 k1]: transpose the 4x4 index (register renaming, free when unrolled)
#pragma unroll
    for (int k0 = 0; k0 < 4; ++k0)
#pragma unroll
        for (int k1 = k0 + 1; k1 < 4; ++k1) { const c2 t = a[4 * k0 + k1]; a[4 * k0 + k1] = a[4 * k1 + k0]; a[4 * k1 + k0] = t; }
}

template <int DIR, bool FUSED = false>
BEGE_D void fft16(c2 (&a)[16]) { if constexpr (FUSED) fft16_fused<DIR>(a); else fft16_plain<DIR>(a); }

// warp-level sum over the 16 lanes of a half-warp (all lanes get the result), fixed order
BEGE_D float hw_sum16(float v) {
    v += __shfl_xor_sync(0xffffffffu, v, 8);
    v += __shfl_xor_sync(0xffffffffu, v, 4);
    v += __shfl_xor_sync(0xffffffffu, v, 2);
    v += __shfl_xor_sync(0xffffffffu, v, 1);
    return v;
}
// sum over the 16 lanes of a pass-2 row (lane map a = (lane & 7) | ((lane >> 4) << 3): xor 16 is a ^ 8), same tree
BEGE_D float row_sum16(float v) {
    v += __shfl_xor_sync(0xffffffffu, v, 16);
    v += __shfl_xor_sync(0xffffffffu, v, 4);
    v += __shfl_xor_sync(0xffffffffu, v, 2);
    v += __shfl_xor_sync(0xffffffffu, v, 1);
    return v;
}
BEGE_D float warp_sum32(float v) {
    v += __shfl_xor_sync(0xffffffffu, v, 16);
    return hw_sum16(v);
}

// "Tile layout" of a stored spectrum (bank, segments).  Tile b holds the columns k1 = 16 b + c; thread t = 16 c + g of a
// pass-1 team owns rows k2 = g + 16 i of column c.  Its kept row-blocks are stored in pairs (one 16-byte word per pair
// ip), and the words of one WARP (32 threads x NI/2 pairs) are contiguous: NI * 256 bytes that the warp brings in with
// one bulk copy and reads back with conflict-free 128-bit loads.  Index of the 16-byte word of (tile b, pair ip, thread t):
__host__ __device__ __forceinline__ uint32_t tile_word(int NI, int b, int ip, int t)
{
    return ((uint32_t)(b * 8 + (t >> 5)) * (uint32_t)(NI / 2) + (uint32_t)ip) * 32u + (uint32_t)(t & 31);
}

}  // namespace bege
