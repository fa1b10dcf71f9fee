// a1 -- template spectra in fp64 arithmetic, rounded to fp32 once at the end (PAPER.md:156 step ii).
//
// Why fp64: templates at the edge of the (f0, fdot) plane (e.g. 350 Hz, -400 Hz/s of BASELINE.json configs[2..4])
// keep only a small part of their energy inside the analysis band.  An fp32 transform of the unit-norm template has
// an absolute error of ~1e-7 per bin, i.e. a relative error of up to 1e-3 on such in-band bins, and the correlation
// then misses the 2e-5 parity bound (measured: 4.5e-4).  The bank is generated once, off the timed path, so the
// transform runs in fp64 (own radix-16 kernel below) and every stored bin carries one fp32 rounding.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>
#include "cplx.cuh"

namespace bege {

struct d2 { double x, y; };
#define BEGE_DD __device__ __forceinline__
BEGE_DD d2 dmk(double x, double y) { d2 r; r.x = x; r.y = y; return r; }
BEGE_DD d2 dadd(d2 a, d2 b) { return dmk(a.x + b.x, a.y + b.y); }
BEGE_DD d2 dsub(d2 a, d2 b) { return dmk(a.x - b.x, a.y - b.y); }
BEGE_DD d2 dmul(d2 a, double c, double s) { return dmk(a.x * c - a.y * s, a.x * s + a.y * c); }   // a * (c + i s)
BEGE_DD d2 dmuli(d2 a) { return dmk(-a.y, a.x); }                                                  // a * i

// forward 4-point DFT (exp(-2 pi i jk/4)), in place, natural order
BEGE_DD void dfft4f(d2& a0, d2& a1, d2& a2, d2& a3)
{
    const d2 s02 = dadd(a0, a2), d02 = dsub(a0, a2), s13 = dadd(a1, a3), d13 = dsub(a1, a3);
    a0 = dadd(s02, s13);
    a2 = dsub(s02, s13);
    a1 = dsub(d02, dmuli(d13));
    a3 = dadd(d02, dmuli(d13));
}

// forward 16-point DFT in registers, natural order in and out (i = i0 + 4 i1, k = k0 + 4 k1)
BEGE_DD void dfft16f(d2 (&a)[16])
{
    constexpr double C1 = 0.92387953251128675613, S1 = 0.38268343236508977173, H = 0.70710678118654752440;
#pragma unroll
    for (int i0 = 0; i0 < 4; ++i0) dfft4f(a[i0], a[i0 + 4], a[i0 + 8], a[i0 + 12]);
    // a[i0 + 4 k0] *= exp(-2 pi i i0 k0 / 16):  (cos, sin) of 2 pi m / 16 for m = 1, 2, 3, 4, 6, 9
    a[1 + 4 * 1] = dmul(a[1 + 4 * 1], C1, -S1);
    a[1 + 4 * 2] = dmul(a[1 + 4 * 2], H, -H);
    a[1 + 4 * 3] = dmul(a[1 + 4 * 3], S1, -C1);
    a[2 + 4 * 1] = dmul(a[2 + 4 * 1], H, -H);
    a[2 + 4 * 2] = dmul(a[2 + 4 * 2], 0.0, -1.0);
    a[2 + 4 * 3] = dmul(a[2 + 4 * 3], -H, -H);
    a[3 + 4 * 1] = dmul(a[3 + 4 * 1], S1, -C1);
    a[3 + 4 * 2] = dmul(a[3 + 4 * 2], -H, -H);
    a[3 + 4 * 3] = dmul(a[3 + 4 * 3], -C1, S1);
#pragma unroll
    for (int k0 = 0; k0 < 4; ++k0) dfft4f(a[4 * k0], a[4 * k0 + 1], a[4 * k0 + 2], a[4 * k0 + 3]);
#pragma unroll
    for (int k0 = 0; k0 < 4; ++k0)
#pragma unroll
        for (int k1 = k0 + 1; k1 < 4; ++k1) { const d2 t = a[4 * k0 + k1]; a[4 * k0 + k1] = a[4 * k1 + k0]; a[4 * k1 + k0] = t; }
}

// One kernel, no global scratch: H[16 m + r] = sum_n (h[n] e^(-2 pi i r n / N)) e^(-2 pi i m n / 4096), n < 4096 -- the
// N = 65536-point spectrum of a template of at most 4096 samples is 16 interleaved 4096-point transforms of the template
// times a slow modulation (r = k mod 16).  A CTA of 256 threads owns a template: it synthesises the 4096 samples once
// (fp64 phase: three sincospi per thread, the rest by the exact recurrences of a quadratic phase) and runs the 16
// transforms one after the other in shared memory (16 x 16 x 16, two exchanges, xor-swizzled), so the only global
// traffic is the 448 KiB of fp32 spectrum it stores, in 256-byte runs.  grid = persistent CTAs over the templates.
//   4096-point index maps:  n = nl + 256 nh,  nl = l0 + 16 l1;   m = m1 + 16 (q0 + 16 q1)
//     S1: thread nl:        over nh -> m1, input twiddle w256^(-r nh) (the modulation), output twiddle wN^(-nl (r + 16 m1))
//     S2: thread (m1, l0):  over l1 -> q0, twiddle w256^(-l0 q0)
//     S3: thread (m1, q0):  over l0 -> q1
//   bin k = 16 m + r = (16 m1 + r) + 256 (q0 + 16 q1): tile b = m1, column c = r, lane g = q0, row-block i = q1.
// hann: L window values times 1 / ||h|| (host, fp64).  tw256d[m] = exp(2 pi i m / 256).
constexpr int kBankSmem = 3 * 4096 * 16;   // samples + two exchange buffers, fp64 complex

// real_tpl = 1: the real template of the dual-stream search, w_n = hann_n cos(2 pi c_n) / ||.||; its
// norm depends on the template and is formed here (fp64 block sum).
// real_tpl = 2: the time-symmetric real template ("superposition of chirp forward and backward in time"),
// w_n = hann_n (cos 2 pi c_n + cos 2 pi c_(L-1-n)) / ||.||.  The reversed phase is itself a quadratic in n,
// c_(L-1-n) = c(T') - (f0 + fdot T') t_n + fdot t_n^2 / 2 with T' = (L-1)/fs, so it runs on a second recurrence.
__global__ void __launch_bounds__(256, 1)
k_bank_gen64(const double* __restrict__ f0, const double* __restrict__ fdot, uint64_t T, double fs, uint32_t L,
             const double* __restrict__ hann, const d2* __restrict__ tw256d, float2* __restrict__ out,
             uint64_t out_stride, int I0, int NI, int real_tpl)
{
    __shared__ double red[8];
    extern __shared__ __align__(16) unsigned char bank64_smem[];
    d2* base = reinterpret_cast<d2*>(bank64_smem);          // [nh][nl]
    // two exchange buffers alternate over r ([m1][l0][l1 ^ l0] after S1); S2 rewrites its own row in place ([m1][l0][q0 ^ l0])
    d2* const buf0 = base + 4096;
    const int t = threadIdx.x;
    const int l0 = t & 15, l1 = t >> 4;                      // S1: nl = t = l0 + 16 l1
    const int m1 = t >> 4;                                   // S2: (m1, l0);  S3: (m1, q0 = l0)
    // exp(-2 pi i nl / N) and its 16th power: the thread's S1 output twiddle is rho^(r + 16 m1)
    d2 rho, rho16;
    {
        double sn, cs;
        sincospi(2.0 * (double)t / 65536.0, &sn, &cs); rho = dmk(cs, -sn);
        sincospi(2.0 * (double)(16 * t) / 65536.0, &sn, &cs); rho16 = dmk(cs, -sn);
    }
    for (uint64_t j = blockIdx.x; j < T; j += gridDim.x) {
        {   // samples n = t + 256 nh: z_nh = exp(2 pi i c(n)), c(n) = f0 n/fs + fdot (n/fs)^2 / 2 cycles;
            // z_(nh+1) = z_nh D_nh, D_(nh+1) = D_nh C (second differences of a quadratic are constant)
            const double f = f0[j], fd = fdot[j], tt = (double)t / fs, dt = 256.0 / fs;
            auto expc = [](double cyc) { double sn, cs; sincospi(2.0 * (cyc - floor(cyc)), &sn, &cs); return dmk(cs, sn); };
            d2 z = expc(f * tt + 0.5 * fd * tt * tt);
            d2 D = expc(f * dt + 0.5 * fd * (2.0 * tt * dt + dt * dt));
            const d2 C = expc(fd * dt * dt);
            // the time-reversed chirp (real_tpl = 2): start frequency -(f0 + fdot T'), same second difference
            const double Tp = (double)(L - 1) / fs, fr = -(f + fd * Tp);
            d2 zr = expc(f * Tp + 0.5 * fd * Tp * Tp + fr * tt + 0.5 * fd * tt * tt);
            d2 Dr = expc(fr * dt + 0.5 * fd * (2.0 * tt * dt + dt * dt));
            double n2 = 0.0;
#pragma unroll
            for (int nh = 0; nh < 16; ++nh) {
                const uint32_t n = (uint32_t)t + 256u * nh;
                const double w = n < L ? hann[n] : 0.0;
                const double xr = real_tpl == 2 ? w * (z.x + zr.x) : w * z.x;
                base[nh * 256 + t] = dmk(xr, real_tpl ? 0.0 : w * z.y);
                n2 += xr * xr;
                z = dmul(z, D.x, D.y);
                D = dmul(D, C.x, C.y);
                if (real_tpl == 2) { zr = dmul(zr, Dr.x, Dr.y); Dr = dmul(Dr, C.x, C.y); }
            }
            if (real_tpl) {                                  // unit L2 norm of the real template
#pragma unroll
                for (int d = 16; d >= 1; d >>= 1) n2 += __shfl_xor_sync(0xffffffffu, n2, d);
                if ((t & 31) == 0) red[t >> 5] = n2;
                __syncthreads();
                double tot = 0.0;
#pragma unroll
                for (int w8 = 0; w8 < 8; ++w8) tot += red[w8];
                const double inv = 1.0 / sqrt(tot);
#pragma unroll
                for (int nh = 0; nh < 16; ++nh) base[nh * 256 + t].x *= inv;
            }
        }
        __syncthreads();
        d2 rho_r = dmk(1.0, 0.0);                            // rho^r
        float4* o = reinterpret_cast<float4*>(out + j * out_stride);
        for (int r = 0; r < 16; ++r) {
            d2* const buf = buf0 + 4096 * (r & 1);
            d2 v[16];
            // ---- S1
#pragma unroll
            for (int nh = 0; nh < 16; ++nh) {
                const d2 w = tw256d[(r * nh) & 255];
                v[nh] = dmul(base[nh * 256 + t], w.x, -w.y);
            }
            dfft16f(v);
            {
                d2 w = rho_r;
#pragma unroll
                for (int mm = 0; mm < 16; ++mm) {
                    buf[mm * 256 + l0 * 16 + (l1 ^ l0)] = dmul(v[mm], w.x, w.y);
                    w = dmul(w, rho16.x, rho16.y);
                }
            }
            rho_r = dmul(rho_r, rho.x, rho.y);
            __syncthreads();
            // ---- S2: thread (m1, l0), in place on the row it has read
#pragma unroll
            for (int k = 0; k < 16; ++k) v[k] = buf[m1 * 256 + l0 * 16 + (k ^ l0)];
            dfft16f(v);
#pragma unroll
            for (int q0 = 0; q0 < 16; ++q0) {
                const d2 w = tw256d[(l0 * q0) & 255];
                buf[m1 * 256 + l0 * 16 + (q0 ^ l0)] = dmul(v[q0], w.x, -w.y);
            }
            // S3 of thread (m1, q0) reads what the 16 threads (m1, .) -- its own half-warp -- have written: no CTA barrier.
            // The buffer of r is written again by S1 of r + 2, after the barrier of r + 1, which every warp reaches only
            // after its S3 of r: one CTA barrier per transform, and the warps are free to drift between them (fp64
            // arithmetic and shared-memory exchanges of different warps then overlap).
            __syncwarp();
            // ---- S3: thread (m1, q0 = l0)
#pragma unroll
            for (int k = 0; k < 16; ++k) v[k] = buf[m1 * 256 + k * 16 + (l0 ^ k)];
            dfft16f(v);
            // v[q1] = H[k], k = (16 m1 + r) + 256 (q0 + 16 q1): tile m1, thread 16 r + q0, row-block q1 (stored in pairs)
            float4* ot = o + tile_word(NI, m1, 0, 16 * r + l0);       // + 32 ip
#pragma unroll
            for (int ip = 0; ip < 8; ++ip) {
                if (2 * ip < NI) {
                    float4 w;
                    if (I0 == 1) w = make_float4((float)v[(2 * ip + 1) & 15].x, (float)v[(2 * ip + 1) & 15].y,
                                                 (float)v[(2 * ip + 2) & 15].x, (float)v[(2 * ip + 2) & 15].y);
                    else         w = make_float4((float)v[2 * ip].x, (float)v[2 * ip].y,
                                                 (float)v[(2 * ip + 1) & 15].x, (float)v[(2 * ip + 1) & 15].y);
                    ot[ip * 32] = w;
                }
            }
        }
        // the next template's samples overwrite `base` only after every thread has passed the barriers of r = 15
    }
}

}  // namespace bege
