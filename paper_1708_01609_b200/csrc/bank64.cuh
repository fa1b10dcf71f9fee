// a1 -- template spectra in fp64 arithmetic, rounded to fp32 once at the end (PAPER.md:156 step ii).
//
// Why fp64: templates at the edge of the (f0, fdot) plane (e.g. 350 Hz, -400 Hz/s of BASELINE.json configs[2..4])
// keep only a small part of their energy inside the analysis band.  An fp32 transform of the unit-norm template has
// an absolute error of ~1e-7 per bin, i.e. a relative error of up to 1e-3 on such in-band bins, and the correlation
// then misses the 2e-5 parity bound (measured: 4.5e-4).  The bank is generated once, off the timed path, so the
// transform runs in fp64 (own radix-16 kernels below, same index maps as the fp32 kernels in bege.cu) and every
// stored bin carries one fp32 rounding.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

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

// step A: chirp synthesis (fp64 phase) + pruned row DFTs.  grid (16, templates in batch), 256 threads.
// Same index map as k_fwd_rows_data (bege.cu): CTA (ia, jl) owns the rows nl = ga + 16 ia; only nh < 16 inputs are
// non-zero (L <= 4096); output G[k1 = p + 16 q][nl] times wN^(-nl k1), tile layout, fp64.
// tw256d[m] = exp(2 pi i m / 256), twNd[m] = exp(2 pi i m / N) (host-built double tables).
__global__ void __launch_bounds__(256)
k_bank_rows64(const double* __restrict__ f0, const double* __restrict__ fdot, uint64_t j0, double fs, uint32_t L,
              double inv_norm, const d2* __restrict__ tw256d, const d2* __restrict__ twNd, d2* __restrict__ G)
{
    __shared__ d2 samp[16][16];          // [nh][ga]
    const int t = threadIdx.x, ia = blockIdx.x;
    const uint64_t jl = blockIdx.y;
    {
        const int ga = t & 15, nh = t >> 4;
        const uint32_t n = ga + 16 * ia + 256 * nh;
        d2 s = dmk(0.0, 0.0);
        if (n < L) {
            const double tt = (double)n / fs;
            const double cyc = f0[j0 + jl] * tt + 0.5 * fdot[j0 + jl] * tt * tt;
            const double fr = cyc - floor(cyc);
            double sn, cs;
            sincospi(2.0 * fr, &sn, &cs);
            const double w = (0.5 - 0.5 * cospi(2.0 * (double)n / (double)(L - 1))) * inv_norm;
            s = dmk(w * cs, w * sn);
        }
        samp[nh][ga] = s;
    }
    __syncthreads();
    const int ga = t >> 4, p = t & 15;
    const int nl = ga + 16 * ia;
    d2 v[16];
#pragma unroll
    for (int nh = 0; nh < 16; ++nh) {
        const d2 w = tw256d[(p * nh) & 255];                    // exp(+2 pi i nh p / 256)
        v[nh] = dmul(samp[nh][ga], w.x, -w.y);
    }
    dfft16f(v);
    d2* out = G + jl * (uint64_t)65536;
#pragma unroll
    for (int q = 0; q < 16; ++q) {
        const int k1 = p + 16 * q;
        const d2 w = twNd[(nl * k1) & 65535];                   // exp(+2 pi i nl k1 / N)
        out[((q * 16 + ia) * 16 + p) * 16 + ga] = dmul(v[q], w.x, -w.y);
    }
}

// step B: 256-point column DFTs over nl in fp64, stores the kept row-blocks [I0, I0 + NI) as fp32 in tile layout.
// grid (16 tiles, batch), 256 threads, 64 KiB dynamic shared memory ([16 half-warps][256] d2, xor swizzled).
__global__ void __launch_bounds__(256)
k_bank_cols64(const d2* __restrict__ G, float2* __restrict__ out, uint64_t out_stride, int I0, int NI,
              const d2* __restrict__ tw256d)
{
    extern __shared__ __align__(16) unsigned char bank64_smem[];
    d2* sm = reinterpret_cast<d2*>(bank64_smem);
    const int t = threadIdx.x, b = blockIdx.x;
    const uint64_t jl = blockIdx.y;
    const int c = t >> 4, g = t & 15;
    const d2* in = G + jl * (uint64_t)65536 + (uint64_t)b * 4096;
    d2 v[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) v[i] = in[(i * 16 + c) * 16 + g];
    dfft16f(v);
    d2* priv = sm + c * 256;
#pragma unroll
    for (int p = 0; p < 16; ++p) {
        const d2 w = tw256d[(g * p) & 255];
        priv[(g << 4) + (p ^ g)] = dmul(v[p], w.x, -w.y);
    }
    __syncwarp();
#pragma unroll
    for (int a = 0; a < 16; ++a) v[a] = priv[(a << 4) + (g ^ a)];
    __syncwarp();
    dfft16f(v);
    // lane p = g holds k2 = p + 16 q; stored layout: row-blocks in pairs, one 16-byte word per thread and pair
    float4* o = reinterpret_cast<float4*>(out + jl * out_stride + (uint64_t)b * NI * 256) + t;
#pragma unroll
    for (int ip = 0; ip < 8; ++ip) {
        if (2 * ip < NI) {
            float4 w;
            if (I0 == 1) { w = make_float4((float)v[(2 * ip + 1) & 15].x, (float)v[(2 * ip + 1) & 15].y,
                                           (float)v[(2 * ip + 2) & 15].x, (float)v[(2 * ip + 2) & 15].y); }
            else         { w = make_float4((float)v[2 * ip].x, (float)v[2 * ip].y,
                                           (float)v[(2 * ip + 1) & 15].x, (float)v[(2 * ip + 1) & 15].y); }
            o[ip * 256] = w;
        }
    }
}

}  // namespace bege
