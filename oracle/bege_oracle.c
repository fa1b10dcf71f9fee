/*
 * bege_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, fp64 CPU statement of what the hot path of arXiv:1708.01609
 * (van Putten, "Deep searches for broadband extended gravitational-wave
 * emission bursts by heterogeneous computing") computes.  It shares no code,
 * header, table or constant with the CUDA path under paper_1708_01609_b200/
 * and neither imports the other.  Only tests/, __graft_entry__.smoke() and
 * the cpu_baseline / --impl reference legs of bench.py may load it.
 *
 * The method reaches exactly (up to rounding order) a result with a plain
 * definition -- circular cross-correlation (eq.3), its rms
 * (eq.6) and a threshold (eq.9) -- so the oracle is
 * that definition written out, in the paper's three steps (PAPER.md:89-92
 * eq.5): forward FFTs, conjugate product, inverse FFT.  No blocking, fusion or
 * reordering beyond that.  Readings of silent / garbled passages are the ones
 * listed in DESIGN.md ("Readings of the paper").
 *
 * Every function is pinned by tests/test_oracle_pins.py against something
 * other than itself (O(N^2) DFT, numpy.fft, direct time-domain sums, closed
 * forms, Gaussian tail laws, the paper's printed arithmetic).  Nothing here is
 * "parity unpinned".
 *
 * All complex arrays are interleaved double (re, im).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define BO_PI 3.14159265358979323846264338327950288

/* record of one tail sample, PAPER.md:221 (Table 3: sample offset, rho, template) */
typedef struct {
    uint32_t template_id;
    uint32_t lag;   /* m*N + n, eq.(13) */
    double   snr;   /* |z[n]| / sigma */
} bo_tail;

/* ------------------------------------------------------------------ FFT -- */
/*
 * Unnormalised DFT  A[k] = sum_n a[n] exp(sign * 2 pi i k n / N), N a power of
 * two, iterative radix-2 decimation in time.  sign = -1 is the forward
 * transform of PAPER.md:113 eq.(8) without its 1/N, sign = +1 the inverse
 * without normalisation.  Twiddles come straight from cos()/sin() of the exact
 * angle, never from a recurrence.
 */
int bo_fft(double* a, uint32_t N, int sign)
{
    if (N == 0 || (N & (N - 1)) != 0 || (sign != 1 && sign != -1)) return 1;
    uint32_t logN = 0;
    while ((1u << logN) < N) ++logN;

    /* bit-reversal permutation */
    for (uint32_t i = 0; i < N; ++i) {
        uint32_t r = 0;
        for (uint32_t b = 0; b < logN; ++b)
            if (i & (1u << b)) r |= 1u << (logN - 1 - b);
        if (r > i) {
            double tr = a[2 * i], ti = a[2 * i + 1];
            a[2 * i] = a[2 * r];  a[2 * i + 1] = a[2 * r + 1];
            a[2 * r] = tr;        a[2 * r + 1] = ti;
        }
    }
    /* twiddle table w[m] = exp(sign * 2 pi i m / N), m < N/2 */
    uint32_t half = N / 2;
    double* w = (double*)malloc(sizeof(double) * 2 * (half ? half : 1));
    if (!w) return 2;
    for (uint32_t m = 0; m < half; ++m) {
        double ang = 2.0 * BO_PI * (double)m / (double)N;
        w[2 * m]     = cos(ang);
        w[2 * m + 1] = (double)sign * sin(ang);
    }
    for (uint32_t len = 2; len <= N; len <<= 1) {
        uint32_t h = len / 2, step = N / len;
        for (uint32_t base = 0; base < N; base += len) {
            for (uint32_t j = 0; j < h; ++j) {
                double wr = w[2 * (j * step)], wi = w[2 * (j * step) + 1];
                uint32_t p = base + j, q = p + h;
                double br = a[2 * q] * wr - a[2 * q + 1] * wi;
                double bi = a[2 * q] * wi + a[2 * q + 1] * wr;
                double ar = a[2 * p], ai = a[2 * p + 1];
                a[2 * p] = ar + br;  a[2 * p + 1] = ai + bi;
                a[2 * q] = ar - br;  a[2 * q + 1] = ai - bi;
            }
        }
    }
    free(w);
    return 0;
}

/* ------------------------------------------------------------ template --- */
/*
 * One chirp template, PAPER.md:156 step (ii) ("a chirp template w of duration
 * tau = 1 s is extended by zeros to length N") with BASELINE.json's waveform:
 *   L = round(tau*fs);  t_n = n/fs;  w_n = 1/2 - 1/2 cos(2 pi n/(L-1))  (symmetric Hann)
 *   c_n = f0 t_n + 1/2 fdot t_n^2  (cycles);  h_n = w_n exp(i 2 pi c_n),  n < L
 *   h <- h / ||h||_2 ;  h_n = 0 for L <= n < N.
 */
int bo_template(double f0, double fdot, double tau, double fs, uint32_t N, double* h)
{
    long Ll = lround(tau * fs);
    if (Ll < 2 || (uint64_t)Ll > N) return 1;
    uint32_t L = (uint32_t)Ll;
    memset(h, 0, sizeof(double) * 2 * (size_t)N);
    double norm2 = 0.0;
    for (uint32_t n = 0; n < L; ++n) {
        double t = (double)n / fs;
        double wn = 0.5 - 0.5 * cos(2.0 * BO_PI * (double)n / (double)(L - 1));
        double c = f0 * t + 0.5 * fdot * t * t;
        c -= floor(c);                       /* exp(i 2 pi c) has period 1 in c */
        h[2 * n]     = wn * cos(2.0 * BO_PI * c);
        h[2 * n + 1] = wn * sin(2.0 * BO_PI * c);
        norm2 += h[2 * n] * h[2 * n] + h[2 * n + 1] * h[2 * n + 1];
    }
    double inv = 1.0 / sqrt(norm2);
    for (uint32_t n = 0; n < L; ++n) { h[2 * n] *= inv; h[2 * n + 1] *= inv; }
    return 0;
}

/* -------------------------------------------------------------- band ----- */
/*
 * Zero every bin whose |f_k| lies outside [lo, hi] (inclusive edges),
 * f_k = (k < N/2 ? k : k - N) fs/N.  PAPER.md:29, 58 ("bandpass filtered to
 * 350-2000 Hz"); DC and Nyquist fall outside any band with lo > 0, hi < fs/2,
 * which gives the zero mean PAPER.md:94 assumes.
 */
void bo_band_mask(double* X, uint32_t N, double fs, double lo, double hi)
{
    for (uint32_t k = 0; k < N; ++k) {
        double f = ((k < N / 2) ? (double)k : (double)k - (double)N) * fs / (double)N;
        double af = fabs(f);
        if (af < lo || af > hi) { X[2 * k] = 0.0; X[2 * k + 1] = 0.0; }
    }
}

/* Step (i): X = DFT_N(x) (forward, unnormalised), then band mask. */
int bo_segment_spectrum(const double* x, uint32_t N, double fs, double lo, double hi, double* X)
{
    memcpy(X, x, sizeof(double) * 2 * (size_t)N);
    int rc = bo_fft(X, N, -1);
    if (rc) return rc;
    bo_band_mask(X, N, fs, lo, hi);
    return 0;
}

/* ----------------------------------------------------------- correlate --- */
/*
 * One (template, segment) pair, eq.(5)-(7):
 *   H = DFT_N(h);  R[k] = conj(H[k]) X[k];                     (eq.5)
 *   sigma^2 = N^-2 sum_{k=0}^{N-1} |R[k]|^2                    (eq.7, complex form)
 *   z[n] = N^-1 sum_k R[k] exp(+2 pi i k n / N)                (eq.5, inverse FFT)
 * X is the band-masked segment spectrum, Hs the template SPECTRUM (already
 * transformed), both length N.  z may be NULL when only sigma is wanted.
 */
int bo_correlate_spectra(const double* X, const double* Hs, uint32_t N, double* z, double* sigma)
{
    double* R = z ? z : (double*)malloc(sizeof(double) * 2 * (size_t)N);
    if (!R) return 2;
    double acc = 0.0;
    for (uint32_t k = 0; k < N; ++k) {
        double hr = Hs[2 * k], hi = -Hs[2 * k + 1];          /* conj(H) */
        double xr = X[2 * k],  xi = X[2 * k + 1];
        double rr = hr * xr - hi * xi, ri = hr * xi + hi * xr;
        R[2 * k] = rr;  R[2 * k + 1] = ri;
        acc += rr * rr + ri * ri;
    }
    if (sigma) *sigma = sqrt(acc) / (double)N;
    if (!z) { free(R); return 0; }
    int rc = bo_fft(z, N, +1);
    if (rc) return rc;
    double invN = 1.0 / (double)N;
    for (uint32_t k = 0; k < 2 * N; ++k) z[k] *= invN;
    return 0;
}

/* Same, from the time-domain template h (length N, zero padded). */
int bo_correlate(const double* X, const double* h, uint32_t N, double* z, double* sigma)
{
    double* Hs = (double*)malloc(sizeof(double) * 2 * (size_t)N);
    if (!Hs) return 2;
    memcpy(Hs, h, sizeof(double) * 2 * (size_t)N);
    int rc = bo_fft(Hs, N, -1);
    if (!rc) rc = bo_correlate_spectra(X, Hs, N, z, sigma);
    free(Hs);
    return rc;
}

/*
 * The definition itself, eq.(3) discretised with circular indexing:
 *   z[n] = sum_{s=0}^{L-1} conj(h[s]) xhat[(n+s) mod N],
 * xhat the band-masked time series.  O(N L); for small N and for sampled lags.
 */
void bo_correlate_direct(const double* xhat, const double* h, uint32_t N, uint32_t L,
                         const uint32_t* lags, uint32_t n_lags, double* z)
{
    for (uint32_t i = 0; i < n_lags; ++i) {
        uint32_t n = lags ? lags[i] : i;
        double ar = 0.0, ai = 0.0;
        for (uint32_t s = 0; s < L; ++s) {
            uint32_t m = (n + s) % N;
            double hr = h[2 * s], hi = -h[2 * s + 1];
            double xr = xhat[2 * m], xi = xhat[2 * m + 1];
            ar += hr * xr - hi * xi;
            ai += hr * xi + hi * xr;
        }
        z[2 * i] = ar;  z[2 * i + 1] = ai;
    }
}

/* --------------------------------------------------------------- search -- */
/*
 * Whole path over a bank: for every template j and segment m form z_jm and
 * sigma_jm as above and keep the tails  |z[n]| > k sigma  (PAPER.md:116-120
 * eq.9, "we implicitly apply the inequality to the absolute value"), each as
 * {j, m*N+n, |z|/sigma} (eq.13).  sigma = 0 gives no tails.
 * Xs: S band-masked segment spectra (S*N complex).  sigma_out (may be NULL):
 * T*S values, template-major.  Records beyond cap are counted, not stored.
 * Returns the true number of tails.  Threads run over templates.
 */
uint64_t bo_search(const double* Xs, uint32_t S, const double* f0, const double* fdot, uint64_t T,
                   double tau, double fs, uint32_t N, double k_sigma,
                   bo_tail* tails, uint64_t cap, double* sigma_out, int n_threads, int* threads_used)
{
    uint64_t count = 0;
    int bad = 0;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
#pragma omp parallel
    {
#ifdef _OPENMP
#pragma omp single
        { if (threads_used) *threads_used = omp_get_num_threads(); }
#else
        if (threads_used) *threads_used = 1;
#endif
        double* Hs = (double*)malloc(sizeof(double) * 2 * (size_t)N);
        double* z  = (double*)malloc(sizeof(double) * 2 * (size_t)N);
        if (!Hs || !z) {
#pragma omp atomic write
            bad = 1;
        }
#pragma omp for schedule(dynamic, 1)
        for (int64_t j = 0; j < (int64_t)T; ++j) {
            if (bad) continue;
            if (bo_template(f0[j], fdot[j], tau, fs, N, Hs) || bo_fft(Hs, N, -1)) {
#pragma omp atomic write
                bad = 1;
                continue;
            }
            for (uint32_t m = 0; m < S; ++m) {
                double sigma = 0.0;
                bo_correlate_spectra(Xs + 2 * (size_t)m * N, Hs, N, z, &sigma);
                if (sigma_out) sigma_out[(size_t)j * S + m] = sigma;
                if (!(sigma > 0.0)) continue;
                double thr = k_sigma * sigma;
                for (uint32_t n = 0; n < N; ++n) {
                    double a = hypot(z[2 * n], z[2 * n + 1]);
                    if (a > thr) {
                        uint64_t slot;
#pragma omp atomic capture
                        slot = count++;
                        if (slot < cap) {
                            tails[slot].template_id = (uint32_t)j;
                            tails[slot].lag = m * N + n;
                            tails[slot].snr = a / sigma;
                        }
                    }
                }
            }
        }
        free(Hs);
        free(z);
    }
    return bad ? UINT64_MAX : count;
}


/* ------------------------------------------------------- max projection -- */
/*
 * The paper's default output, eq.(13)-(17) and Fig.4: per sample offset m*N + n keep only the
 * largest rho over all templates, with the template it came from ("In collecting B, we select data with maximal
 * rho values at t_{n+mN}"), provided it is a tail (eq.14, read with kappa as in eq.15; DESIGN.md
 * reading 6).  snr_out[m*N+n] = max_j |z_jm[n]|/sigma_jm over the templates with |z| > k sigma (0 if none),
 * id_out[m*N+n] = that template (UINT32_MAX if none); equal values go to the smaller template id, which makes the
 * result unique where the paper's racy update is not.  Plain serial loops, no threads.
 */
int bo_search_maxproj(const double* Xs, uint32_t S, const double* f0, const double* fdot, uint64_t T,
                      double tau, double fs, uint32_t N, double k_sigma, double* snr_out, uint32_t* id_out)
{
    double* Hs = (double*)malloc(sizeof(double) * 2 * (size_t)N);
    double* z  = (double*)malloc(sizeof(double) * 2 * (size_t)N);
    if (!Hs || !z) { free(Hs); free(z); return 2; }
    for (size_t i = 0; i < (size_t)S * N; ++i) { snr_out[i] = 0.0; id_out[i] = UINT32_MAX; }
    for (uint64_t j = 0; j < T; ++j) {
        if (bo_template(f0[j], fdot[j], tau, fs, N, Hs) || bo_fft(Hs, N, -1)) { free(Hs); free(z); return 1; }
        for (uint32_t m = 0; m < S; ++m) {
            double sigma = 0.0;
            bo_correlate_spectra(Xs + 2 * (size_t)m * N, Hs, N, z, &sigma);
            if (!(sigma > 0.0)) continue;
            for (uint32_t n = 0; n < N; ++n) {
                double a = hypot(z[2 * n], z[2 * n + 1]);
                if (a > k_sigma * sigma) {
                    double r = a / sigma;
                    size_t i = (size_t)m * N + n;
                    if (r > snr_out[i]) { snr_out[i] = r; id_out[i] = (uint32_t)j; }   /* j ascending: ties keep the smaller id */
                }
            }
        }
    }
    free(Hs); free(z);
    return 0;
}


/* ------------------------------------------------------- band threshold -- */
/*
 * PAPER.md:281 (sec.5): "excess tail sizes can conceivably be curtailed by generalising (9) to a finite band,
 * kappa_1 sigma > rho(t_n) > kappa_2 sigma".  Same loops as bo_search (serial), with both inequalities strict:
 * keep n iff k_lo*sigma < |z[n]| < k_hi*sigma.  Returns the true count; records beyond cap are not stored.
 */
uint64_t bo_search_band(const double* Xs, uint32_t S, const double* f0, const double* fdot, uint64_t T,
                        double tau, double fs, uint32_t N, double k_lo, double k_hi, bo_tail* tails, uint64_t cap)
{
    double* Hs = (double*)malloc(sizeof(double) * 2 * (size_t)N);
    double* z  = (double*)malloc(sizeof(double) * 2 * (size_t)N);
    if (!Hs || !z) { free(Hs); free(z); return UINT64_MAX; }
    uint64_t count = 0;
    for (uint64_t j = 0; j < T; ++j) {
        if (bo_template(f0[j], fdot[j], tau, fs, N, Hs) || bo_fft(Hs, N, -1)) { free(Hs); free(z); return UINT64_MAX; }
        for (uint32_t m = 0; m < S; ++m) {
            double sigma = 0.0;
            bo_correlate_spectra(Xs + 2 * (size_t)m * N, Hs, N, z, &sigma);
            if (!(sigma > 0.0)) continue;
            for (uint32_t n = 0; n < N; ++n) {
                double a = hypot(z[2 * n], z[2 * n + 1]);
                if (a > k_lo * sigma && a < k_hi * sigma) {
                    if (count < cap) {
                        tails[count].template_id = (uint32_t)j;
                        tails[count].lag = m * N + n;
                        tails[count].snr = a / sigma;
                    }
                    ++count;
                }
            }
        }
    }
    free(Hs); free(z);
    return count;
}

/* ------------------------------------------------------------ dual stream -- */
/*
 * The paper's own setting, PAPER.md:155 step (i): "FFT is applied to arrays of complex numbers, merging pairs of real
 * H1 and L1 data", x = H1 + i L1, filtered with REAL chirp templates, so that one complex correlation
 * holds both detectors' outputs:  z[n] = sum_s w[s] x[(n+s) mod N]  =>  rho_1 = Re z (H1),  rho_2 = Im z (L1).
 *
 * Real template (reading 23): the real part of BASELINE.json's waveform,
 *   w_n = hann_L[n] cos(2 pi c_n),  c_n = f0 t_n + fdot t_n^2 / 2,  n < L;  w <- w / ||w||_2;  zero padded to N.
 */
int bo_template_real(double f0, double fdot, double tau, double fs, uint32_t N, double* h)
{
    long Ll = lround(tau * fs);
    if (Ll < 2 || (uint64_t)Ll > N) return 1;
    uint32_t L = (uint32_t)Ll;
    memset(h, 0, sizeof(double) * 2 * (size_t)N);
    double norm2 = 0.0;
    for (uint32_t n = 0; n < L; ++n) {
        double t = (double)n / fs;
        double wn = 0.5 - 0.5 * cos(2.0 * BO_PI * (double)n / (double)(L - 1));
        double c = f0 * t + 0.5 * fdot * t * t;
        c -= floor(c);
        h[2 * n] = wn * cos(2.0 * BO_PI * c);
        norm2 += h[2 * n] * h[2 * n];
    }
    double inv = 1.0 / sqrt(norm2);
    for (uint32_t n = 0; n < L; ++n) h[2 * n] *= inv;
    return 0;
}

/*
 * Time-symmetric real template, PAPER.md:70 (Fig.2 caption): "The chirps used in butterfly filtering are symmetric in
 * time, obtained by superposition of chirp forward and backward in time, suitable in searches for both ascending and
 * descending chirps."  With u_n = hann_L[n] cos(2 pi c_n) the one-way template of bo_template_real before normalisation
 * (reading 27):
 *   w_n = u_n + u_(L-1-n),  n < L;   w <- w / ||w||_2;   zero padded to N.
 * The Hann window is itself symmetric, so w_n = hann_L[n] (cos 2 pi c_n + cos 2 pi c_(L-1-n)) and w_n = w_(L-1-n).
 */
int bo_template_real_sym(double f0, double fdot, double tau, double fs, uint32_t N, double* h)
{
    long Ll = lround(tau * fs);
    if (Ll < 2 || (uint64_t)Ll > N) return 1;
    uint32_t L = (uint32_t)Ll;
    memset(h, 0, sizeof(double) * 2 * (size_t)N);
    double norm2 = 0.0;
    for (uint32_t n = 0; n < L; ++n) {
        double wn = 0.5 - 0.5 * cos(2.0 * BO_PI * (double)n / (double)(L - 1));
        double t = (double)n / fs, tr = (double)(L - 1 - n) / fs;
        double c = f0 * t + 0.5 * fdot * t * t, cr = f0 * tr + 0.5 * fdot * tr * tr;
        c -= floor(c); cr -= floor(cr);
        h[2 * n] = wn * (cos(2.0 * BO_PI * c) + cos(2.0 * BO_PI * cr));
        norm2 += h[2 * n] * h[2 * n];
    }
    double inv = 1.0 / sqrt(norm2);
    for (uint32_t n = 0; n < L; ++n) h[2 * n] *= inv;
    return 0;
}

/*
 * One (real template, packed segment) pair.  z as in bo_correlate_spectra (eq.5); per detector
 * stream the standard deviation of its REAL output by the definition PAPER.md:96 eq.(6):
 *   sigma_1^2 = N^-1 sum_n (Re z[n])^2,   sigma_2^2 = N^-1 sum_n (Im z[n])^2.
 * Hs: template spectrum.  z may be NULL.
 */
int bo_correlate_dual(const double* X, const double* Hs, uint32_t N, double* z, double* sigma1, double* sigma2)
{
    double* zz = z ? z : (double*)malloc(sizeof(double) * 2 * (size_t)N);
    if (!zz) return 2;
    for (uint32_t k = 0; k < N; ++k) {                    /* R = conj(H) X */
        double hr = Hs[2 * k], hi = Hs[2 * k + 1], xr = X[2 * k], xi = X[2 * k + 1];
        zz[2 * k]     = hr * xr + hi * xi;
        zz[2 * k + 1] = hr * xi - hi * xr;
    }
    int rc = bo_fft(zz, N, +1);
    double s1 = 0.0, s2 = 0.0, inv = 1.0 / (double)N;
    for (uint32_t n = 0; n < N; ++n) {
        zz[2 * n] *= inv; zz[2 * n + 1] *= inv;
        s1 += zz[2 * n] * zz[2 * n];
        s2 += zz[2 * n + 1] * zz[2 * n + 1];
    }
    *sigma1 = sqrt(s1 * inv);
    *sigma2 = sqrt(s2 * inv);
    if (!z) free(zz);
    return rc;
}

/*
 * The same two standard deviations from the SPECTRUM, eq.(7) (Parseval for a real series, whose Fourier
 * coefficients are Hermitian: the sum over half the spectrum, times sqrt 2).  The coefficients of Re z and Im z are
 * the Hermitian and anti-Hermitian parts of R:  A[k] = (R[k] + conj(R[N-k]))/2,  B[k] = (R[k] - conj(R[N-k]))/(2i);
 * sigma_1 = (sqrt 2 / N) sqrt( sum_{k=1}^{N/2-1} |A[k]|^2 + (|A[0]|^2 + |A[N/2]|^2)/2 ), likewise sigma_2 with B (the
 * paper drops the DC and Nyquist terms, which vanish for band-limited data).  Used by the pins only.
 */
void bo_sigma_dual_parseval(const double* X, const double* Hs, uint32_t N, double* sigma1, double* sigma2)
{
    double sa = 0.0, sb = 0.0;
    for (uint32_t k = 0; k <= N / 2; ++k) {
        uint32_t km = (N - k) % N;
        double r1r = Hs[2 * k] * X[2 * k] + Hs[2 * k + 1] * X[2 * k + 1];           /* R[k]     */
        double r1i = Hs[2 * k] * X[2 * k + 1] - Hs[2 * k + 1] * X[2 * k];
        double r2r = Hs[2 * km] * X[2 * km] + Hs[2 * km + 1] * X[2 * km + 1];       /* R[N-k]   */
        double r2i = Hs[2 * km] * X[2 * km + 1] - Hs[2 * km + 1] * X[2 * km];
        double ar = 0.5 * (r1r + r2r), ai = 0.5 * (r1i - r2i);                       /* (R[k] + conj R[N-k]) / 2 */
        double br = 0.5 * (r1i + r2i), bi = -0.5 * (r1r - r2r);                      /* (R[k] - conj R[N-k]) / 2i */
        double w = (k == 0 || k == N / 2) ? 0.5 : 1.0;
        sa += w * (ar * ar + ai * ai);
        sb += w * (br * br + bi * bi);
    }
    *sigma1 = sqrt(2.0) / (double)N * sqrt(sa);
    *sigma2 = sqrt(2.0) / (double)N * sqrt(sb);
}

/*
 * Dual-stream search in the paper's output form, Table 3 ("sample offset i, rho_1, f_1, rho_2, f_2 ...
 * Zeros represent no hit"): per sample offset m*N + n and per detector stream d the largest |rho_d|/sigma_d over the
 * bank among the hits |rho_d[n]| > k sigma_d (eq.9 on each real stream, two-sided), with its template
 * ("we select data with maximal rho values"); 0 / UINT32_MAX where no template hits; ties go to the
 * smaller template id.  sigma_out (may be NULL): T*S*2 values, [j][m][stream].  Plain serial loops.
 */
static int search_dual_impl(const double* Xs, uint32_t S, const double* f0, const double* fdot, uint64_t T,
                            double tau, double fs, uint32_t N, double k_sigma,
                            double* snr1, uint32_t* id1, double* snr2, uint32_t* id2, double* sigma_out, int symmetric)
{
    double* Hs = (double*)malloc(sizeof(double) * 2 * (size_t)N);
    double* z  = (double*)malloc(sizeof(double) * 2 * (size_t)N);
    if (!Hs || !z) { free(Hs); free(z); return 2; }
    for (size_t i = 0; i < (size_t)S * N; ++i) { snr1[i] = snr2[i] = 0.0; id1[i] = id2[i] = UINT32_MAX; }
    for (uint64_t j = 0; j < T; ++j) {
        if ((symmetric ? bo_template_real_sym(f0[j], fdot[j], tau, fs, N, Hs) : bo_template_real(f0[j], fdot[j], tau, fs, N, Hs))
            || bo_fft(Hs, N, -1)) { free(Hs); free(z); return 1; }
        for (uint32_t m = 0; m < S; ++m) {
            double s1 = 0.0, s2 = 0.0;
            bo_correlate_dual(Xs + 2 * (size_t)m * N, Hs, N, z, &s1, &s2);
            if (sigma_out) { sigma_out[((size_t)j * S + m) * 2] = s1; sigma_out[((size_t)j * S + m) * 2 + 1] = s2; }
            for (uint32_t n = 0; n < N; ++n) {
                size_t i = (size_t)m * N + n;
                double a1 = fabs(z[2 * n]), a2 = fabs(z[2 * n + 1]);
                if (s1 > 0.0 && a1 > k_sigma * s1 && a1 / s1 > snr1[i]) { snr1[i] = a1 / s1; id1[i] = (uint32_t)j; }
                if (s2 > 0.0 && a2 > k_sigma * s2 && a2 / s2 > snr2[i]) { snr2[i] = a2 / s2; id2[i] = (uint32_t)j; }
            }
        }
    }
    free(Hs); free(z);
    return 0;
}

int bo_search_dual(const double* Xs, uint32_t S, const double* f0, const double* fdot, uint64_t T,
                   double tau, double fs, uint32_t N, double k_sigma,
                   double* snr1, uint32_t* id1, double* snr2, uint32_t* id2, double* sigma_out)
{
    return search_dual_impl(Xs, S, f0, fdot, T, tau, fs, N, k_sigma, snr1, id1, snr2, id2, sigma_out, 0);
}

/* The same search with the time-symmetric templates of bo_template_real_sym. */
int bo_search_dual_sym(const double* Xs, uint32_t S, const double* f0, const double* fdot, uint64_t T,
                       double tau, double fs, uint32_t N, double k_sigma,
                       double* snr1, uint32_t* id1, double* snr2, uint32_t* id2, double* sigma_out)
{
    return search_dual_impl(Xs, S, f0, fdot, T, tau, fs, N, k_sigma, snr1, id1, snr2, id2, sigma_out, 1);
}

/*
 * H1-L1 coincidences of a dual-stream output, PAPER.md:219 ("simultaneous hits with frequency pairs (f_1, f_2) of H1
 * and L1 that are relatively close, |f_1 - f_2| < Delta"): offsets where both streams hold a hit, and among those the
 * ones whose templates' start frequencies differ by less than delta_hz.
 */
void bo_dual_coincidences(const uint32_t* id1, const uint32_t* id2, uint64_t n, const double* f0, double delta_hz,
                          uint64_t* n_simultaneous, uint64_t* n_coincident)
{
    uint64_t a = 0, b = 0;
    for (uint64_t i = 0; i < n; ++i) {
        if (id1[i] != UINT32_MAX && id2[i] != UINT32_MAX) {
            ++a;
            if (fabs(f0[id1[i]] - f0[id2[i]]) < delta_hz) ++b;
        }
    }
    *n_simultaneous = a; *n_coincident = b;
}

/* PAPER.md:134 eq.(10), :160: nominal flops of one FFT_N. */
double bo_fft_flops(uint32_t N)
{
    return 5.0 * (double)N * log2((double)N);
}
