/*
 * bege.h -- C ABI of the B200-native hot path of arXiv:1708.01609 (van Putten,
 * "Deep searches for broadband extended gravitational-wave emission bursts by
 * heterogeneous computing"): FFT matched filtering of 16 s strain segments against
 * a bank of one-second chirp templates, Parseval sigma, k-sigma tails.
 *
 * Citations are PAPER.md:<line> plus the section / equation they fall in.
 *
 * Conventions (all entry points)
 *   - plain C, no C++/torch types; every call returns a bege_status and never
 *     throws; on error the outputs are left untouched and bege_last_error(plan)
 *     describes the failure.
 *   - "host" / "device" says where a pointer must live; where either is accepted
 *     the library detects it (cudaPointerGetAttributes).
 *   - the caller keeps ownership of every array it passes in; the plan owns its
 *     device state (or borrows the workspace given to bege_plan_set_workspace).
 *   - one plan = one CUDA device and one stream; a plan is not thread safe.
 *   - every step of the path runs in the library's own sm_100a kernels; there is
 *     no CPU fallback.  Without a CUDA device bege_plan_create returns BEGE_ECUDA.
 */
#ifndef BEGE_H
#define BEGE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct bege_plan bege_plan;   /* opaque */

/* One tail sample, PAPER.md:221 (Table 3: sample offset, rho, template identity). 12 bytes. */
typedef struct {
    uint32_t template_id;   /* index into the arrays given to bege_bank_generate          */
    uint32_t lag;           /* m*N + n: segment m, sample offset n, eq.(13)   */
    float    snr;           /* |z[n]| / sigma_jm                                          */
} bege_tail;

typedef enum {
    BEGE_OK        = 0,
    BEGE_EINVAL    = 1,   /* bad argument (N not 2^16, band outside (0, fs/2), NULL pointer ...) */
    BEGE_ESTATE    = 2,   /* call out of order (search before bank / segments are loaded ...)    */
    BEGE_ENOMEM    = 3,   /* workspace too small / device allocation failed                      */
    BEGE_ECUDA     = 4,   /* CUDA runtime error; text in bege_last_error                         */
    BEGE_EOVERFLOW = 5    /* more tails than `cap`; *n_tails is still the true count             */
} bege_status;

/* Counters for benches (bege_plan_get_stats). */
typedef struct {
    uint64_t kernel_launches;      /* kernels of this library launched since plan creation / last reset   */
    uint64_t correlations;         /* (template, segment) pairs searched since last reset                 */
    double   fused_kernel_ms;      /* CUDA-event time spent in the dominant search kernel(s), accumulated
                                      only while profiling is on (bege_plan_set_profiling)               */
    uint64_t fused_kernel_launches;/* launches that fused_kernel_ms covers                                */
    uint64_t hbm_bytes_per_template; /* bytes of one stored template spectrum (the algorithmic HBM read)  */
} bege_stats;

/*
 * Create a plan for transforms of length N (must be 65536 = 2^16: "FFT_{N,M} of
 * length N = 2^16") at sampling rate fs [Hz] with the analysis band band_lo_hz <= |f| <= band_hi_hz
 * (inclusive edges; 350-2000 Hz).  0 < band_lo < band_hi < fs/2.
 * device: CUDA device ordinal.  cuda_stream: a cudaStream_t (e.g. torch's current stream handle; pass
 * cudaStreamLegacy, not 0, for the legacy default stream) or NULL for a non-blocking stream the plan creates.
 * All work of the plan is ordered on that stream: device inputs (bege_segment_load) must have been produced on
 * it or be complete before the call.  A second, internal stream carries the device->host copy of the tails
 * while the search goes on.
 */
int bege_plan_create(bege_plan** out, uint32_t N, double fs, double band_lo_hz, double band_hi_hz,
                     int device, void* cuda_stream);

/*
 * Device bytes the plan needs for a bank of n_templates, n_segments segments and room for `cap`
 * tail records (bank spectra + segment spectra + FFT staging + sigma + records).
 */
int bege_plan_workspace_bytes(const bege_plan*, uint64_t n_templates, uint32_t n_segments,
                              uint64_t cap, uint64_t* bytes);

/*
 * Lend the plan a device buffer (e.g. a torch tensor's storage, 256-byte aligned) of `bytes` bytes; it
 * must outlive the plan or the next call of this function.  Loaded banks / segments are forgotten.
 * dev_ptr == NULL: the plan allocates (cudaMalloc) what it needs on demand and owns it.
 */
int bege_plan_set_workspace(bege_plan*, void* dev_ptr, uint64_t bytes);

/*
 * a1 -- template spectra (PAPER.md:156 step ii: "a chirp template w of duration tau = 1 s is extended by
 * zeros to length N and its transform w~ is loaded into Global Memory").  For j < n_templates:
 *   L = round(tau_s*fs); t_n = n/fs; h_j[n] = hann_L[n] * exp(i 2 pi (f0_j t_n + fdot_j t_n^2 / 2)), n < L,
 *   unit L2 norm, zero padded to N; H_j = DFT_N(h_j).  Phases and the whole transform run in fp64; each stored
 *   bin is rounded to fp32 once.  The in-band rows of H_j are stored in HBM in the tiled layout the search
 *   kernel streams.
 * f0_hz, fdot_hz_s: host arrays of n_templates doubles.  Replaces any previous bank.  1 <= L <= N/16.
 */
int bege_bank_generate(bege_plan*, const double* f0_hz, const double* fdot_hz_s,
                       uint64_t n_templates, double tau_s);

/*
 * a2 -- segment spectra (PAPER.md:155 step i).  x: n_segments*N complex samples, interleaved
 * (re, im) fp32, host or device.  X_m = DFT_N(x_m), bins outside the band set to zero.
 * Replaces previously loaded segments.  n_segments*N must fit 32 bits (lag = m*N + n).
 */
int bege_segment_load(bege_plan*, const float* x_interleaved_c64, uint32_t n_segments);

/*
 * a3-a7 -- the search (PAPER.md:89-100 eq.5-7, :116-120 eq.9, :156-160 steps ii-iv, :162).  For every
 * template j of the bank and loaded segment m:  R = conj(H_j) X_m;  sigma_jm^2 = N^-2 sum_k |R[k]|^2;
 * z = IDFT_N(R) (four-step 256x256, never written to HBM);  every n with |z[n]| > k_sigma*sigma_jm is
 * appended as {j, m*N+n, |z[n]|/sigma_jm}.  Only these records cross PCIe (side stream; for large searches the
 * bank is searched in up to 8 slices and the records of slice i are copied while slice i+1 is searched).
 * tails_out: host array of `cap` records (pinned memory is copied into directly), may be NULL if cap = 0.
 * *n_tails: the TRUE number of tails.  If it exceeds cap, exactly cap records are written (which ones
 * is unspecified) and BEGE_EOVERFLOW is returned.  Record order is unspecified.  Synchronous at return.
 */
int bege_search(bege_plan*, float k_sigma, bege_tail* tails_out, uint64_t cap, uint64_t* n_tails);

/*
 * NEXT row of the scope table -- band threshold ("generalising (9) to a finite band, kappa_1 sigma >
 * rho(t_n) > kappa_2 sigma", to curtail the tails of very deep searches): as bege_search, but a lag n is kept only if
 * k_lo*sigma_jm < |z[n]| < k_hi*sigma_jm (both strict).  k_hi >= k_lo; k_hi = INFINITY is bege_search.
 */
int bege_search_band(bege_plan*, float k_lo, float k_hi, bege_tail* tails_out, uint64_t cap, uint64_t* n_tails);

/*
 * NEXT row of the scope table -- the paper's default output mode (eq.13-17, Fig.4): the tails of
 * the whole bank projected onto the sample offsets.  For every offset i = m*N + n of the loaded segments:
 * snr_out[i] = max over the templates j with |z_jm[n]| > k_sigma*sigma_jm of |z_jm[n]|/sigma_jm (0 if none) and
 * id_out[i] = the template that attains it (UINT32_MAX if none); equal values go to the smaller template id, so the
 * result is unique (the paper accepts a data race here; this implementation has none: one 64-bit
 * atomicMax per tail).  A fixed n_segments*N*8 bytes cross PCIe instead of a variable record list.
 * snr_out, id_out: host arrays of n_segments*N entries.  *n_hits (may be NULL): offsets that hold a tail.
 * Same kernels, sigma and threshold as bege_search; bege_get_sigma is valid afterwards.  Synchronous at return.
 */
int bege_search_maxproj(bege_plan*, float k_sigma, float* snr_out, uint32_t* id_out, uint64_t* n_hits);

/*
 * NEXT row of the scope table -- the paper's own input and output form (PAPER.md:155 step i: "FFT is applied to arrays
 * of complex numbers, merging pairs of real H1 and L1 data"; real chirp templates; Table 3).
 * bege_bank_generate_real: as bege_bank_generate with the REAL template w_n = hann_L[n] cos(2 pi (f0 t_n + fdot t_n^2/2)),
 *   unit L2 norm.  bege_search works on such a bank too; bege_search_dual requires it.
 * bege_search_dual: the loaded segments are read as x = H1 + i L1, so Re z and Im z of the one complex correlation are the
 *   two detectors' filter outputs.  Per stream d, sigma_d = rms of its real output, predicted from the product spectrum
 *   by Parseval's theorem for a real series (eq.7, Hermitian split of R); a hit is |rho_d[n]| > k_sigma
 *   sigma_d (eq.9, two-sided).  For every offset i = m*N + n: snrD_out[i] = the largest |rho_d|/sigma_d over
 *   the bank among the hits (0 if none), idD_out[i] = its template (UINT32_MAX if none; equal values go to the smaller
 *   id).  *n_simultaneous (may be NULL): offsets with a hit in both streams; *n_coincident (may be NULL): those whose two
 *   templates' start frequencies differ by less than delta_hz (|f_1 - f_2| < Delta).
 *   Host arrays of n_segments*N entries each.  The band must lie inside bins [4096, 61440) (BEGE_EINVAL otherwise).
 * bege_get_sigma_dual: sigma_1, sigma_2 of the last bege_search_dual, n_templates*n_segments floats each, template-major.
 */
int bege_bank_generate_real(bege_plan*, const double* f0_hz, const double* fdot_hz_s, uint64_t n_templates, double tau_s);
/*
 * The paper's own template form (Fig.2 caption: "The chirps used in butterfly filtering are symmetric in time,
 * obtained by superposition of chirp forward and backward in time, suitable in searches for both ascending and descending
 * chirps"): as bege_bank_generate_real with w_n = u_n + u_(L-1-n), u_n = hann_L[n] cos(2 pi (f0 t_n + fdot t_n^2/2)) the one-way
 * template, L = round(tau_s fs), unit L2 norm -- the ascending chirp (f0, fdot) plus the descending chirp that starts where it
 * ends.  One such template answers to both; each at about 1/sqrt 2 of the one-way template's output.  A bank made here counts
 * as a real bank for bege_search_dual.
 */
int bege_bank_generate_real_symmetric(bege_plan*, const double* f0_hz, const double* fdot_hz_s, uint64_t n_templates, double tau_s);
int bege_search_dual(bege_plan*, float k_sigma, float* snr1_out, uint32_t* id1_out, float* snr2_out, uint32_t* id2_out,
                     double delta_hz, uint64_t* n_simultaneous, uint64_t* n_coincident);
int bege_get_sigma_dual(bege_plan*, float* sigma1_out, float* sigma2_out);

/* sigma_jm of the last bege_search, host array of n_templates*n_segments floats, template-major. */
int bege_get_sigma(bege_plan*, float* sigma_out);

/*
 * Off the timed path, for parity tests: the full correlation z_jm (host, N complex fp32 interleaved)
 * and its sigma for one (template, segment) pair, computed by the same kernels as bege_search.
 */
int bege_debug_correlate(bege_plan*, uint64_t template_id, uint32_t segment, float* z_out_c64,
                         float* sigma_out);

/* Off the timed path: stored spectrum of one template / one segment, natural order, N complex fp32 (host). */
int bege_debug_template_spectrum(bege_plan*, uint64_t template_id, float* H_out_c64);
int bege_debug_segment_spectrum(bege_plan*, uint32_t segment, float* X_out_c64);

/*
 * Off the timed path, for tests: the search kernel counts the (template, segment) items of a CTA group in 32 bits, so
 * bege_search splits a search of more than 2^30 items per group into several launches.  This lowers that limit
 * (1 <= max_items < 2^30; default 2^30 - 1) so that a test can reach the split with a small bank.  Results do not
 * depend on it.
 */
int bege_debug_set_max_items(bege_plan*, uint64_t max_items);

/*
 * Segment spectra WITHOUT any device allocation (a2, PAPER.md:155 step i; four-step transform as PAPER.md:201-203
 * describes for lengths beyond one work-group's local memory).
 *
 * Who needs this: every other call of this library obtains device memory, either by cudaMalloc or from a workspace the
 * caller had to allocate first.  Some callers cannot do either at the moment they need a spectrum:
 *   - a data-acquisition or low-latency loop, where cudaMalloc / cudaFree are off limits because they synchronise the
 *     whole device and take a driver lock of unbounded duration while other streams are feeding the GPU;
 *   - a process in which another component has already claimed (nearly) all of HBM -- e.g. a framework's caching pool, or
 *     this library's own bank chunk sized to fill the card -- so that a fresh allocation may simply fail;
 *   - code running under a "no allocation after start-up" rule (fixed memory budgets of a production pipeline).
 * For them this ONE entry point keeps what it needs inside the library image itself: the staging area between the two
 * kernels of the transform and its twiddle tables are file-scope __device__ arrays, 2.5 MiB in total, resident on every GPU
 * that loads the library until the process exits.  The call creates no plan, takes no workspace and calls no cudaMalloc,
 * cudaFree or any other allocating routine.
 *
 * Computes, for m < n_segments:  X_m = DFT_N(x_m), N = 65536, bins outside band_lo_hz <= |f| <= band_hi_hz set to zero
 * (same band rule, same kernels for the row pass and the same arithmetic as bege_segment_load), and writes them in NATURAL
 * bin order: X_out[(m*N + k)*2 + {0,1}] = Re, Im of X_m[k].
 *   device        CUDA ordinal (made current on the calling thread, as in every other call).
 *   cuda_stream   a cudaStream_t on that device; NULL = the legacy default stream.  The work is ENQUEUED on it and the
 *                 call returns without waiting: X_out is complete when the stream has reached that point.
 *   x_dev_c64     DEVICE memory, n_segments*N complex fp32 interleaved; produced on cuda_stream or already complete.
 *   X_out_dev_c64 DEVICE memory, same size, caller-owned, must not overlap x_dev_c64.
 *   n_segments    1 .. BEGE_STATIC_MAX_SEGMENTS.  More is refused with BEGE_EINVAL (the staging array has a fixed size);
 *                 split the batch or use a plan.
 *   errbuf        optional (may be NULL): receives a NUL-terminated description of any failure, at most errbuf_len bytes.
 * Returns BEGE_OK, BEGE_EINVAL (arguments, host pointers, size limit) or BEGE_ECUDA (no sm_100 device, runtime error).
 *
 * First call on a device: it looks up the device addresses of the built-in arrays, fills the twiddle tables with a small
 * kernel and WAITS for cuda_stream once (later calls do not wait).  Make that first call during start-up, before the
 * stream is put into capture mode and before timing anything.
 * Sharing: all calls on a device use the same staging array, from any thread and any stream, and nothing locks it on the
 * GPU.  Two calls whose kernels can run at the same time (different streams with no ordering between them) overwrite each
 * other's staging data and return garbage; calls on one stream, or ordered by events, are safe.  The array keeps whatever the
 * last call left there; no part of it needs clearing, because every call rewrites all the words it later reads.
 */
#define BEGE_STATIC_MAX_SEGMENTS 4
int bege_segment_spectrum_static(int device, void* cuda_stream, double fs, double band_lo_hz, double band_hi_hz,
                                 const float* x_dev_c64, uint32_t n_segments, float* X_out_dev_c64,
                                 char* errbuf, uint64_t errbuf_len);

int  bege_plan_set_profiling(bege_plan*, int on);    /* CUDA events around the dominant kernel (adds syncs) */
int  bege_plan_get_stats(const bege_plan*, bege_stats* out);
int  bege_plan_reset_stats(bege_plan*);

const char* bege_last_error(const bege_plan*);       /* never NULL; valid until the next call on the plan */
void bege_plan_destroy(bege_plan*);
const char* bege_version(void);

#ifdef __cplusplus
}
#endif
#endif /* BEGE_H */
