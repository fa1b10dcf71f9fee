/*
 * bege_probe.h -- C ABI of libbege_probe.so: measurement probes kept OUT of the product library (libbege.so, bege.h).
 * Status codes are bege.h's.
 */
#ifndef BEGE_PROBE_H
#define BEGE_PROBE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/*
 * SURVEY.md section 8(f) NEXT #4, bake-off probe of the OVERLAP-SAVE variant -- a measurement aid, not part of the search
 * path.  Templates are tau*fs = 4096 samples long, so the circular correlation of PAPER.md:74 eq.(3) over N = 65536 lags
 * can be assembled from n_blocks = 6 correlations of P = 16384 points over blocks of the band-limited segment that
 * overlap by 4096 samples (block i: samples 12288 i .. 12288 i + 16383 mod N, valid lags 12288 i .. 12288 i + 12287);
 * a P-point transform fits one SM (PAPER.md:201-203 on transforms beyond local memory).  The probe runs, per (template,
 * block): conj(H16) X16 -> inverse P-point transform in shared memory -> |z|^2 > thr2 on the valid lags, hits counted.
 * It owns its device memory and stream.  h16 (host, T x 16384 complex fp32: H16[k] = H[4 k]) and x16 (host, n_blocks x
 * 16384 complex fp32: transforms of the blocks) may each be NULL: the device buffers are then filled with finite
 * numbers (timing only).  z_dbg (host, n_blocks x 16384 complex fp32, may be NULL): the blocks' correlations for
 * template dbg_j, lag n of block i at [i*16384 + n], normalised by 1/P.  *ms_out: mean device time of one pass over all
 * T x n_blocks items (`reps` passes after one warm-up pass); *hits_out (may be NULL): hits of one pass.
 */
int bege_ovs_probe(int device, uint64_t n_templates, uint32_t n_blocks, uint32_t reps, float thr2, const float* h16,
                   const float* x16, float* z_dbg, uint64_t dbg_j, double* ms_out, uint64_t* hits_out);

#ifdef __cplusplus
}
#endif
#endif /* BEGE_PROBE_H */
