"""Pins of the fp64 CPU oracle against things other than itself (CPU only, `-m "not gpu"`).

Each test names the passage of PAPER.md (or the DESIGN.md reading) it fixes and is chosen so
that a plausible mistake in oracle/bege_oracle.c -- a dropped term, a wrong sign or index, a
transposed operand, a missing conjugate or normalisation -- fails at least one of them.
"""
import math
import os

import numpy as np
import pytest

from oracle import bege_oracle as bo
import bege_synth as synth

FS, N, BAND, TAU = synth.FS, synth.N_SEG, synth.BAND, synth.TAU
GOLD = os.path.join(os.path.dirname(__file__), "golden", "paper_numbers.txt")


def _gold():
    out = {}
    with open(GOLD) as fh:
        for line in fh:
            if line.startswith("#") or not line.strip():
                continue
            name, val, tol, _cite = [p.strip() for p in line.split("|", 3)]
            out[name] = (float(val), float(tol))
    return out


# ------------------------------------------------------------------ FFT (eq.8)
@pytest.mark.parametrize("n", [1, 2, 4, 8, 64, 256, 1024])
@pytest.mark.parametrize("sign", [-1, 1])
def test_fft_equals_textbook_dft_matrix(n, sign):
    rng = np.random.default_rng(n + 7)
    a = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    k = np.arange(n)
    F = np.exp(sign * 2j * np.pi * np.outer(k, k) / n)      # the O(N^2) definition
    ref = F @ a
    got = bo.fft(a, sign)
    assert np.max(np.abs(got - ref)) <= 1e-11 * max(1.0, np.linalg.norm(a))


def test_fft_matches_library_routine_at_full_size():
    rng = np.random.default_rng(11)
    a = rng.standard_normal(N) + 1j * rng.standard_normal(N)
    assert np.linalg.norm(bo.fft(a, -1) - np.fft.fft(a)) <= 1e-13 * np.linalg.norm(a) * math.sqrt(N)
    assert np.linalg.norm(bo.fft(a, +1) - np.fft.ifft(a) * N) <= 1e-13 * np.linalg.norm(a) * math.sqrt(N)


def test_fft_roundtrip_and_parseval():
    rng = np.random.default_rng(12)
    a = rng.standard_normal(N) + 1j * rng.standard_normal(N)
    A = bo.fft(a, -1)
    back = bo.fft(A, +1) / N
    assert np.max(np.abs(back - a)) < 1e-12
    # PAPER.md:98 Parseval: sum |x|^2 = N^-1 sum |X|^2
    assert abs(np.sum(np.abs(a) ** 2) - np.sum(np.abs(A) ** 2) / N) < 1e-12 * N


def test_fft_rejects_non_power_of_two():
    with pytest.raises(ValueError):
        bo.fft(np.zeros(12, dtype=complex), -1)


def test_fft_delta_and_tone():
    # a unit impulse at n0 transforms to exp(-2 pi i k n0/N): fixes the sign of the exponent
    n, n0 = 256, 3
    a = np.zeros(n, dtype=complex)
    a[n0] = 1.0
    assert np.allclose(bo.fft(a, -1), np.exp(-2j * np.pi * np.arange(n) * n0 / n), atol=1e-13)
    # a tone exp(+2 pi i k0 n/N) has its forward transform at bin +k0
    k0 = 5
    A = bo.fft(np.exp(2j * np.pi * k0 * np.arange(n) / n), -1)
    assert abs(A[k0] - n) < 1e-10 and np.sum(np.abs(A)) - abs(A[k0]) < 1e-9


# ------------------------------------------------------- band mask
def test_band_mask_bins():
    X = bo.band_mask(np.ones(N, dtype=complex), FS, *BAND)
    keep = np.flatnonzero(X.real)
    # 350 Hz = bin 5600, 2000 Hz = bin 32000 at df = 1/16 Hz, inclusive; mirrored at N-k
    expect = np.concatenate([np.arange(5600, 32001), np.arange(N - 32000, N - 5600 + 1)])
    assert np.array_equal(keep, expect)
    assert keep.size == 52802 and X[0] == 0 and X[N // 2] == 0


def test_segment_spectrum_is_fft_then_mask():
    x = synth.white_noise(5, 4096)
    X = bo.segment_spectrum(x, FS, *BAND)
    f = np.abs(np.fft.fftfreq(4096, 1 / FS))
    ref = np.fft.fft(x) * ((f >= BAND[0]) & (f <= BAND[1]))
    assert np.linalg.norm(X - ref) < 1e-10 * np.linalg.norm(ref)


# ---------------------------------------------------- template (BASELINE cfg0)
def test_template_norm_window_padding():
    h = bo.template(1000.0, 50.0, TAU, FS, N)
    L = 4096
    assert abs(np.linalg.norm(h) - 1.0) < 1e-14
    assert np.all(h[L:] == 0) and h[0] == 0 and abs(h[L - 1]) < 1e-15   # symmetric Hann: zero at both ends
    # closed form: sum_n hann^2 = 3 (L-1)/8  =>  envelope = hann/sqrt(3 (L-1)/8); L even, so the largest
    # sample sits half a step off the window centre: hann(2047) = 1/2 - 1/2 cos(2 pi 2047/4095)
    env = np.abs(h[:L])
    w_max = 0.5 - 0.5 * math.cos(2 * math.pi * 2047 / 4095)
    assert abs(env.max() - w_max / math.sqrt(3 * (L - 1) / 8)) < 1e-15
    assert np.allclose(env, env[::-1], atol=1e-15)                      # symmetric window


def test_template_instantaneous_frequency():
    # d(phase)/dt / 2 pi = f0 + fdot t: fixes the 1/2 in front of fdot and the sign of i
    f0, fd = 700.0, -120.0
    h = bo.template(f0, fd, TAU, FS, N)[1:4095]
    dphi = np.angle(h[1:] * np.conj(h[:-1]))
    t_mid = (np.arange(1, 4094) + 0.5) / FS
    finst = dphi * FS / (2 * np.pi)
    assert np.max(np.abs(finst - (f0 + fd * t_mid))) < 1e-6


def test_template_spectrum_of_pure_tone():
    # fdot = 0, bin-centred f0: the spectrum is the Hann kernel centred on bin f0*N/fs, positive frequency
    f0 = 1000.0
    H = bo.fft(bo.template(f0, 0.0, TAU, FS, N), -1)
    assert int(np.argmax(np.abs(H))) == int(f0 * N / FS)
    # Hann main lobe is +-2 Hz for a 1 s window, side lobes fall at 18 dB/octave: all but <1e-6 of
    # the energy lies within +-8 Hz of f0, and none of it at negative frequencies
    k0, w = int(f0 * N / FS), 128
    tot = np.sum(np.abs(H) ** 2)
    assert abs(tot - N) < 1e-8 * N                        # unit-norm h, unnormalised DFT (Parseval)
    assert np.sum(np.abs(H[k0 - w:k0 + w + 1]) ** 2) / tot > 1 - 1e-6
    assert np.sum(np.abs(H[N // 2:]) ** 2) / tot < 1e-9


def test_template_matches_library_expression():
    f0, fd = 1234.5, 333.0
    t = np.arange(4096) / FS
    ref = np.hanning(4096) * np.exp(2j * np.pi * (f0 * t + 0.5 * fd * t * t))
    ref /= np.linalg.norm(ref)
    assert np.max(np.abs(bo.template(f0, fd, TAU, FS, N)[:4096] - ref)) < 1e-12


def test_template_rejects_bad_length():
    with pytest.raises(ValueError):
        bo.template(100.0, 0.0, 20.0, FS, N)       # tau*fs > N


# -------------------------------------- correlation = definition (PAPER.md:74 eq.3, :81, :89-92 eq.5)
def _brute_corr(xhat, h, L):
    """eq.(3) with circular indexing, written with python loops (tiny sizes only)."""
    n = xhat.size
    z = np.zeros(n, dtype=complex)
    for lag in range(n):
        acc = 0j
        for s in range(L):
            acc += np.conj(h[s]) * xhat[(lag + s) % n]
        z[lag] = acc
    return z


@pytest.mark.parametrize("n", [64, 256, 1024])
def test_fft_correlation_equals_direct_sum(n):
    fs, band, L = 256.0, (20.0, 100.0), n // 16
    rng = np.random.default_rng(n)
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)      # general complex x
    h = bo.template(40.0, 30.0, L / fs, fs, n)
    X = bo.segment_spectrum(x, fs, *band)
    z, sigma = bo.correlate(X, h)
    xhat = bo.fft(X, +1) / n
    # oracle's direct routine vs python loops, then FFT route vs direct: two independent restatements
    zd = bo.correlate_direct(xhat, h, L)
    if n <= 256:
        assert np.max(np.abs(zd - _brute_corr(xhat, h, L))) < 1e-12
    assert np.max(np.abs(z - zd)) < 1e-12
    # PAPER.md:94-100 eq.(6)=(7): Parseval sigma is the rms of the output, identically
    assert abs(sigma - math.sqrt(np.mean(np.abs(z) ** 2))) < 1e-13


def test_correlation_sampled_lags_full_size():
    x = synth.noise_segment(21).astype(np.complex128)
    X = bo.segment_spectrum(x, FS, *BAND)
    h = bo.template(900.0, 150.0, TAU, FS, N)
    z, sigma = bo.correlate(X, h)
    lags = np.array([0, 1, 4095, 4096, 29901, N - 4096, N - 1], dtype=np.uint32)   # incl. wrap-around lags
    zd = bo.correlate_direct(bo.fft(X, +1) / N, h, 4096, lags)
    assert np.max(np.abs(z[lags] - zd)) < 1e-12
    assert abs(sigma - math.sqrt(np.mean(np.abs(z) ** 2))) < 1e-13


def test_shifted_template_gives_autocorrelation_peak():
    # x = A * template shifted to n0 (band = everything but DC/Nyquist) => z peaks at n0 with value A
    n, fs, L, n0, A = 1024, 1024.0, 128, 300, 3.5
    h = bo.template(200.0, 100.0, L / fs, fs, n)
    x = A * np.roll(h, n0)
    X = bo.segment_spectrum(x, fs, 0.5, 511.5)
    z, _ = bo.correlate(X, h)
    assert int(np.argmax(np.abs(z))) == n0
    assert abs(z[n0] - A) < 1e-3          # removed DC/Nyquist bins carry ~nothing
    assert abs(z[n0].imag) < 1e-6         # conj on the template, not on the data


def test_bin_centred_tone_gives_constant_modulus():
    # fdot = 0 template on a tone at the same bin-centred frequency: |z| independent of lag
    n, fs, L = 1024, 1024.0, 64
    x = np.exp(2j * np.pi * 128.0 * np.arange(n) / fs)
    X = bo.segment_spectrum(x, fs, 10.0, 500.0)
    z, sigma = bo.correlate(X, bo.template(128.0, 0.0, L / fs, fs, n))
    assert np.ptp(np.abs(z)) < 1e-12 and abs(sigma - np.abs(z[0])) < 1e-12
    # and the phase advances with the lag like the tone itself (z[n] ~ x[n]): fixes y(t+s), not y(t-s)
    assert abs(np.angle(z[1] / z[0]) - 2 * np.pi * 128.0 / fs) < 1e-9


# ----------------------------------------- sigma / Gaussian tails (reading 4)
@pytest.fixture(scope="module")
def cfg0_interior():
    """z/sigma of cfg0's 14x14 interior templates (edge templates lose energy out of band)."""
    w = synth.config0()
    X = bo.segment_spectrum(w.x[0], FS, *BAND)
    ids = [i * 16 + j for i in range(1, 15) for j in range(1, 15)]
    zs, sig = [], []
    for t in ids:
        z, s = bo.correlate(X, bo.template(w.f0[t], w.fdot[t], TAU, FS, N))
        zs.append(z / s)
        sig.append(s)
    return np.array(zs), np.array(sig)


def test_sigma_predicts_empirical_std_on_noise(cfg0_interior):
    zs, sig = cfg0_interior
    L = 4096
    # rms over the VALID (non wrap-around) lags only: non-trivial version of the "within 1 %" pin
    rms_valid = np.sqrt(np.mean(np.abs(zs[:, : N - L]) ** 2, axis=1))
    # pooled over templates within 1 %; a single narrow-band template (small |fdot|: output correlated
    # over ~1e3 lags, so only ~60 independent samples) scatters by a few % when 1/16 of the lags is dropped
    assert abs(np.sqrt(np.mean(rms_valid ** 2)) - 1.0) < 0.01
    assert np.max(np.abs(rms_valid - 1.0)) < 0.05
    # over ALL lags (circular output) it is an identity, eq.(6)=(7)
    assert np.max(np.abs(np.sqrt(np.mean(np.abs(zs) ** 2, axis=1)) - 1.0)) < 1e-12
    # closed form: E[sigma^2] = in-band energy fraction of the unit-norm template on unit white noise
    assert 0.9 < np.mean(sig ** 2) < 1.1


def test_tail_counts_follow_gaussian_laws(cfg0_interior):
    zs, _ = cfg0_interior
    n_out = zs.size
    # circular complex Gaussian: P(|z| > k sigma) = exp(-k^2); each quadrature at sigma/sqrt2 is erfc(k/sqrt2)
    for k in (2.0, 2.5, 3.0):
        got = np.count_nonzero(np.abs(zs) > k)
        exp = n_out * math.exp(-k * k)
        # outputs are correlated over ~13 lags (band-limited): allow 6 x Poisson on clustered counts
        assert abs(got - exp) < 6 * math.sqrt(13 * exp) + 0.03 * exp, (k, got, exp)
        for q in (zs.real, zs.imag):
            gq = np.count_nonzero(np.abs(q) > k / math.sqrt(2))
            eq = n_out * math.erfc(k / math.sqrt(2))
            assert abs(gq - eq) < 6 * math.sqrt(13 * eq) + 0.03 * eq, (k, gq, eq)
    # circularity: equal variance in both quadratures, no correlation between them
    assert abs(np.var(zs.real) / np.var(zs.imag) - 1) < 0.01
    assert abs(np.mean(zs.real * zs.imag)) < 0.005


# ------------------------------------------------- injection recovery (BASELINE cfg1; readings 14, 18)
def test_injected_chirp_recovered_at_true_template_and_lag():
    w = synth.config1()
    X = bo.segment_spectrum(w.x[0], FS, *BAND)
    rows, cols = range(112, 121), range(96, 109)
    ids = np.array([i * 256 + j for i in rows for j in cols])
    f0 = np.append(w.f0[ids], 1100.0)            # exact template appended last
    fd = np.append(w.fdot[ids], -80.0)
    tails, n_true, sigma, _ = bo.search(X[None, :], f0, fd, TAU, FS, 5.0)
    assert n_true == tails.size > 0
    grid = tails[tails["template_id"] < ids.size]
    best = grid[np.argmax(grid["snr"])]
    assert ids[best["template_id"]] == w.meta["true_id"] == 29798
    assert abs(int(best["lag"]) - 29870) <= 2          # chirp degeneracy: n0 + df0*fs/fdot = 29901 - 31
    assert 9.0 < best["snr"] < 12.5
    exact = tails[tails["template_id"] == ids.size]
    assert int(exact[np.argmax(exact["snr"])]["lag"]) == w.meta["n0"] == 29901
    assert 9.5 < exact["snr"].max() < 12.5             # sigma includes the signal (reading 13)
    # sigma of the matching template is raised by the injection, a far template stays ~1
    assert sigma[-1, 0] > 1.05 and 0.9 < sigma[0, 0] < 1.1


# ------------------------------------------------------------- search bookkeeping (eq.13)
def test_search_records_ids_lags_sigma_layout():
    n, fs, band, tau = 1024, 1024.0, (50.0, 450.0), 0.125
    xs = np.stack([synth.band_limit(synth.white_noise(s, n), fs, *band) for s in (1, 2, 3)])
    Xs = np.stack([bo.segment_spectrum(x, fs, *band) for x in xs])
    f0, fd = synth.bank_grid(3, 2, 100.0, 300.0, -80.0, 80.0)
    k = 1.7
    tails, n_true, sigma, used = bo.search(Xs, f0, fd, tau, fs, k)
    assert used >= 1 and n_true == tails.size and sigma.shape == (6, 3)
    exp = []
    for j in range(6):
        h = bo.template(f0[j], fd[j], tau, fs, n)
        for m in range(3):
            z, s = bo.correlate(Xs[m], h)
            assert abs(s - sigma[j, m]) < 1e-15
            for lag in np.flatnonzero(np.abs(z) > k * s):
                exp.append((j, m * n + lag, abs(z[lag]) / s))
    assert tails.size == len(exp)
    assert np.array_equal(tails["template_id"], [e[0] for e in exp])
    assert np.array_equal(tails["lag"], [e[1] for e in exp])
    assert np.allclose(tails["snr"], [e[2] for e in exp], rtol=1e-13)
    # cap smaller than the count: true count still returned
    t2, n2, _, _ = bo.search(Xs, f0, fd, tau, fs, k, cap=5)
    assert n2 == n_true and t2.size == 5


def test_zero_data_gives_no_tails():
    f0, fd = synth.bank_grid(2, 2, 400.0, 500.0, -10.0, 10.0)
    tails, n_true, sigma, _ = bo.search(np.zeros((1, 4096), dtype=complex), f0, fd, 0.25, FS, 3.0)
    assert n_true == 0 and np.all(sigma == 0)


def test_search_thread_count_does_not_change_results():
    n, fs, band = 2048, 1024.0, (50.0, 450.0)
    X = bo.segment_spectrum(synth.white_noise(9, n), fs, *band)[None, :]
    f0, fd = synth.bank_grid(4, 4, 100.0, 300.0, -80.0, 80.0)
    a = bo.search(X, f0, fd, 0.25, fs, 2.0, n_threads=1)
    b = bo.search(X, f0, fd, 0.25, fs, 2.0, n_threads=4)
    assert a[1] == b[1] and np.array_equal(a[0], b[0]) and np.array_equal(a[2], b[2])


# ------------------------------------------------------------------ the paper's printed arithmetic
def test_paper_printed_numbers():
    g = _gold()

    def close(name, val):
        ref, tol = g[name]
        assert abs(val - ref) <= tol * ref, (name, val, ref)

    fl = bo.fft_flops(N)
    close("flops_per_fft_N65536", fl)
    close("realtime_tflops", fl * 2 ** 23 / 16.0)
    corr = 2 ** 23 * 288 * 2048
    close("s6_total_correlations", corr)
    close("s6_total_flop", corr * fl)
    close("block_flop_M2", 2048 ** 2 * fl)
    close("block_output_bytes", 2048 ** 2 * N * 8)
    close("block_bytes", 2048 * N * 8)
    close("file_bytes", 8 * 2048 * N * 8)
    close("segment_bytes", N * 8)


# ----------------------------------------------------------------------------- max projection
def test_max_projection_is_the_per_lag_maximum_of_the_extended_output():
    """eq.(15)-(17): B keeps, per sample offset m*N+n, the largest rho over the bank and its template.  Pinned by
    brute force against the (separately pinned) extended output of bo_search on two segments and 40 templates,
    with a planted tie to check that equal values go to the smaller template id."""
    w = synth.config0()
    x2, _ = synth.inject_chirp(synth.band_limit(synth.white_noise(9)), 1000.0, 50.0, 5.0, 9.0)
    xs = np.stack([w.x[0], synth.as_segment(x2)])
    Xs = np.stack([bo.segment_spectrum(x, FS, *BAND) for x in xs])
    f0 = np.concatenate([w.f0[::8], [1000.0, 1000.0], w.f0[3:8]])       # templates 32 and 33 are identical
    fd = np.concatenate([w.fdot[::8], [50.0, 50.0], w.fdot[3:8]])
    k = 2.8
    tails, n, _, _ = bo.search(Xs, f0, fd, TAU, FS, k)
    snr, ids = bo.search_maxproj(Xs, f0, fd, TAU, FS, k)
    assert snr.shape == (2, N) and ids.shape == (2, N)
    want_snr = np.zeros(2 * N)
    want_id = np.full(2 * N, np.iinfo(np.uint32).max, dtype=np.uint32)
    for rec in tails:                                                   # tails are sorted by (template_id, lag)
        if rec["snr"] > want_snr[rec["lag"]]:
            want_snr[rec["lag"]] = rec["snr"]
            want_id[rec["lag"]] = rec["template_id"]
    assert np.array_equal(snr.ravel(), want_snr)
    assert np.array_equal(ids.ravel(), want_id)
    assert (snr > 0).sum() < n                                          # several templates share lags
    assert np.all((snr == 0) == (ids == np.iinfo(np.uint32).max))
    # the planted duplicate never wins, the first copy does at the injection
    assert not np.any(ids == 33)
    peak = np.unravel_index(np.argmax(snr), snr.shape)
    assert peak[0] == 1 and ids[peak] == 32


# ----------------------------------------------------------------------------- band threshold
def test_band_threshold_is_the_extended_output_minus_its_top():
    """kappa_1 sigma > rho > kappa_2 sigma: pinned against the (separately pinned) one-sided search -- the band
    result is its tail set with the entries at or above kappa_1 removed; a band up to infinity changes nothing."""
    w = synth.config0()
    X = bo.segment_spectrum(w.x[0], FS, *BAND)
    ids = np.arange(0, 256, 8)
    full, n_full, _, _ = bo.search(X[None, :], w.f0[ids], w.fdot[ids], TAU, FS, 2.5)
    band, n_band = bo.search_band(X[None, :], w.f0[ids], w.fdot[ids], TAU, FS, 2.5, 3.0)
    keep = full[full["snr"] < 3.0]
    assert 0 < n_band == keep.size < n_full
    for f in ("template_id", "lag", "snr"):
        assert np.array_equal(band[f], keep[f])
    same, n_same = bo.search_band(X[None, :], w.f0[ids], w.fdot[ids], TAU, FS, 2.5, np.inf)
    assert n_same == n_full and np.array_equal(same["lag"], full["lag"])
    _, n_none = bo.search_band(X[None, :], w.f0[ids], w.fdot[ids], TAU, FS, 3.0, 3.0)
    assert n_none == 0


# ------------------------------------------------------------------ dual-stream search (PAPER.md:155, :70, :100 eq.7, :221 Table 3)
def _packed_noise(seed_h1, seed_l1):
    """x = H1 + i L1: two independent band-limited Gaussian streams packed into one complex segment."""
    h1 = synth.band_limit(synth.white_noise(seed_h1))
    l1 = synth.band_limit(synth.white_noise(seed_l1))
    return h1, l1, (h1 + 1j * l1)


def test_real_template_is_the_normalised_real_part():
    """bo_template_real: w_n = hann cos(2 pi c_n), unit norm, no imaginary part -- written out here with numpy."""
    f0, fd = 777.0, -123.0
    w = bo.template_real(f0, fd, TAU, FS, N)
    L = int(round(TAU * FS))
    n = np.arange(L)
    ref = np.hanning(L) * np.cos(2 * np.pi * (f0 * n / FS + 0.5 * fd * (n / FS) ** 2))
    ref /= np.linalg.norm(ref)
    assert np.all(w.imag == 0) and np.all(w[L:] == 0)
    assert abs(np.linalg.norm(w) - 1) < 1e-14
    assert np.max(np.abs(w.real[:L] - ref)) < 1e-12
    # and it is proportional to the real part of the complex template of the single-stream search
    h = bo.template(f0, fd, TAU, FS, N)
    c = np.vdot(h.real, w.real) / np.vdot(h.real, h.real)
    assert np.max(np.abs(w.real - c * h.real)) < 1e-12


def test_symmetric_template_is_chirp_plus_time_reverse():
    """bo_template_real_sym (Fig.2 caption: "symmetric in time, obtained by superposition of chirp forward
    and backward in time"): w[n] = w[L-1-n]; equal to the normalised sum of the one-way template (pinned above)
    and its reversal; and equal to the superposition of the ascending chirp (f0, fdot) and the descending chirp that
    starts where it ends, (f0 + fdot T', -fdot) with a phase offset, T' = (L-1)/fs -- written out with numpy."""
    L = int(round(TAU * FS))
    n = np.arange(L)
    for (f0, fd) in ((777.0, -123.0), (400.0, 390.0), (1500.0, 0.0)):
        w = bo.template_real_sym(f0, fd, TAU, FS, N)
        assert np.all(w.imag == 0) and np.all(w[L:] == 0)
        assert abs(np.linalg.norm(w) - 1) < 1e-14
        assert np.max(np.abs(w.real[:L] - w.real[:L][::-1])) < 1e-15       # symmetric in time (to the window's rounding)
        u = bo.template_real(f0, fd, TAU, FS, N).real[:L]                   # one-way template (same norm for both directions)
        ref = u + u[::-1]
        ref /= np.linalg.norm(ref)
        assert np.max(np.abs(w.real[:L] - ref)) < 1e-12
        Tp = (L - 1) / FS
        t = n / FS
        up = np.cos(2 * np.pi * (f0 * t + 0.5 * fd * t ** 2))
        phi0 = f0 * Tp + 0.5 * fd * Tp ** 2
        down = np.cos(2 * np.pi * (phi0 - ((f0 + fd * Tp) * t - 0.5 * fd * t ** 2)))   # starts at f0 + fd T', rate -fd
        ref2 = np.hanning(L) * (up + down)
        ref2 /= np.linalg.norm(ref2)
        assert np.max(np.abs(w.real[:L] - ref2)) < 1e-9


def test_symmetric_template_finds_ascending_and_descending_chirps():
    """One time-symmetric template recovers an injection of the ascending chirp AND one of its descending mirror
    ("suitable in searches for both ascending and descending chirps"), each at the injected offset and
    with about 1/sqrt 2 of the one-way template's output; the one-way template of the ascending chirp sees the
    descending one at noise level."""
    f0, fd = 900.0, 300.0
    L = int(round(TAU * FS))
    Tp = (L - 1) / FS
    w_sym = bo.template_real_sym(f0, fd, TAU, FS, N)
    w_up = bo.template_real(f0, fd, TAU, FS, N)
    noise = synth.band_limit(synth.white_noise(31))
    x_up, n_up = synth.inject_chirp(noise, f0, fd, 4.0, 12.0)
    x_dn, n_dn = synth.inject_chirp(noise, f0 + fd * Tp, -fd, 11.0, 12.0)
    for x, n0, one_way_sees_it in ((x_up, n_up, True), (x_dn, n_dn, False)):
        X = bo.segment_spectrum(x.astype(np.complex128), FS, *BAND)
        z, s1, _ = bo.correlate_dual(X, w_sym)
        rho = np.abs(z.real) / s1
        peak = int(np.argmax(rho))
        assert abs(peak - n0) <= 8 and rho[peak] > 6.5
        z1, t1, _ = bo.correlate_dual(X, w_up)
        rho1 = np.abs(z1.real) / t1
        if one_way_sees_it:
            assert abs(int(np.argmax(rho1)) - n0) <= 8
            assert 0.6 < rho[peak] / rho1.max() < 0.85                      # ~ 1/sqrt 2
        else:
            assert rho1[n0 - 64: n0 + 64].max() < 5.5                       # the one-way template misses the mirror chirp


def test_symmetric_dual_search_is_the_per_template_maximum():
    """bo_search_dual_sym is bo_search_dual with the symmetric template: rebuilt offset by offset from
    bo_correlate_dual on a small bank."""
    h1, l1, x = _packed_noise(25, 26)
    X = bo.segment_spectrum(x, FS, *BAND)
    f0, fd = np.array([500.0, 1200.0, 1700.0]), np.array([150.0, -300.0, 50.0])
    k = 3.0
    o1, i1, o2, i2, sig = bo.search_dual(X[None, :], f0, fd, TAU, FS, k, symmetric=True)
    b1, b2 = np.zeros(N), np.zeros(N)
    j1, j2 = np.full(N, 0xFFFFFFFF, dtype=np.uint32), np.full(N, 0xFFFFFFFF, dtype=np.uint32)
    for j in range(3):
        z, s1, s2 = bo.correlate_dual(X, bo.template_real_sym(f0[j], fd[j], TAU, FS, N))
        assert abs(sig[j, 0, 0] - s1) < 1e-15 and abs(sig[j, 0, 1] - s2) < 1e-15
        for b, jj, a, s in ((b1, j1, np.abs(z.real), s1), (b2, j2, np.abs(z.imag), s2)):
            hit = (a > k * s) & (a / s > b)
            b[hit] = (a / s)[hit]
            jj[hit] = j
    assert np.array_equal(o1[0], b1) and np.array_equal(o2[0], b2)
    assert np.array_equal(i1[0], j1) and np.array_equal(i2[0], j2)
    assert (i1[0] != 0xFFFFFFFF).sum() > 100


def test_dual_sigma_is_eq6_and_eq7():
    """sigma per detector stream: the definition (eq.6, rms of the real output) against an independent numpy
    evaluation, and against Parseval's half-spectrum form for a real series (eq.7), which is the
    form the paper prints (sqrt 2 / N sqrt(sum over half the spectrum))."""
    h1, l1, x = _packed_noise(21, 22)
    X = bo.segment_spectrum(x, FS, *BAND)
    for (f0, fd) in ((500.0, 120.0), (1500.0, -350.0), (1990.0, 400.0)):
        w = bo.template_real(f0, fd, TAU, FS, N)
        z, s1, s2 = bo.correlate_dual(X, w)
        zn = np.fft.ifft(np.conj(np.fft.fft(w)) * X)                    # the library's transform, eq.(5)
        assert np.linalg.norm(z - zn) < 1e-12 * np.linalg.norm(zn)
        assert abs(s1 - np.sqrt(np.mean(zn.real ** 2))) < 1e-13 * s1   # eq.(6) on the H1 output
        assert abs(s2 - np.sqrt(np.mean(zn.imag ** 2))) < 1e-13 * s2   # eq.(6) on the L1 output
        p1, p2 = bo.sigma_dual_parseval(X, w)                           # eq.(7)
        assert abs(p1 - s1) < 1e-12 * s1 and abs(p2 - s2) < 1e-12 * s2


def test_dual_packing_equals_two_separate_real_searches():
    """Packing is exact: Re z of (H1 + i L1) is the correlation of H1 alone, Im z that of L1 alone (linearity of
    eq.3 with a real template) -- checked against the single-stream functions, which are pinned on their own, and
    against the direct time-domain sum of eq.(3) on sampled lags."""
    h1, l1, x = _packed_noise(23, 24)
    X = bo.segment_spectrum(x, FS, *BAND)
    X1 = bo.segment_spectrum(h1.astype(np.complex128), FS, *BAND)
    X2 = bo.segment_spectrum(l1.astype(np.complex128), FS, *BAND)
    w = bo.template_real(900.0, 200.0, TAU, FS, N)
    z, s1, s2 = bo.correlate_dual(X, w)
    z1, _ = bo.correlate(X1, w)
    z2, _ = bo.correlate(X2, w)
    assert np.max(np.abs(z1.imag)) < 1e-12 and np.max(np.abs(z2.imag)) < 1e-12
    assert np.max(np.abs(z.real - z1.real)) < 1e-12 and np.max(np.abs(z.imag - z2.real)) < 1e-12
    assert abs(s1 - np.sqrt(np.mean(z1.real ** 2))) < 1e-13 and abs(s2 - np.sqrt(np.mean(z2.real ** 2))) < 1e-13
    lags = np.array([0, 1, 4095, 30000, N - 4096, N - 1], dtype=np.uint32)
    L = int(round(TAU * FS))
    for stream, part in ((h1, z.real), (l1, z.imag)):
        xhat = bo.fft(bo.band_mask(bo.fft(stream.astype(np.complex128), -1), FS, *BAND), +1) / N
        d = bo.correlate_direct(xhat, w, L, lags)
        assert np.max(np.abs(d.real - part[lags])) < 1e-11


def test_dual_tail_counts_follow_the_real_two_sided_law():
    """Each stream's output is real and near-Gaussian: P(|rho| > k sigma) = erfc(k / sqrt 2)."""
    h1, l1, x = _packed_noise(25, 26)
    X = bo.segment_spectrum(x, FS, *BAND)
    f0, fd = synth.bank_grid(6, 4, 500.0, 1800.0, -150.0, 150.0)
    k = 3.0
    c1 = c2 = 0
    for a, b in zip(f0, fd):
        z, s1, s2 = bo.correlate_dual(X, bo.template_real(a, b, TAU, FS, N))
        c1 += int(np.sum(np.abs(z.real) > k * s1))
        c2 += int(np.sum(np.abs(z.imag) > k * s2))
    expect = f0.size * N * math.erfc(k / math.sqrt(2.0))                # 4247
    for c in (c1, c2):
        assert abs(c - expect) < 0.12 * expect, (c, expect)            # outputs are correlated over ~10 lags: several x Poisson


def test_search_dual_against_brute_force_and_injection_in_one_stream():
    """bo_search_dual (Table 3 form) rebuilt offset by offset from bo_correlate_dual; a chirp injected into H1 only is
    found in stream 1 at its template and lag, and not in stream 2; simultaneous / coincident counts by hand."""
    h1, l1, _ = _packed_noise(27, 28)
    h1, n0 = synth.inject_chirp(h1, 1000.0, 50.0, 5.0, 12.0)
    x = h1 + 1j * l1
    X = bo.segment_spectrum(x, FS, *BAND)
    f0 = np.array([600.0, 1000.0, 1000.0, 1400.0])                        # entries 1 and 2 identical: a planted tie
    fd = np.array([-100.0, 50.0, 50.0, 200.0])
    k = 3.2
    snr1, id1, snr2, id2, sig = bo.search_dual(X[None, :], f0, fd, TAU, FS, k)
    none = np.iinfo(np.uint32).max
    b1, b2 = np.zeros(N), np.zeros(N)
    j1, j2 = np.full(N, none, dtype=np.uint32), np.full(N, none, dtype=np.uint32)
    for j in range(f0.size):
        z, s1, s2 = bo.correlate_dual(X, bo.template_real(f0[j], fd[j], TAU, FS, N))
        assert abs(sig[j, 0, 0] - s1) < 1e-15 and abs(sig[j, 0, 1] - s2) < 1e-15
        r1, r2 = np.abs(z.real) / s1, np.abs(z.imag) / s2
        u1, u2 = (r1 > k) & (r1 > b1), (r2 > k) & (r2 > b2)
        b1[u1], j1[u1] = r1[u1], j
        b2[u2], j2[u2] = r2[u2], j
    assert np.array_equal(snr1[0], b1) and np.array_equal(id1[0], j1)
    assert np.array_equal(snr2[0], b2) and np.array_equal(id2[0], j2)
    assert not np.any(id1 == 2) or np.all(snr1[id1 == 2] > 0)             # ties keep the smaller id ...
    assert not np.any((id1 == 2))                                          # ... so the duplicate never wins
    peak = int(np.argmax(snr1[0]))
    # a real correlation output oscillates at the carrier (4 samples per cycle at 1 kHz): the largest |rho| may sit a
    # cycle or two off the envelope maximum at n0
    assert id1[0, peak] == 1 and abs(peak - n0) <= 8 and snr1[0, peak] > 8.0
    assert snr2[0, max(0, n0 - 50): n0 + 50].max() < 5.0                  # nothing in the other detector there
    both = (id1[0] != none) & (id2[0] != none)
    n_sim, n_coi = bo.dual_coincidences(id1, id2, f0, 50.0)
    assert n_sim == int(both.sum())
    assert n_coi == int(np.sum(np.abs(f0[id1[0][both]] - f0[id2[0][both]]) < 50.0))
