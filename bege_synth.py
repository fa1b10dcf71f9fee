"""Seeded synthetic inputs shaped like the paper's workload.

This module serves BOTH the oracle-side tests and the CUDA-side bench; it holds
none of the method's arithmetic (no correlation, no sigma, no threshold) and
imports neither `oracle/` nor the CUDA binding.  It stands in for the paper's
LIGO S6 H1^L1 data base, which is not available here:
16 s segments at 4096 Hz (N = 2^16), near-Gaussian noise band-passed to
350-2000 Hz, one-second chirp banks on the (f, fdot)
plane and Q = 9 sine-Gaussian bursts.

`numpy.fft` is used only to band-pass the *data* (the paper's data-base
preparation), never as a step of the search.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

FS = 4096.0
N_SEG = 1 << 16
BAND = (350.0, 2000.0)
TAU = 1.0


# --------------------------------------------------------------------------- data
def band_limit(x: np.ndarray, fs: float = FS, lo: float = BAND[0], hi: float = BAND[1]) -> np.ndarray:
    """Zero all FFT bins with |f| outside [lo, hi] (inclusive); returns a real/complex fp64 series."""
    n = x.shape[-1]
    f = np.abs(np.fft.fftfreq(n, d=1.0 / fs))
    keep = (f >= lo) & (f <= hi)
    y = np.fft.ifft(np.fft.fft(x, axis=-1) * keep, axis=-1)
    return y.real if np.isrealobj(x) else y


def white_noise(seed: int, n: int = N_SEG) -> np.ndarray:
    """`default_rng(seed).standard_normal(n)`: mean 0, std 1 BEFORE band-limiting."""
    return np.random.default_rng(seed).standard_normal(n)


def as_segment(x: np.ndarray) -> np.ndarray:
    """Store a real fp64 series the way the path takes it: complex64, zero imaginary part."""
    return np.ascontiguousarray(x.astype(np.float32).astype(np.complex64))


def noise_segment(seed: int, n: int = N_SEG, fs: float = FS, band=BAND) -> np.ndarray:
    return as_segment(band_limit(white_noise(seed, n), fs, *band))


def chirp_signal(f0: float, fdot: float, tau: float = TAU, fs: float = FS) -> np.ndarray:
    """Unit-norm Hann-windowed linear chirp of L = round(tau*fs) samples (the signal model injected
    into the data; the search's own template synthesis lives in the oracle and in the CUDA path)."""
    L = int(round(tau * fs))
    t = np.arange(L) / fs
    s = np.hanning(L) * np.exp(2j * np.pi * (f0 * t + 0.5 * fdot * t * t))
    return s / np.linalg.norm(s)


def in_band_fraction(s: np.ndarray, n: int, fs: float = FS, band=BAND) -> float:
    """Share of the energy of `s` (zero-padded to n) at |f| inside the band."""
    p = np.abs(np.fft.fft(s, n)) ** 2
    f = np.abs(np.fft.fftfreq(n, d=1.0 / fs))
    return float(p[(f >= band[0]) & (f <= band[1])].sum() / p.sum())


def inject_chirp(x: np.ndarray, f0: float, fdot: float, t0: float, snr: float,
                 tau: float = TAU, fs: float = FS, band=BAND) -> tuple[np.ndarray, int]:
    """Add A*Re(chirp) starting at sample n0 = round(t0*fs) (wrapping circularly).
    A = 2*snr/sqrt(in-band energy fraction): the noise-free matched output at the exact template is
    ~A/2 times that fraction while sigma on unit white noise is its square root (reading 14)."""
    n = x.shape[-1]
    s = chirp_signal(f0, fdot, tau, fs)
    amp = 2.0 * snr / np.sqrt(in_band_fraction(s, n, fs, band))
    n0 = int(round(t0 * fs))
    idx = (n0 + np.arange(s.size)) % n
    y = x.copy()
    y[idx] += amp * s.real
    return y, n0


def sine_gaussian(n: int, fc: float, t0: float, snr: float, phi: float, q: float = 9.0,
                  fs: float = FS) -> np.ndarray:
    """s(t) = A sin(2 pi fc (t-t0) + phi) exp(-(t-t0)^2/tg^2), tg = Q/(sqrt(2) pi fc), ||s||_2 = snr
    (Table 4 gives only (f, Q = 9); reading 15)."""
    t = np.arange(n) / fs
    tg = q / (np.sqrt(2.0) * np.pi * fc)
    s = np.sin(2 * np.pi * fc * (t - t0) + phi) * np.exp(-((t - t0) ** 2) / tg ** 2)
    return s * (snr / np.linalg.norm(s))


# --------------------------------------------------------------------------- bank
def bank_grid(n_f0: int, n_fdot: int, f0_lo: float, f0_hi: float, fdot_lo: float, fdot_hi: float):
    """f0-major flattening: id = i_f0 * n_fdot + i_fdot, linspace endpoints inclusive."""
    f0 = np.linspace(f0_lo, f0_hi, n_f0)
    fd = np.linspace(fdot_lo, fdot_hi, n_fdot)
    return (np.ascontiguousarray(np.repeat(f0, n_fdot)),
            np.ascontiguousarray(np.tile(fd, n_f0)))


# ------------------------------------------------------------------------ configs
@dataclass
class Workload:
    name: str
    x: np.ndarray                 # (S, N) complex64
    f0: np.ndarray                # (T,) fp64
    fdot: np.ndarray              # (T,) fp64
    k_sigma: float
    fs: float = FS
    band: tuple = BAND
    tau: float = TAU
    meta: dict = field(default_factory=dict)

    @property
    def n_templates(self) -> int:
        return int(self.f0.size)

    @property
    def n_segments(self) -> int:
        return int(self.x.shape[0])


def config0() -> Workload:
    """BASELINE.json configs[0]: 1 noise segment (seed 0), 16x16 bank, k = 5."""
    f0, fd = bank_grid(16, 16, 400.0, 1900.0, -200.0, 200.0)
    return Workload("cfg0_256x1", noise_segment(0)[None, :], f0, fd, 5.0)


def config1(sub: int | None = None) -> Workload:
    """configs[1]: seed 1 + chirp (1100 Hz, -80 Hz/s, t0 = 7.3 s, SNR 12), 256x256 bank, k = 5."""
    x = band_limit(white_noise(1))
    x, n0 = inject_chirp(x, 1100.0, -80.0, 7.3, 12.0)
    f0, fd = bank_grid(256, 256, 350.0, 2000.0, -400.0, 400.0)
    return Workload("cfg1_65536x1", as_segment(x)[None, :], f0, fd, 5.0,
                    meta={"n0": n0, "inj": (1100.0, -80.0), "true_id": 116 * 256 + 102})


def config2_bank():
    """configs[2] bank: 1024x1024 grid, 2^20 templates."""
    return bank_grid(1024, 1024, 350.0, 2000.0, -400.0, 400.0)


def config2() -> Workload:
    """configs[2]: paper-scale bank, 1 noise segment (seed 2), k = 6."""
    f0, fd = config2_bank()
    return Workload("cfg2_1048576x1", noise_segment(2)[None, :], f0, fd, 6.0)


def config3(n_seg: int = 64) -> Workload:
    """configs[3]: 64 segments (seeds 100..163), 4 carrying chirps (SNR 8-15), 256x256 bank, k = 5."""
    pick = np.sort(np.random.default_rng(1000).choice(n_seg, size=min(4, n_seg), replace=False))
    xs, inj = [], {}
    for m in range(n_seg):
        seed = 100 + m
        x = band_limit(white_noise(seed))
        if m in pick:
            r = np.random.default_rng(1000 + seed)
            p = dict(f0=r.uniform(400.0, 1800.0), fdot=r.uniform(-300.0, 300.0),
                     t0=r.uniform(0.0, 15.0), snr=r.uniform(8.0, 15.0))
            x, n0 = inject_chirp(x, p["f0"], p["fdot"], p["t0"], p["snr"])
            p["n0"] = n0
            inj[m] = p
        xs.append(as_segment(x))
    f0, fd = bank_grid(256, 256, 350.0, 2000.0, -400.0, 400.0)
    return Workload(f"cfg3_65536x{n_seg}", np.stack(xs), f0, fd, 5.0, meta={"injections": inj})


def config4() -> Workload:
    """configs[4]: seed 3 + 40 Q=9 sine-Gaussian glitches, 512x512 bank, k = 3 (tail-heavy)."""
    r = np.random.default_rng(3)
    x = r.standard_normal(N_SEG)
    for _ in range(40):
        fc, t0 = r.uniform(350.0, 2000.0), r.uniform(0.5, 15.5)
        snr, phi = r.uniform(10.0, 50.0), r.uniform(0.0, 2 * np.pi)
        x = x + sine_gaussian(N_SEG, fc, t0, snr, phi)
    f0, fd = bank_grid(512, 512, 350.0, 2000.0, -400.0, 400.0)
    return Workload("cfg4_262144x1", as_segment(band_limit(x))[None, :], f0, fd, 3.0)


def subsample(w: Workload, ids) -> Workload:
    """Same data, a subset of the bank (parity tests on a sub-sampled bank)."""
    ids = np.asarray(ids, dtype=np.int64)
    return Workload(w.name + f"_sub{ids.size}", w.x, np.ascontiguousarray(w.f0[ids]),
                    np.ascontiguousarray(w.fdot[ids]), w.k_sigma, w.fs, w.band, w.tau,
                    dict(w.meta, ids=ids))
