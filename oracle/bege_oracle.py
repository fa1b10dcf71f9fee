"""ctypes face of oracle/bege_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
reference legs may import this module.  It marshals numpy arrays into the plain
fp64 C oracle and holds no arithmetic of the method itself.  It never imports
the CUDA package.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "bege_oracle.c"
_LIB = _HERE / "libbege_oracle.so"


def build(force: bool = False) -> Path:
    """Compile the C oracle with gcc (fp64, OpenMP over templates)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".so.tmp{os.getpid()}")
        subprocess.check_call(
            ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp",
             "-ffp-contract=off", "-o", str(tmp), str(_SRC), "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class _Tail(ctypes.Structure):
    _fields_ = [("template_id", ctypes.c_uint32), ("lag", ctypes.c_uint32), ("snr", ctypes.c_double)]


TAIL_DTYPE = np.dtype([("template_id", "<u4"), ("lag", "<u4"), ("snr", "<f8")], align=True)
assert TAIL_DTYPE.itemsize == ctypes.sizeof(_Tail)

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(str(build()))
        dp = ctypes.POINTER(ctypes.c_double)
        u32, u64, dbl = ctypes.c_uint32, ctypes.c_uint64, ctypes.c_double
        L.bo_fft.argtypes = [dp, u32, ctypes.c_int]
        L.bo_fft.restype = ctypes.c_int
        L.bo_template.argtypes = [dbl, dbl, dbl, dbl, u32, dp]
        L.bo_template.restype = ctypes.c_int
        L.bo_band_mask.argtypes = [dp, u32, dbl, dbl, dbl]
        L.bo_band_mask.restype = None
        L.bo_segment_spectrum.argtypes = [dp, u32, dbl, dbl, dbl, dp]
        L.bo_segment_spectrum.restype = ctypes.c_int
        L.bo_correlate_spectra.argtypes = [dp, dp, u32, dp, dp]
        L.bo_correlate_spectra.restype = ctypes.c_int
        L.bo_correlate.argtypes = [dp, dp, u32, dp, dp]
        L.bo_correlate.restype = ctypes.c_int
        L.bo_correlate_direct.argtypes = [dp, dp, u32, u32, ctypes.POINTER(u32), u32, dp]
        L.bo_correlate_direct.restype = None
        L.bo_search.argtypes = [dp, u32, dp, dp, u64, dbl, dbl, u32, dbl,
                                ctypes.POINTER(_Tail), u64, dp, ctypes.c_int,
                                ctypes.POINTER(ctypes.c_int)]
        L.bo_search.restype = u64
        L.bo_search_maxproj.argtypes = [dp, u32, dp, dp, u64, dbl, dbl, u32, dbl, dp, ctypes.POINTER(u32)]
        L.bo_search_maxproj.restype = ctypes.c_int
        L.bo_search_band.argtypes = [dp, u32, dp, dp, u64, dbl, dbl, u32, dbl, dbl, ctypes.POINTER(_Tail), u64]
        L.bo_search_band.restype = u64
        L.bo_template_real.argtypes = [dbl, dbl, dbl, dbl, u32, dp]
        L.bo_template_real.restype = ctypes.c_int
        L.bo_template_real_sym.argtypes = [dbl, dbl, dbl, dbl, u32, dp]
        L.bo_template_real_sym.restype = ctypes.c_int
        L.bo_search_dual_sym.argtypes = [dp, u32, dp, dp, u64, dbl, dbl, u32, dbl, dp, ctypes.POINTER(u32), dp,
                                         ctypes.POINTER(u32), dp]
        L.bo_search_dual_sym.restype = ctypes.c_int
        L.bo_correlate_dual.argtypes = [dp, dp, u32, dp, dp, dp]
        L.bo_correlate_dual.restype = ctypes.c_int
        L.bo_sigma_dual_parseval.argtypes = [dp, dp, u32, dp, dp]
        L.bo_sigma_dual_parseval.restype = None
        L.bo_search_dual.argtypes = [dp, u32, dp, dp, u64, dbl, dbl, u32, dbl, dp, ctypes.POINTER(u32), dp,
                                     ctypes.POINTER(u32), dp]
        L.bo_search_dual.restype = ctypes.c_int
        L.bo_dual_coincidences.argtypes = [ctypes.POINTER(u32), ctypes.POINTER(u32), u64, dp, dbl,
                                           ctypes.POINTER(u64), ctypes.POINTER(u64)]
        L.bo_dual_coincidences.restype = None
        L.bo_fft_flops.argtypes = [u32]
        L.bo_fft_flops.restype = dbl
        _lib = L
    return _lib


def _dp(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _c128(a) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a, dtype=np.complex128))


def fft(a, sign: int) -> np.ndarray:
    """Unnormalised DFT with exp(sign*2*pi*i*k*n/N) (bo_fft)."""
    out = _c128(a).copy()
    rc = lib().bo_fft(_dp(out.view(np.float64)), out.size, int(sign))
    if rc:
        raise ValueError(f"bo_fft rc={rc}")
    return out


def template(f0: float, fdot: float, tau: float, fs: float, N: int) -> np.ndarray:
    h = np.zeros(N, dtype=np.complex128)
    rc = lib().bo_template(float(f0), float(fdot), float(tau), float(fs), N, _dp(h.view(np.float64)))
    if rc:
        raise ValueError(f"bo_template rc={rc}")
    return h


def band_mask(X, fs: float, lo: float, hi: float) -> np.ndarray:
    out = _c128(X).copy()
    lib().bo_band_mask(_dp(out.view(np.float64)), out.size, float(fs), float(lo), float(hi))
    return out


def segment_spectrum(x, fs: float, lo: float, hi: float) -> np.ndarray:
    x = _c128(x)
    X = np.empty_like(x)
    rc = lib().bo_segment_spectrum(_dp(x.view(np.float64)), x.size, float(fs), float(lo), float(hi),
                                   _dp(X.view(np.float64)))
    if rc:
        raise ValueError(f"bo_segment_spectrum rc={rc}")
    return X


def correlate(X, h, want_z: bool = True):
    """(z, sigma) of one pair from the masked spectrum X and time-domain template h."""
    X, h = _c128(X), _c128(h)
    z = np.empty_like(X) if want_z else None
    sig = ctypes.c_double(0.0)
    rc = lib().bo_correlate(_dp(X.view(np.float64)), _dp(h.view(np.float64)), X.size,
                            _dp(z.view(np.float64)) if want_z else None, ctypes.byref(sig))
    if rc:
        raise ValueError(f"bo_correlate rc={rc}")
    return z, sig.value


def correlate_direct(xhat, h, L: int, lags=None) -> np.ndarray:
    """z at the given lags (all N if None) by the time-domain sum of eq.(3)."""
    xhat, h = _c128(xhat), _c128(h)
    N = xhat.size
    if lags is None:
        lag_arr, n = None, N
    else:
        lag_arr = np.ascontiguousarray(np.asarray(lags, dtype=np.uint32))
        n = lag_arr.size
    z = np.empty(n, dtype=np.complex128)
    lib().bo_correlate_direct(
        _dp(xhat.view(np.float64)), _dp(h.view(np.float64)), N, int(L),
        lag_arr.ctypes.data_as(ctypes.POINTER(ctypes.c_uint32)) if lag_arr is not None else None,
        n, _dp(z.view(np.float64)))
    return z


def search(Xs, f0, fdot, tau: float, fs: float, k_sigma: float, cap: int = 1 << 22,
           n_threads: int = 0):
    """Whole path.  Xs: (S, N) masked spectra.  Returns (tails sorted by (id, lag),
    n_tails_true, sigma[T, S], threads_used)."""
    Xs = np.atleast_2d(_c128(Xs))
    S, N = Xs.shape
    f0 = np.ascontiguousarray(np.asarray(f0, dtype=np.float64))
    fdot = np.ascontiguousarray(np.asarray(fdot, dtype=np.float64))
    T = f0.size
    assert fdot.size == T
    tails = np.zeros(max(cap, 1), dtype=TAIL_DTYPE)
    sigma = np.zeros((T, S), dtype=np.float64)
    used = ctypes.c_int(0)
    n = lib().bo_search(_dp(Xs.view(np.float64)), S, _dp(f0), _dp(fdot), T, float(tau), float(fs), N,
                        float(k_sigma), tails.ctypes.data_as(ctypes.POINTER(_Tail)), cap,
                        _dp(sigma), int(n_threads), ctypes.byref(used))
    if n == 2**64 - 1:
        raise RuntimeError("bo_search failed")
    tails = tails[: min(n, cap)]
    tails = tails[np.lexsort((tails["lag"], tails["template_id"]))]
    return tails, int(n), sigma, used.value


def search_maxproj(Xs, f0, fdot, tau: float, fs: float, k_sigma: float):
    """Max projection over the bank (bo_search_maxproj): (snr[S, N] fp64, template_id[S, N] uint32)."""
    Xs = np.atleast_2d(_c128(Xs))
    S, N = Xs.shape
    f0 = np.ascontiguousarray(np.asarray(f0, dtype=np.float64))
    fdot = np.ascontiguousarray(np.asarray(fdot, dtype=np.float64))
    snr = np.zeros((S, N), dtype=np.float64)
    ids = np.zeros((S, N), dtype=np.uint32)
    rc = lib().bo_search_maxproj(_dp(Xs.view(np.float64)), S, _dp(f0), _dp(fdot), f0.size, float(tau), float(fs), N,
                                 float(k_sigma), _dp(snr), ids.ctypes.data_as(ctypes.POINTER(ctypes.c_uint32)))
    if rc:
        raise RuntimeError(f"bo_search_maxproj rc={rc}")
    return snr, ids


def search_band(Xs, f0, fdot, tau: float, fs: float, k_lo: float, k_hi: float, cap: int = 1 << 22):
    """Band threshold k_lo*sigma < |z| < k_hi*sigma (bo_search_band): (tails sorted by (id, lag), n_true)."""
    Xs = np.atleast_2d(_c128(Xs))
    S, N = Xs.shape
    f0 = np.ascontiguousarray(np.asarray(f0, dtype=np.float64))
    fdot = np.ascontiguousarray(np.asarray(fdot, dtype=np.float64))
    tails = np.zeros(max(cap, 1), dtype=TAIL_DTYPE)
    n = lib().bo_search_band(_dp(Xs.view(np.float64)), S, _dp(f0), _dp(fdot), f0.size, float(tau), float(fs), N,
                             float(k_lo), float(k_hi), tails.ctypes.data_as(ctypes.POINTER(_Tail)), cap)
    if n == 2**64 - 1:
        raise RuntimeError("bo_search_band failed")
    tails = tails[: min(n, cap)]
    return tails[np.lexsort((tails["lag"], tails["template_id"]))], int(n)


def template_real(f0: float, fdot: float, tau: float, fs: float, N: int) -> np.ndarray:
    """Real chirp template of the dual-stream search (bo_template_real), as a complex128 array with zero imaginary part."""
    h = np.zeros(N, dtype=np.complex128)
    if lib().bo_template_real(float(f0), float(fdot), float(tau), float(fs), N, _dp(h.view(np.float64))):
        raise ValueError("bo_template_real: bad arguments")
    return h


def template_real_sym(f0: float, fdot: float, tau: float, fs: float, N: int) -> np.ndarray:
    """Time-symmetric real template (bo_template_real_sym): the chirp plus its time reverse, unit norm."""
    h = np.zeros(N, dtype=np.complex128)
    if lib().bo_template_real_sym(float(f0), float(fdot), float(tau), float(fs), N, _dp(h.view(np.float64))):
        raise ValueError("bo_template_real_sym: bad arguments")
    return h


def correlate_dual(X, h):
    """(z, sigma_1, sigma_2) for a packed segment spectrum X and a real template h (time domain)."""
    X = _c128(X)
    N = X.size
    Hs = fft(h, -1)
    z = np.zeros(N, dtype=np.complex128)
    s1, s2 = ctypes.c_double(), ctypes.c_double()
    if lib().bo_correlate_dual(_dp(X.view(np.float64)), _dp(Hs.view(np.float64)), N, _dp(z.view(np.float64)),
                               ctypes.byref(s1), ctypes.byref(s2)):
        raise RuntimeError("bo_correlate_dual failed")
    return z, s1.value, s2.value


def sigma_dual_parseval(X, h):
    """(sigma_1, sigma_2) from the product spectrum alone, eq.(7)."""
    X = _c128(X)
    Hs = fft(h, -1)
    s1, s2 = ctypes.c_double(), ctypes.c_double()
    lib().bo_sigma_dual_parseval(_dp(X.view(np.float64)), _dp(Hs.view(np.float64)), X.size, ctypes.byref(s1), ctypes.byref(s2))
    return s1.value, s2.value


def search_dual(Xs, f0, fdot, tau: float, fs: float, k_sigma: float, symmetric: bool = False):
    """Dual-stream search (bo_search_dual; symmetric: bo_search_dual_sym, the time-symmetric templates of PAPER.md:70):
    (snr1[S, N], id1[S, N], snr2[S, N], id2[S, N], sigma[T, S, 2])."""
    Xs = np.atleast_2d(_c128(Xs))
    S, N = Xs.shape
    f0 = np.ascontiguousarray(np.asarray(f0, dtype=np.float64))
    fdot = np.ascontiguousarray(np.asarray(fdot, dtype=np.float64))
    snr1, snr2 = np.zeros((S, N)), np.zeros((S, N))
    id1, id2 = np.zeros((S, N), dtype=np.uint32), np.zeros((S, N), dtype=np.uint32)
    sig = np.zeros((f0.size, S, 2))
    u32p = ctypes.POINTER(ctypes.c_uint32)
    fn = lib().bo_search_dual_sym if symmetric else lib().bo_search_dual
    rc = fn(_dp(Xs.view(np.float64)), S, _dp(f0), _dp(fdot), f0.size, float(tau), float(fs), N,
                              float(k_sigma), _dp(snr1), id1.ctypes.data_as(u32p), _dp(snr2), id2.ctypes.data_as(u32p),
                              _dp(sig))
    if rc:
        raise RuntimeError(f"bo_search_dual rc={rc}")
    return snr1, id1, snr2, id2, sig


def dual_coincidences(id1, id2, f0, delta_hz: float):
    """(offsets with a hit in both streams, those with |f_1 - f_2| < delta_hz)."""
    id1 = np.ascontiguousarray(id1, dtype=np.uint32).ravel()
    id2 = np.ascontiguousarray(id2, dtype=np.uint32).ravel()
    f0 = np.ascontiguousarray(np.asarray(f0, dtype=np.float64))
    a, b = ctypes.c_uint64(), ctypes.c_uint64()
    u32p = ctypes.POINTER(ctypes.c_uint32)
    lib().bo_dual_coincidences(id1.ctypes.data_as(u32p), id2.ctypes.data_as(u32p), id1.size, _dp(f0), float(delta_hz),
                               ctypes.byref(a), ctypes.byref(b))
    return int(a.value), int(b.value)


def fft_flops(N: int) -> float:
    return lib().bo_fft_flops(N)
