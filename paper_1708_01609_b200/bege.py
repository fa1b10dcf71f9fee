"""Thin Python binding over the C-ABI library (include/bege.h): argument marshalling only.

Every step of the path runs in the library's sm_100a kernels.  PyTorch is used for device memory
(the workspace tensor), pinned host buffers and the stream handle; numpy for host arrays.
There is no CPU fallback: if `libbege.so` is missing or no CUDA device is present, calls raise.
"""
from __future__ import annotations

import ctypes
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
LIB_PATH = _HERE / "libbege.so"
PROBE_LIB_PATH = _HERE / "libbege_probe.so"      # measurement probes (include/bege_probe.h), not part of the product ABI

TAIL_DTYPE = np.dtype([("template_id", "<u4"), ("lag", "<u4"), ("snr", "<f4")])
assert TAIL_DTYPE.itemsize == 12

OK, EINVAL, ESTATE, ENOMEM, ECUDA, EOVERFLOW = range(6)
CUDA_STREAM_LEGACY = 0x1          # cudaStreamLegacy (driver_types.h): the legacy default stream as an explicit handle
_STATUS = {0: "BEGE_OK", 1: "BEGE_EINVAL", 2: "BEGE_ESTATE", 3: "BEGE_ENOMEM", 4: "BEGE_ECUDA", 5: "BEGE_EOVERFLOW"}

# every symbol include/bege.h declares (tests check that the library exports all of them)
SYMBOLS = [
    "bege_plan_create", "bege_plan_workspace_bytes", "bege_plan_set_workspace", "bege_bank_generate",
    "bege_segment_load", "bege_search", "bege_search_band", "bege_search_maxproj", "bege_get_sigma", "bege_debug_correlate",
    "bege_bank_generate_real", "bege_search_dual", "bege_get_sigma_dual",
    "bege_debug_template_spectrum", "bege_debug_segment_spectrum", "bege_debug_set_max_items", "bege_plan_set_profiling",
    "bege_plan_get_stats", "bege_plan_reset_stats", "bege_last_error", "bege_plan_destroy", "bege_version",
    "bege_segment_spectrum_static", "bege_bank_generate_real_symmetric",
]
PROBE_SYMBOLS = ["bege_ovs_probe"]   # include/bege_probe.h
STATIC_MAX_SEGMENTS = 4           # BEGE_STATIC_MAX_SEGMENTS (include/bege.h)


class BegeError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"{_STATUS.get(status, status)}: {msg}")
        self.status = status


class Stats(ctypes.Structure):
    _fields_ = [("kernel_launches", ctypes.c_uint64), ("correlations", ctypes.c_uint64),
                ("fused_kernel_ms", ctypes.c_double), ("fused_kernel_launches", ctypes.c_uint64),
                ("hbm_bytes_per_template", ctypes.c_uint64)]


_lib = None


def load_library() -> ctypes.CDLL:
    """dlopen the in-tree CUDA library; fails loudly when it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not LIB_PATH.exists():
        raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_1708_01609_b200.build` "
                           "(or __graft_entry__.build()); there is no CPU fallback")
    L = ctypes.CDLL(str(LIB_PATH))
    vp, u32, u64, dbl, i32 = ctypes.c_void_p, ctypes.c_uint32, ctypes.c_uint64, ctypes.c_double, ctypes.c_int
    L.bege_plan_create.argtypes = [ctypes.POINTER(vp), u32, dbl, dbl, dbl, i32, vp]
    L.bege_plan_workspace_bytes.argtypes = [vp, u64, u32, u64, ctypes.POINTER(u64)]
    L.bege_plan_set_workspace.argtypes = [vp, vp, u64]
    L.bege_bank_generate.argtypes = [vp, vp, vp, u64, dbl]
    L.bege_segment_load.argtypes = [vp, vp, u32]
    L.bege_search.argtypes = [vp, ctypes.c_float, vp, u64, ctypes.POINTER(u64)]
    L.bege_search_band.argtypes = [vp, ctypes.c_float, ctypes.c_float, vp, u64, ctypes.POINTER(u64)]
    L.bege_search_maxproj.argtypes = [vp, ctypes.c_float, vp, vp, ctypes.POINTER(u64)]
    L.bege_get_sigma.argtypes = [vp, vp]
    L.bege_bank_generate_real.argtypes = [vp, vp, vp, u64, dbl]
    L.bege_bank_generate_real_symmetric.argtypes = [vp, vp, vp, u64, dbl]
    L.bege_search_dual.argtypes = [vp, ctypes.c_float, vp, vp, vp, vp, dbl, ctypes.POINTER(u64), ctypes.POINTER(u64)]
    L.bege_get_sigma_dual.argtypes = [vp, vp, vp]
    L.bege_debug_correlate.argtypes = [vp, u64, u32, vp, ctypes.POINTER(ctypes.c_float)]
    L.bege_debug_template_spectrum.argtypes = [vp, u64, vp]
    L.bege_debug_segment_spectrum.argtypes = [vp, u32, vp]
    L.bege_debug_set_max_items.argtypes = [vp, u64]
    L.bege_segment_spectrum_static.argtypes = [i32, vp, dbl, dbl, dbl, vp, u32, vp, ctypes.c_char_p, u64]
    L.bege_plan_set_profiling.argtypes = [vp, i32]
    L.bege_plan_get_stats.argtypes = [vp, ctypes.POINTER(Stats)]
    L.bege_plan_reset_stats.argtypes = [vp]
    L.bege_last_error.argtypes = [vp]
    L.bege_last_error.restype = ctypes.c_char_p
    L.bege_plan_destroy.argtypes = [vp]
    L.bege_plan_destroy.restype = None
    L.bege_version.restype = ctypes.c_char_p
    for name in SYMBOLS:
        if name not in ("bege_last_error", "bege_plan_destroy", "bege_version"):
            getattr(L, name).restype = i32
    _lib = L
    return L


_probe_lib = None


def load_probe_library() -> ctypes.CDLL:
    """dlopen the in-tree probe library (experiments that are deliberately not in libbege.so)."""
    global _probe_lib
    if _probe_lib is None:
        if not PROBE_LIB_PATH.exists():
            raise RuntimeError(f"{PROBE_LIB_PATH} is missing: build it with `python -m paper_1708_01609_b200.build`")
        L = ctypes.CDLL(str(PROBE_LIB_PATH))
        vp, u32, u64, dbl, i32 = ctypes.c_void_p, ctypes.c_uint32, ctypes.c_uint64, ctypes.c_double, ctypes.c_int
        L.bege_ovs_probe.argtypes = [i32, u64, u32, u32, ctypes.c_float, vp, vp, vp, u64, ctypes.POINTER(dbl), ctypes.POINTER(u64)]
        L.bege_ovs_probe.restype = i32
        _probe_lib = L
    return _probe_lib


class Plan:
    """One plan = one device, one stream (include/bege.h).  Names follow the C ABI."""

    def __init__(self, N: int = 1 << 16, fs: float = 4096.0, band=(350.0, 2000.0), device: int = 0,
                 stream: int | str | None = None):
        """stream: a cudaStream_t handle (e.g. torch.cuda.Stream().cuda_stream), None for torch's current stream,
        or "own" for a private non-blocking stream created and owned by the plan (cuda_stream = NULL in the C ABI)."""
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("bege needs a CUDA device (sm_100a); there is no CPU fallback")
        self._L = load_library()
        self.N, self.fs, self.band, self.device = int(N), float(fs), tuple(band), int(device)
        if stream == "own":
            stream = None                 # NULL in the C ABI: the plan creates (and owns) a non-blocking stream
        elif stream is None:
            stream = torch.cuda.current_stream(self.device).cuda_stream
        if stream == 0:
            # torch's default stream is the legacy default stream; handle 0 would read as "no stream given" and make
            # the plan create a private non-blocking stream that is NOT ordered after work torch has queued (e.g. the
            # kernel that produced a CUDA tensor passed to segment_load).  cudaStreamLegacy names it explicitly.
            stream = CUDA_STREAM_LEGACY
        h = ctypes.c_void_p()
        rc = self._L.bege_plan_create(ctypes.byref(h), self.N, self.fs, float(band[0]), float(band[1]),
                                      self.device, ctypes.c_void_p(stream))
        if rc != OK:
            raise BegeError(rc, "bege_plan_create failed")
        self._h = h
        self._ws = None
        self._pinned = None
        self.n_templates = 0
        self.n_segments = 0

    # -- helpers
    def _check(self, rc: int, allow=()):
        if rc != OK and rc not in allow:
            raise BegeError(rc, self._L.bege_last_error(self._h).decode())
        return rc

    def close(self):
        if getattr(self, "_h", None):
            self._L.bege_plan_destroy(self._h)
            self._h = None
            self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    # -- C ABI, one method per entry point
    def workspace_bytes(self, n_templates: int, n_segments: int, cap: int) -> int:
        out = ctypes.c_uint64()
        self._check(self._L.bege_plan_workspace_bytes(self._h, n_templates, n_segments, cap, ctypes.byref(out)))
        return out.value

    def set_workspace(self, tensor=None):
        """tensor: a torch uint8 CUDA tensor the plan may carve up (kept alive here), or None."""
        if tensor is None:
            self._check(self._L.bege_plan_set_workspace(self._h, None, 0))
        else:
            assert tensor.is_cuda and tensor.is_contiguous()
            self._check(self._L.bege_plan_set_workspace(self._h, ctypes.c_void_p(tensor.data_ptr()),
                                                        tensor.numel() * tensor.element_size()))
        self._ws = tensor
        self.n_templates = self.n_segments = 0

    def alloc_workspace(self, n_templates: int, n_segments: int, cap: int):
        import torch

        nbytes = self.workspace_bytes(n_templates, n_segments, cap)
        self.set_workspace(torch.empty(nbytes, dtype=torch.uint8, device=f"cuda:{self.device}"))
        return nbytes

    def bank_generate(self, f0, fdot, tau: float = 1.0):
        f0 = np.ascontiguousarray(np.asarray(f0, dtype=np.float64))
        fdot = np.ascontiguousarray(np.asarray(fdot, dtype=np.float64))
        assert f0.ndim == 1 and f0.shape == fdot.shape
        self._check(self._L.bege_bank_generate(self._h, f0.ctypes.data, fdot.ctypes.data, f0.size, float(tau)))
        self.n_templates = int(f0.size)

    def bank_generate_real(self, f0, fdot, tau: float = 1.0, symmetric: bool = False):
        """Bank of real templates (dual-stream search).  symmetric: bege_bank_generate_real_symmetric, the paper's
        time-symmetric chirps (forward + backward in time)."""
        f0 = np.ascontiguousarray(np.asarray(f0, dtype=np.float64))
        fdot = np.ascontiguousarray(np.asarray(fdot, dtype=np.float64))
        assert f0.ndim == 1 and f0.shape == fdot.shape
        fn = self._L.bege_bank_generate_real_symmetric if symmetric else self._L.bege_bank_generate_real
        self._check(fn(self._h, f0.ctypes.data, fdot.ctypes.data, f0.size, float(tau)))
        self.n_templates = int(f0.size)

    def segment_load(self, x):
        """x: (S, N) complex64 -- numpy array, or torch tensor (CPU, pinned or CUDA)."""
        if isinstance(x, np.ndarray):
            x = np.ascontiguousarray(np.atleast_2d(x), dtype=np.complex64)
            assert x.shape[1] == self.N
            ptr, S, keep = x.ctypes.data, x.shape[0], x
        else:
            import torch

            assert x.dtype == torch.complex64 and x.is_contiguous()
            x = x.reshape(-1, self.N)
            ptr, S, keep = x.data_ptr(), x.shape[0], x
        self._check(self._L.bege_segment_load(self._h, ctypes.c_void_p(ptr), S))
        del keep
        self.n_segments = int(S)

    def pinned_tails(self, cap: int):
        """Pinned host buffer of `cap` records (reused between calls)."""
        import torch

        if self._pinned is None or self._pinned.numel() < cap * 12:
            self._pinned = torch.empty(max(cap, 1) * 12, dtype=torch.uint8).pin_memory()
        return self._pinned

    def search(self, k_sigma: float, cap: int = 1 << 20, copy: bool = True, allow_overflow: bool = False):
        """Returns (tails, n_tails): structured array of min(n_tails, cap) records (order unspecified)
        and the true count."""
        buf = self.pinned_tails(cap)
        n = ctypes.c_uint64()
        rc = self._check(self._L.bege_search(self._h, ctypes.c_float(k_sigma), ctypes.c_void_p(buf.data_ptr()),
                                             cap, ctypes.byref(n)),
                         allow=(EOVERFLOW,) if allow_overflow else ())
        got = min(n.value, cap)
        view = buf.numpy()[: got * 12].view(TAIL_DTYPE)
        return (view.copy() if copy else view), int(n.value)

    def search_band(self, k_lo: float, k_hi: float, cap: int = 1 << 20, copy: bool = True):
        """Band threshold k_lo*sigma < |z| < k_hi*sigma: (tails, n_tails) as `search`."""
        buf = self.pinned_tails(cap)
        n = ctypes.c_uint64()
        self._check(self._L.bege_search_band(self._h, ctypes.c_float(k_lo), ctypes.c_float(k_hi),
                                             ctypes.c_void_p(buf.data_ptr()), cap, ctypes.byref(n)))
        got = min(n.value, cap)
        view = buf.numpy()[: got * 12].view(TAIL_DTYPE)
        return (view.copy() if copy else view), int(n.value)

    def search_maxproj(self, k_sigma: float):
        """Max projection over the bank: (snr[S, N] float32, template_id[S, N] uint32, n_hits)."""
        snr = np.empty((self.n_segments, self.N), dtype=np.float32)
        ids = np.empty((self.n_segments, self.N), dtype=np.uint32)
        n = ctypes.c_uint64()
        self._check(self._L.bege_search_maxproj(self._h, ctypes.c_float(k_sigma), snr.ctypes.data, ids.ctypes.data,
                                                ctypes.byref(n)))
        return snr, ids, int(n.value)

    def search_dual(self, k_sigma: float, delta_hz: float = 50.0):
        """Dual-stream search (x = H1 + i L1): (snr1, id1, snr2, id2) of shape (S, N), n_simultaneous, n_coincident."""
        shape = (self.n_segments, self.N)
        snr1, snr2 = np.empty(shape, dtype=np.float32), np.empty(shape, dtype=np.float32)
        id1, id2 = np.empty(shape, dtype=np.uint32), np.empty(shape, dtype=np.uint32)
        ns, nc = ctypes.c_uint64(), ctypes.c_uint64()
        self._check(self._L.bege_search_dual(self._h, ctypes.c_float(k_sigma), snr1.ctypes.data, id1.ctypes.data,
                                             snr2.ctypes.data, id2.ctypes.data, float(delta_hz),
                                             ctypes.byref(ns), ctypes.byref(nc)))
        return snr1, id1, snr2, id2, int(ns.value), int(nc.value)

    def get_sigma_dual(self):
        s1 = np.empty((self.n_templates, self.n_segments), dtype=np.float32)
        s2 = np.empty((self.n_templates, self.n_segments), dtype=np.float32)
        self._check(self._L.bege_get_sigma_dual(self._h, s1.ctypes.data, s2.ctypes.data))
        return s1, s2

    def get_sigma(self) -> np.ndarray:
        out = np.empty((self.n_templates, self.n_segments), dtype=np.float32)
        self._check(self._L.bege_get_sigma(self._h, out.ctypes.data))
        return out

    def debug_correlate(self, template_id: int, segment: int = 0):
        z = np.empty(self.N, dtype=np.complex64)
        sig = ctypes.c_float()
        self._check(self._L.bege_debug_correlate(self._h, template_id, segment, z.ctypes.data, ctypes.byref(sig)))
        return z, float(sig.value)

    def debug_template_spectrum(self, template_id: int) -> np.ndarray:
        H = np.empty(self.N, dtype=np.complex64)
        self._check(self._L.bege_debug_template_spectrum(self._h, template_id, H.ctypes.data))
        return H

    def debug_segment_spectrum(self, segment: int) -> np.ndarray:
        X = np.empty(self.N, dtype=np.complex64)
        self._check(self._L.bege_debug_segment_spectrum(self._h, segment, X.ctypes.data))
        return X

    def debug_set_max_items(self, max_items: int):
        """(template, segment) items one kernel launch may take per CTA group; tests lower it to reach the launch split."""
        self._check(self._L.bege_debug_set_max_items(self._h, int(max_items)))

    def set_profiling(self, on: bool):
        self._check(self._L.bege_plan_set_profiling(self._h, int(bool(on))))

    def stats(self) -> dict:
        s = Stats()
        self._check(self._L.bege_plan_get_stats(self._h, ctypes.byref(s)))
        return {k: getattr(s, k) for k, _ in Stats._fields_}

    def reset_stats(self):
        self._check(self._L.bege_plan_reset_stats(self._h))


def ovs_probe(n_templates: int, n_blocks: int = 6, reps: int = 3, thr2: float = 3.0e38, h16=None, x16=None,
              want_z: bool = False, dbg_j: int = 0, device: int = 0):
    """bege_ovs_probe (include/bege_probe.h, libbege_probe.so): the overlap-save bake-off probe.
    Returns (ms per pass, hits, z or None)."""
    L = load_probe_library()
    ms, hits = ctypes.c_double(0.0), ctypes.c_uint64(0)
    z = np.empty((n_blocks, 16384), dtype=np.complex64) if want_z else None
    if h16 is not None:
        h16 = np.ascontiguousarray(h16, dtype=np.complex64)
        assert h16.shape == (n_templates, 16384)
    if x16 is not None:
        x16 = np.ascontiguousarray(x16, dtype=np.complex64)
        assert x16.shape == (n_blocks, 16384)
    rc = L.bege_ovs_probe(device, n_templates, n_blocks, reps, ctypes.c_float(thr2),
                          h16.ctypes.data if h16 is not None else None, x16.ctypes.data if x16 is not None else None,
                          z.ctypes.data if z is not None else None, dbg_j, ctypes.byref(ms), ctypes.byref(hits))
    if rc != OK:
        raise BegeError(rc, "bege_ovs_probe failed")
    return ms.value, hits.value, z


def segment_spectrum_static(x, fs: float = 4096.0, band=(350.0, 2000.0), out=None, stream: int | None = None):
    """bege_segment_spectrum_static (include/bege.h): band-limited spectra of up to STATIC_MAX_SEGMENTS segments with
    no device allocation inside the library -- for callers that may not call cudaMalloc when the spectrum is needed
    (latency-critical loops, processes whose HBM is already fully claimed, fixed-memory-budget pipelines).  The
    transform's staging area and tables are arrays built into libbege.so.

    x: torch CUDA tensor, complex64, (S, 65536) contiguous, S <= STATIC_MAX_SEGMENTS.  out: a tensor of the same shape to
    receive the spectra in natural bin order; pass one you made earlier if torch must not allocate either (None: a new
    tensor from torch's allocator).  The work is queued on `stream` (default: torch's current stream on x's device) and
    this returns without waiting.  All calls on a device share the built-in staging array: keep them on one stream or
    order them with events, unordered concurrent calls corrupt each other.  The first call on a device also does the
    one-time set-up and waits for the stream once; make it at start-up.  Raises BegeError with the library's message
    (e.g. when S exceeds the limit)."""
    import torch

    L = load_library()
    assert x.is_cuda and x.dtype == torch.complex64 and x.is_contiguous() and x.dim() == 2
    S, dev = int(x.shape[0]), x.device.index
    if out is None:
        out = torch.empty_like(x)
    assert out.is_cuda and out.dtype == torch.complex64 and out.is_contiguous() and out.shape == x.shape and out.device == x.device
    if stream is None:
        stream = torch.cuda.current_stream(dev).cuda_stream
    err = ctypes.create_string_buffer(256)
    rc = L.bege_segment_spectrum_static(dev, ctypes.c_void_p(stream or CUDA_STREAM_LEGACY), float(fs), float(band[0]),
                                        float(band[1]), ctypes.c_void_p(x.data_ptr()), S, ctypes.c_void_p(out.data_ptr()),
                                        err, len(err))
    if rc != OK:
        raise BegeError(rc, err.value.decode())
    return out


def version() -> str:
    return load_library().bege_version().decode()
