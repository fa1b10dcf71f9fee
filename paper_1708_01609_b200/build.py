"""Builds the C-ABI library `libbege.so` (the product) and `libbege_probe.so` (measurement probes kept out of the
product) in-tree with nvcc for sm_100a (no GPU needed to compile)."""
from __future__ import annotations

import os
import subprocess
import sys
from pathlib import Path

HERE = Path(__file__).resolve().parent
CSRC = HERE / "csrc"
LIB = HERE / "libbege.so"
PROBE_LIB = HERE / "libbege_probe.so"
SOURCES = [CSRC / "bege.cu"]
PROBE_SOURCES = [CSRC / "bege_probe.cu"]
# everything the libraries are compiled from: a change to any of these makes the built .so stale
HEADERS = sorted(CSRC.glob("*.cuh")) + sorted((HERE.parent / "include").glob("*.h"))

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-shared", "-Xcompiler", "-fPIC", "--use_fast_math=false"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def stale(lib: Path = LIB, sources=None) -> bool:
    if not lib.exists():
        return True
    t = lib.stat().st_mtime
    return any(f.stat().st_mtime > t for f in (sources or SOURCES) + HEADERS)


def _build(lib: Path, sources, force: bool, verbose: bool) -> Path:
    if not force and not stale(lib, sources):
        return lib
    tmp = lib.with_suffix(f".so.tmp{os.getpid()}")
    flags = [f for f in NVCC_FLAGS if not f.startswith("--use_fast_math")]
    cmd = [_nvcc(), *flags, *(["-Xptxas", "-v"] if verbose else []), "-o", str(tmp), *map(str, sources)]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose:
        sys.stderr.write(res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + res.stdout + res.stderr)
    os.replace(tmp, lib)
    return lib


def build_library(force: bool = False, verbose: bool = False) -> Path:
    """The product library (and, beside it, the probe library: tests and `bench.py --impl ovs_probe` load it)."""
    _build(PROBE_LIB, PROBE_SOURCES, force, verbose)
    return _build(LIB, SOURCES, force, verbose)


if __name__ == "__main__":
    print(build_library(force=True, verbose="-v" in sys.argv))
