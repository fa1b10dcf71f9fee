"""bege -- B200-native FFT matched filtering over chirp-template banks (arXiv:1708.01609 hot path).

`paper_1708_01609_b200.bege` is the thin Python binding over the C-ABI library
(`include/bege.h`, built from `csrc/`).  The seeded synthetic inputs that serve both
the oracle-side tests and the CUDA-side bench live outside the product package, in
`bege_synth.py` at the repo root.  Importing this package does not load the CUDA
library; the first use of the binding does, and fails loudly if it is missing.
"""
__all__ = ["bege", "shard", "build"]
