"""The allocation-free entry point `bege_segment_spectrum_static` against the plan's own segment transform.  `-m gpu`.

Why the entry point exists: every other call of the library gets device memory from cudaMalloc or from a workspace the
caller allocated.  A caller inside a latency-critical loop (cudaMalloc stalls the whole device), in a process whose HBM is
already fully claimed by someone else, or under a no-allocation-after-start-up rule can do neither; for them the
library carries a small staging array and its twiddle tables as built-in device arrays (room for
BEGE_STATIC_MAX_SEGMENTS = 4 segments) and this call uses only those.

What is checked: its output equals the spectrum `bege_segment_load` stores (read back with
`bege_debug_segment_spectrum`) to the tolerance of test_gpu_parity.test_segment_spectrum_matches_oracle (rel-L2 < 1e-6,
identical set of zeroed bins), on TWO CALLS IN A ROW -- the second with fewer segments and other data, so that
whatever the first left in the shared staging array would show -- and that a batch over the limit is refused with a
message naming the limit.  The file sorts last on purpose: under `pytest -x` a failure here hides no other test.  It
builds its own inputs and plan, so it does not care whether it runs alone in a fresh process (then its first call is
also the per-device set-up) or after the other GPU tests.
"""
import ctypes

import numpy as np
import pytest

import bege_synth as synth

pytestmark = pytest.mark.gpu

FS, N, BAND = synth.FS, synth.N_SEG, synth.BAND
SPEC_REL_L2 = 1e-6     # same bar as test_segment_spectrum_matches_oracle


@pytest.fixture(scope="module")
def bege():
    from paper_1708_01609_b200 import bege as m, build
    build.build_library()
    return m


def _segments(seed, S):
    rng = np.random.default_rng(seed)
    return (rng.standard_normal((S, N)) + 1j * rng.standard_normal((S, N))).astype(np.complex64)


def _plan_spectra(bege, x):
    """The existing path: a plan (which allocates) transforms the segments; spectra come back in natural order."""
    with bege.Plan(N, FS, BAND) as plan:
        plan.segment_load(x)
        return np.stack([plan.debug_segment_spectrum(m) for m in range(x.shape[0])])


def _assert_same(Xs, Xp):
    for m in range(Xp.shape[0]):
        a, b = Xs[m].astype(np.complex128), Xp[m].astype(np.complex128)
        assert np.linalg.norm(a - b) / np.linalg.norm(b) < SPEC_REL_L2, m
        assert np.array_equal(a == 0, b == 0), m          # exactly the same bins are masked
    assert np.count_nonzero(Xp) > 0


def test_static_spectrum_matches_plan_path_on_two_calls_in_a_row(bege):
    import torch

    xa, xb = _segments(101, 3), _segments(202, 2)
    dxa, dxb = torch.from_numpy(xa).cuda(), torch.from_numpy(xb).cuda()
    outa, outb = torch.empty_like(dxa), torch.empty_like(dxb)   # the caller owns inputs and outputs
    # two calls back to back on one stream, nothing read in between
    assert bege.segment_spectrum_static(dxa, FS, BAND, out=outa) is outa
    bege.segment_spectrum_static(dxb, FS, BAND, out=outb)
    torch.cuda.synchronize()
    Xa, Xb = outa.cpu().numpy(), outb.cpu().numpy()
    _assert_same(Xa, _plan_spectra(bege, xa))
    _assert_same(Xb, _plan_spectra(bege, xb))
    # and once more at the full size the staging array allows, after the plans above have come and gone
    xc = _segments(303, bege.STATIC_MAX_SEGMENTS)
    Xc = bege.segment_spectrum_static(torch.from_numpy(xc).cuda(), FS, BAND)
    torch.cuda.synchronize()
    _assert_same(Xc.cpu().numpy(), _plan_spectra(bege, xc))


def test_static_spectrum_refuses_more_than_the_limit(bege):
    import torch

    S = bege.STATIC_MAX_SEGMENTS + 1
    x = torch.zeros((S, N), dtype=torch.complex64, device="cuda")
    out = torch.full_like(x, 7.0)
    with pytest.raises(bege.BegeError) as ei:
        bege.segment_spectrum_static(x, FS, BAND, out=out)
    assert ei.value.status == bege.EINVAL
    assert "BEGE_STATIC_MAX_SEGMENTS = 4" in str(ei.value)
    torch.cuda.synchronize()
    assert bool((out == 7.0).all())                       # refused before anything was launched
    # a host pointer is refused too, with a message (raw C ABI: the binding only ever passes device tensors)
    h = np.zeros(N, dtype=np.complex64)
    err = ctypes.create_string_buffer(256)
    rc = bege.load_library().bege_segment_spectrum_static(0, None, FS, BAND[0], BAND[1], h.ctypes.data, 1,
                                                          out.data_ptr(), err, len(err))
    assert rc == bege.EINVAL and b"device memory" in err.value
