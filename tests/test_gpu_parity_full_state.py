"""Parity at the state the search kernel is in at full size.  `-m gpu`.

The tests of test_gpu_parity.py pass small banks through every variant of `k_search`; with 9 CTA groups on a B200 their
groups see fewer than 16 (template, segment) items, so the 16-deep ring between the two passes never wraps, no pass-1
warp ever waits for a slot (done2), and in batched calls the stationary template tile is never replaced after a wrap.
Here every variant gets >= 40 items per group: the batched 14-row-block kernel with template changes after the wrap,
the dual-stream variant, the max projection; configs[3] is checked at bench size against a sampled oracle; and a plan
runs on a caller's non-default stream and on a stream of its own.  Bars as in test_gpu_parity.py (north_star)."""
import numpy as np
import pytest

import bege_synth as synth
from test_gpu_parity import FS, N, BAND, TAU, REL_L2, GUARD, SIGMA_RTOL, check_tail_sets, check_maxproj, rel_l2

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def bo():
    from oracle import bege_oracle
    return bege_oracle


@pytest.fixture(scope="module")
def bege():
    from paper_1708_01609_b200 import bege as m, build
    build.build_library()
    return m


def test_batched_search_wraps_ring_and_changes_template(bo, bege):
    """T = 45, S = 12: each of the 9 groups runs 5 templates x 12 segments = 60 items -- the ring wraps three times and
    the stationary template tile is replaced four times, at items that differ between the two teams of a pass."""
    S = 12
    xs = np.stack([synth.noise_segment(700 + s) for s in range(S)])
    x2, n0 = synth.inject_chirp(xs[7].real.astype(np.float64), 900.0, -80.0, 6.0, 9.0)
    xs[7] = synth.as_segment(x2)
    f0, fd = synth.bank_grid(9, 5, 500.0, 1800.0, -200.0, 200.0)
    f0[22], fd[22] = 900.0, -80.0                               # template 22 is the injected chirp
    assert f0.size == 45
    Xs = np.stack([bo.segment_spectrum(x, FS, *BAND) for x in xs])
    k = 3.0
    lo_tails, _, sigma_o, _ = bo.search(Xs, f0, fd, TAU, FS, k - 1e-3)
    with bege.Plan(N, FS, BAND) as plan:
        plan.bank_generate(f0, fd, TAU)
        plan.segment_load(xs)
        tails, n = plan.search(k)
        must, _ = check_tail_sets(tails, n, lo_tails, k)
        assert must > 3000
        sg = plan.get_sigma()
        assert sg.shape == (45, S)
        assert np.max(np.abs(sg - sigma_o) / sigma_o) <= SIGMA_RTOL
        best = tails[np.argmax(tails["snr"])]
        assert best["template_id"] == 22 and best["lag"] // N == 7 and abs(int(best["lag"]) % N - n0) <= 2
        for (j, m) in ((0, 0), (22, 7), (36, 11), (44, 5), (17, 3)):       # templates 2nd .. 5th of their groups too
            z, s = bo.correlate(Xs[m], bo.template(f0[j], fd[j], TAU, FS, N))
            zg, sgj = plan.debug_correlate(j, m)
            assert rel_l2(zg.astype(np.complex128), z) <= REL_L2, (j, m)
            assert abs(sgj - s) / s <= SIGMA_RTOL, (j, m)


def _dual_inputs(n_seg):
    xs, n0 = [], None
    for m in range(n_seg):
        h1 = synth.band_limit(synth.white_noise(800 + 2 * m))
        l1 = synth.band_limit(synth.white_noise(801 + 2 * m))
        if m == n_seg - 1:
            l1, n0 = synth.inject_chirp(l1, 1234.0, 77.0, 9.0, 11.0)
        xs.append((h1 + 1j * l1).astype(np.complex64))
    return np.stack(xs), n0


@pytest.mark.parametrize("n_seg", [1, 2])
def test_dual_stream_search_wraps_ring(bo, bege, n_seg):
    """360 real templates: 40 items per group and segment in k_search<DUAL> (the ring wraps twice per launch)."""
    xs, n0 = _dual_inputs(n_seg)
    Xs = np.stack([bo.segment_spectrum(x, FS, *BAND) for x in xs])
    f0, fd = synth.bank_grid(20, 18, 400.0, 1900.0, -300.0, 300.0)
    f0[201], fd[201] = 1234.0, 77.0
    assert f0.size == 360
    k = 3.3
    o1, oi1, o2, oi2, sig_o = bo.search_dual(Xs, f0, fd, TAU, FS, k - 1e-3)
    with bege.Plan(N, FS, BAND) as plan:
        plan.bank_generate_real(f0, fd, TAU)
        plan.segment_load(xs)
        g1, gi1, g2, gi2, n_sim, n_coi = plan.search_dual(k, 200.0)
        s1, s2 = plan.get_sigma_dual()
    assert np.max(np.abs(s1 - sig_o[:, :, 0]) / sig_o[:, :, 0]) <= SIGMA_RTOL
    assert np.max(np.abs(s2 - sig_o[:, :, 1]) / sig_o[:, :, 1]) <= SIGMA_RTOL
    none = np.iinfo(np.uint32).max
    n_checked = 0
    for g, gi, o, oi, stream in ((g1, gi1, o1, oi1, 0), (g2, gi2, o2, oi2, 1)):
        assert np.all((g == 0) == (gi == none))
        must, may = o > k + GUARD, o > k - GUARD
        assert not np.any(must & (g == 0)), "oracle offsets missing on the GPU"
        assert not np.any((g > 0) & ~may), "GPU offsets the oracle does not have"
        both = must & (g > 0)
        assert np.max(np.abs(g[both] - o[both]) / o[both]) < 2e-5
        diff = both & (gi != oi)                                # near-ties: the other template must be as good
        assert diff.sum() < 50
        for m, n in zip(*np.nonzero(diff)):
            z, t1, t2 = bo.correlate_dual(Xs[m], bo.template_real(f0[gi[m, n]], fd[gi[m, n]], TAU, FS, N))
            val = abs(z[n].real) / t1 if stream == 0 else abs(z[n].imag) / t2
            assert abs(val - o[m, n]) / o[m, n] < 2e-6
        n_checked += int(both.sum())
    assert n_checked > 20000 * n_seg
    peak = np.unravel_index(np.argmax(g2), g2.shape)
    assert peak[0] == n_seg - 1 and gi2[peak] == 201 and abs(int(peak[1]) - n0) <= 8 and g2[peak] > 8.0
    sim = (gi1 != none) & (gi2 != none)
    assert n_sim == int(sim.sum())
    assert n_coi == int(np.sum(np.abs(f0[gi1[sim]] - f0[gi2[sim]]) < 200.0))


def test_max_projection_wraps_ring(bo, bege):
    """360 templates x 2 segments: 80 items per group on the way to the projection."""
    xs = np.stack([synth.noise_segment(900), synth.noise_segment(901)])
    Xs = np.stack([bo.segment_spectrum(x, FS, *BAND) for x in xs])
    f0, fd = synth.bank_grid(20, 18, 400.0, 1900.0, -300.0, 300.0)
    k = 2.8
    snr_o, id_o = bo.search_maxproj(Xs, f0, fd, TAU, FS, k - 1e-3)
    with bege.Plan(N, FS, BAND) as plan:
        plan.bank_generate(f0, fd, TAU)
        plan.segment_load(xs)
        snr_g, id_g, nh = plan.search_maxproj(k)
    assert nh == int((snr_g > 0).sum())
    n_both, n_diff = check_maxproj(bo, snr_g, id_g, snr_o, id_o, Xs, f0, fd, k)
    assert n_both > 10000 and n_diff < 50


def test_config3_full_size_sampled(bo, bege):
    """configs[3] as bench.py runs it (64 segments x 65,536 templates, k = 5, one batched search of 4.2 M pairs): record
    fields, the count's partition over segments and templates, and all records of 24 sampled templates x 4 segments
    (two of them carrying an injection) against the oracle."""
    w = synth.config3()
    T, S = w.n_templates, w.x.shape[0]
    assert (T, S) == (1 << 16, 64)
    k = w.k_sigma
    inj = sorted(w.meta["injections"])
    with bege.Plan(N, FS, BAND) as plan:
        plan.bank_generate(w.f0, w.fdot, TAU)
        plan.segment_load(w.x)
        tails, n = plan.search(k, cap=1 << 22)
        sg = plan.get_sigma()
    assert n == tails.size and 50_000 < n < 1 << 22
    assert int(tails["template_id"].max()) < T and int(tails["lag"].max()) < S * N
    assert float(tails["snr"].min()) >= k * (1 - 1e-6)
    key = tails["template_id"].astype(np.uint64) << np.uint64(32) | tails["lag"].astype(np.uint64)
    assert np.unique(key).size == n
    seg_of = tails["lag"] // N
    per_seg = np.bincount(seg_of, minlength=S)
    assert per_seg.sum() == n and per_seg[inj].sum() > 0.9 * n                  # the injections carry the tails
    top = tails[np.argmax(tails["snr"])]
    segs = np.array(sorted({int(top["lag"]) // N, next(m for m in inj if m != int(top["lag"]) // N), 0, S - 1}))
    extra = [int(tm["template_id"][np.argmax(tm["snr"])]) for tm in (tails[seg_of == m] for m in segs) if tm.size]
    sample = np.unique(np.concatenate([np.arange(11, T, T // 22)[:22], extra]).astype(np.int64))
    Xs = np.stack([bo.segment_spectrum(w.x[m], FS, *BAND) for m in segs])
    lo_tails, _, sigma_o, _ = bo.search(Xs, w.f0[sample], w.fdot[sample], TAU, FS, k - 1e-3, cap=1 << 22)
    pick = np.isin(tails["template_id"], sample) & np.isin(seg_of, segs)
    sel = tails[pick].copy()
    sel["template_id"] = np.searchsorted(sample, sel["template_id"]).astype(np.uint32)
    sel["lag"] = (np.searchsorted(segs, sel["lag"] // N) * N + sel["lag"] % N).astype(np.uint32)
    must, _ = check_tail_sets(sel, sel.size, lo_tails, k)
    assert must >= 3
    assert np.max(np.abs(sg[np.ix_(sample, segs)] - sigma_o) / sigma_o) <= SIGMA_RTOL


@pytest.mark.parametrize("which", ["user_stream", "own_stream"])
def test_plan_on_other_streams(bo, bege, which):
    """bege_plan_create with a caller's non-default stream, and with cuda_stream = NULL (the plan makes its own):
    a device-resident input produced on that stream, a search, destroy."""
    import torch

    w = synth.config0()
    ids = np.arange(0, 256, 8)
    X = bo.segment_spectrum(w.x[0], FS, *BAND)
    k = 3.0
    lo_tails, _, sigma_o, _ = bo.search(X[None, :], w.f0[ids], w.fdot[ids], TAU, FS, k - 1e-3)
    user = torch.cuda.Stream()
    assert user.cuda_stream != 0
    plan = bege.Plan(N, FS, BAND, stream=user.cuda_stream if which == "user_stream" else "own")
    try:
        plan.bank_generate(w.f0[ids], w.fdot[ids], TAU)
        if which == "user_stream":
            with torch.cuda.stream(user):                       # input made on the plan's stream, no sync in between
                xd = torch.from_numpy(w.x).pin_memory().to("cuda", non_blocking=True) * 1.0
                plan.segment_load(xd)
        else:
            plan.segment_load(w.x)
        tails, n = plan.search(k)
        check_tail_sets(tails, n, lo_tails, k)
        sg = plan.get_sigma()[:, 0]
        assert np.max(np.abs(sg - sigma_o[:, 0]) / sigma_o[:, 0]) <= SIGMA_RTOL
        snr_g, id_g, nh = plan.search_maxproj(k)
        assert nh == int((snr_g > 0).sum()) > 0
    finally:
        plan.close()
    torch.cuda.synchronize()
    # the caller's stream is left usable and without the plan's L2 window
    with torch.cuda.stream(user):
        y = torch.ones(1 << 20, device="cuda").sum()
    assert float(y) == float(1 << 20)
