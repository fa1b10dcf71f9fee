"""CPU-only checks of the host logic: the C-ABI library loads and exports every symbol include/bege.h
declares (no compute calls without a GPU), argument validation that needs no device, bank sharding, and the
world_size-2 gather of tail records over gloo."""
import ctypes
import os
import re
import socket
import sys

import numpy as np
import pytest

from paper_1708_01609_b200 import bege, shard, build
import bege_synth as synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build_library()
    return bege.load_library()


def test_library_exports_every_declared_symbol(lib):
    header = open(os.path.join(ROOT, "include", "bege.h")).read()
    declared = set(re.findall(r"\b(bege_[a-z_]+)\s*\(", header))
    assert declared == set(bege.SYMBOLS)
    for name in declared:
        assert hasattr(lib, name), name
    assert lib.bege_version().decode().startswith("bege")
    # the probe library has its own header; nothing of it is in the product ABI
    probe_header = open(os.path.join(ROOT, "include", "bege_probe.h")).read()
    probe_declared = set(re.findall(r"\b(bege_[a-z_]+)\s*\(", probe_header))
    assert probe_declared == set(bege.PROBE_SYMBOLS) and not (probe_declared & declared)
    probe = bege.load_probe_library()
    for name in probe_declared:
        assert hasattr(probe, name) and not hasattr(lib, name), name


def test_tail_record_is_12_bytes(lib):
    header = open(os.path.join(ROOT, "include", "bege.h")).read()
    assert "uint32_t template_id" in header and "uint32_t lag" in header and "float    snr" in header
    assert bege.TAIL_DTYPE.itemsize == 12 and bege.TAIL_DTYPE.names == ("template_id", "lag", "snr")


def test_argument_validation_without_device(lib):
    h = ctypes.c_void_p()
    assert lib.bege_plan_create(None, 65536, 4096.0, 350.0, 2000.0, 0, None) == bege.EINVAL
    assert lib.bege_plan_create(ctypes.byref(h), 1024, 4096.0, 350.0, 2000.0, 0, None) == bege.EINVAL
    assert lib.bege_plan_create(ctypes.byref(h), 65536, 4096.0, 0.0, 2000.0, 0, None) == bege.EINVAL
    assert lib.bege_plan_create(ctypes.byref(h), 65536, 4096.0, 2000.0, 350.0, 0, None) == bege.EINVAL
    assert lib.bege_plan_create(ctypes.byref(h), 65536, 4096.0, 350.0, 2048.0, 0, None) == bege.EINVAL
    import torch
    if not torch.cuda.is_available():
        # valid arguments, but no device: fails loudly, no CPU fallback
        assert lib.bege_plan_create(ctypes.byref(h), 65536, 4096.0, 350.0, 2000.0, 0, None) == bege.ECUDA
        with pytest.raises(RuntimeError):
            bege.Plan()
    assert lib.bege_search(None, 5.0, None, 0, None) == bege.EINVAL
    assert lib.bege_last_error(None) == b"null plan"
    lib.bege_plan_destroy(None)


def test_product_code_never_touches_the_oracle():
    pkg = os.path.join(ROOT, "paper_1708_01609_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", src, re.M), f
                assert "bege_oracle" not in src and "libbege_oracle" not in src and "bo_" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_1708_01609_b200" not in src and "from paper_1708_01609_b200" not in src


# ------------------------------------------------------------------------------- sharding
@pytest.mark.parametrize("T,world", [(0, 1), (1, 4), (10, 3), (1 << 20, 8), (65537, 2)])
def test_shard_ranges_partition_the_bank(T, world):
    rs = [shard.shard_range(T, r, world) for r in range(world)]
    assert rs[0][0] == 0 and rs[-1][1] == T
    assert all(a[1] == b[0] for a, b in zip(rs, rs[1:]))
    sizes = [hi - lo for lo, hi in rs]
    assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard.shard_range(T, world, world)


def test_chunk_ranges():
    assert shard.chunk_ranges(5, 5, 3) == []
    assert shard.chunk_ranges(0, 10, 4) == [(0, 4), (4, 8), (8, 10)]
    assert shard.chunk_ranges(7, 9, 100) == [(7, 9)]
    with pytest.raises(ValueError):
        shard.chunk_ranges(0, 1, 0)


def test_bank_grid_flattening():
    f0, fd = synth.bank_grid(3, 2, 100.0, 300.0, -1.0, 1.0)
    assert np.array_equal(f0, [100, 100, 200, 200, 300, 300]) and np.array_equal(fd, [-1, 1, -1, 1, -1, 1])
    f0, fd = synth.config2_bank()
    assert f0.size == 1 << 20 and f0[1023] == 350.0 and f0[1024] > 350.0 and fd[1023] == 400.0


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    import torch.distributed as dist
    from oracle import bege_oracle as bo
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    try:
        n, fs, band, tau, k = 2048, 1024.0, (50.0, 450.0), 0.25, 2.0
        X = bo.segment_spectrum(synth.white_noise(9, n), fs, *band)[None, :]
        f0, fd = synth.bank_grid(5, 3, 100.0, 300.0, -80.0, 80.0)        # 15 templates over 2 ranks: 8 + 7
        lo, hi = shard.shard_range(f0.size, rank, world)
        # the per-rank search stands in for bege_search (no GPU here): the oracle, on this rank's slice only
        t, cnt, _, _ = bo.search(X, f0[lo:hi], fd[lo:hi], tau, fs, k)
        local = np.zeros(t.size, dtype=bege.TAIL_DTYPE)
        local["template_id"], local["lag"], local["snr"] = t["template_id"], t["lag"], t["snr"]
        if rank == 1:
            local = local[:0] if os.environ.get("BEGE_TEST_EMPTY_RANK") else local
        allt = shard.gather_tails(shard.globalize(local, lo))
        if rank == 0:
            full, nfull, _, _ = bo.search(X, f0, fd, tau, fs, k)
            allt = allt[np.lexsort((allt["lag"], allt["template_id"]))]
            ok = (allt.size == nfull and np.array_equal(allt["template_id"], full["template_id"])
                  and np.array_equal(allt["lag"], full["lag"])
                  and np.allclose(allt["snr"], full["snr"], rtol=1e-6))
            q.put(bool(ok))
        else:
            assert allt is None
    finally:
        dist.destroy_process_group()


def test_two_rank_bank_sharding_over_gloo():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    assert q.get(timeout=5) is True


def _gather_worker(rank, world, port, q):
    """gather_tails alone: rank 1 holds 10^6 records, rank 0 three, rank 2 none -- exact sizes, rank order, every byte."""
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        n = (3, 1_000_000, 0)[rank]
        t = np.zeros(n, dtype=bege.TAIL_DTYPE)
        t["template_id"] = np.arange(n, dtype=np.uint32) * np.uint32(rank + 1)
        t["lag"] = np.arange(n, dtype=np.uint32)[::-1]
        t["snr"] = 5.0 + rank
        out = shard.gather_tails(t)
        out2 = shard.gather_tails(t[: n // 2])               # a second call reuses the group
        if rank == 0:
            ok = (out.size == 1_000_003 and np.array_equal(out["template_id"][:3], [0, 1, 2])
                  and np.array_equal(out["template_id"][3:], np.arange(1_000_000, dtype=np.uint32) * np.uint32(2))
                  and np.array_equal(out["lag"][3:], np.arange(1_000_000, dtype=np.uint32)[::-1])
                  and np.all(out["snr"][:3] == 5.0) and np.all(out["snr"][3:] == 6.0) and out2.size == 1 + 500_000)
            q.put(bool(ok))
        else:
            assert out is None and out2 is None
    finally:
        dist.destroy_process_group()


def test_gather_tails_exact_sizes_three_ranks():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_gather_worker, args=(r, 3, port, q)) for r in range(3)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    assert q.get(timeout=5) is True


def test_bench_starts_its_own_ranks_and_gathers_tails():
    """`python bench.py --gpus 2` with no torchrun environment must start two ranks by itself, rendezvous on
    127.0.0.1, time with max-over-ranks and gather the tail records on rank 0.  No GPU here: --selftest-launch
    swaps the plan for a stand-in that produces three fixed records per chunk (gloo backend); everything else is
    bench.py's real launch path."""
    import json
    import subprocess
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    env["PYTHONPATH"] = os.path.join(ROOT, "tests") + os.pathsep + env.get("PYTHONPATH", "")   # the stand-in plan lives here
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "1", "--warmup", "0",
                          "--selftest-launch", "launch_selftest_plan:LaunchSelfTestPlan", "--templates", "1000",
                          "--chunk", "400"],
                         capture_output=True, text=True, timeout=300, env=env)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, out.stdout                      # rank 0 alone prints
    line = json.loads(lines[0])
    assert line["selftest_launch"] is True and line["value"] is None
    assert line["n_gpus"] == 2
    assert line["gathered_tails"] == 2 * 3 * 3              # 2 ranks x 3 chunks x 3 records
    assert line["gathered_ids_ok"] is True                  # ids were made global: both ranks' shards are present
