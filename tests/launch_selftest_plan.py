"""Stand-in plan for `bench.py --selftest-launch launch_selftest_plan:LaunchSelfTestPlan` (tests/test_host_logic.py).
Test scaffolding: it fabricates three fixed records per chunk so that bench.py's multi-rank launch path can be run on a
box without GPUs.  Lives under tests/ so that nothing in the benchmark program itself makes up results."""
import time

import numpy as np


class LaunchSelfTestPlan:
    """NOT a search.  `--selftest-launch` exercises bench.py's own multi-rank plumbing (spawn, rendezvous, barrier,
    max-over-ranks timing, gather of tail records on rank 0) on a box without GPUs; it stands in for bege.Plan with
    the same method names, produces a few fixed records per chunk and never runs under any other flag.  The JSON
    line of such a run carries "selftest_launch": true and value null."""

    def __init__(self, rank):
        self.rank, self.n, self.launches = rank, 0, 0

    def stats(self):
        return {"hbm_bytes_per_template": 14 * 32768, "kernel_launches": self.launches, "fused_kernel_ms": 1.0,
                "fused_kernel_launches": 1}

    def alloc_workspace(self, *a):
        return 0

    def bank_generate(self, f0, fdot, tau):
        self.n = len(f0)

    def segment_load(self, x):
        self.launches += 2

    def search(self, k, cap=0, copy=True):
        from paper_1708_01609_b200 import bege
        self.launches += 1
        t = np.zeros(3, dtype=bege.TAIL_DTYPE)
        t["template_id"] = [0, self.n // 2, self.n - 1]
        t["lag"] = 100 + self.rank
        t["snr"] = 7.0
        time.sleep(0.01)
        return t, 3

    def set_profiling(self, on): pass
    def reset_stats(self): pass
    def close(self): pass
