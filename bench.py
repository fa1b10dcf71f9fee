#!/usr/bin/env python
"""bench.py -- template correlations/s at N = 2^16 (C2C fp32) on B200, BASELINE.json configs[2].

One "step" = one pass of the whole 2^20-template bank (1024 x 1024 grid, 350-2000 Hz x +-400 Hz/s)
against one 16 s segment of band-limited Gaussian noise (seed 2), k = 6.  The bank (2^20 x 448 KiB of
in-band spectra) does not fit HBM, so it is processed in chunks: chunk generation (bege_bank_generate) is
untimed, as BASELINE.json configs[2] states ("template spectra are precomputed once, and the search is
timed separately from generation") but its time is reported beside the number; the timed region of a step
is the sum over chunks of bege_search, each bracketed by a device synchronize and CUDA events on the
plan's stream.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference|cufft] [--templates T]

The same JSON line also carries two more workloads of BASELINE.json: `segment_batched`
(configs[3]: 64 segments x 2^16 templates) and `tail_heavy` (configs[4]: 2^18 templates at k = 3, tens of
millions of records crossing PCIe while the search goes on).

--gpus N > 1 without a torchrun environment: bench.py starts N ranks itself (torch.distributed.run,
127.0.0.1).  Every rank searches its own 2^20-template shard of an N-times finer fdot grid (weak scaling,
no data-path collective); after the timed region the tail records of all ranks are gathered on rank 0
(shard.gather_tails).  --impl reference times the fp64 CPU oracle (oracle/) on the host cores, on a
bounded sample.  --impl cufft times the same steps built from library kernels (torch + cuFFT): a
reference point for context only.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import bege_synth as synth  # noqa: E402

METRIC = "template correlations/sec at N=2^16 C2C fp32 on 1 B200; % of FFT roofline"   # BASELINE.json, verbatim
UNIT = "correlations/s"
FFT_FLOP = 5.0 * 65536 * 16                       # PAPER.md:134 eq.(10): 5 N log2 N
ALG_BYTES_PER_CORR = 52802 * 8                    # two-sided in-band template spectrum, S = 1
# dram__bytes_read.sum + dram__bytes_write.sum of k_search per correlation: an OFFLINE constant, taken from the
# `ncu --set full` capture of the kernel as committed (profiles/r3_search_kernel.md: 36,864-template launch,
# 16.913 GB read + 0.0245 GB written); it does not follow later kernel changes by itself.
NCU_DRAM_BYTES_PER_CORR = (16.913445e9 + 0.02447232e9) / 36864
NCU_SOURCE = "profiles/r3_search_kernel.md"
FP32_PEAK = 148 * 128 * 2 * 1.965e9               # SMs x fp32 lanes x 2 flop x max SM clock
FMA_PIPE_CEILING = 8.6e6                          # what the FMA pipe allows for k_search's instruction mix
# ncu figures of k_search from the same capture (north_star: "ncu dram throughput and FP32 pipe utilisation shown"):
# OFFLINE constants like the traffic above, percent of peak sustained over the kernel's duration
NCU_OFFLINE = {"source": NCU_SOURCE, "pipe_fmaheavy_pct": 53.7, "issue_slots_pct": 57.5, "lsu_wavefronts_pct": 66.9,
               "dram_throughput_gbs": (16.913445e9 + 0.02447232e9) / 7.605216e-3 * 1e-9, "warps_active_pct": 50.0,
               "note": "measured under ncu (serialised, cold cache) on the build named in source; not re-measured in this run"}


# ------------------------------------------------------------------------------------------ clocks
class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap,clocks.mem")

    def __init__(self, index: int):
        self.index, self.rows, self.proc, self.thr = index, [], None, None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100",
                 "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            return
        self.thr = threading.Thread(target=self._pump, daemon=True)
        self.thr.start()

    def _pump(self):
        for line in self.proc.stdout:
            self.rows.append((time.perf_counter(), line.strip()))

    def stop(self):
        if self.proc:
            self.proc.terminate()
            try:
                self.proc.wait(2)
            except Exception:
                self.proc.kill()

    def summary(self, windows):
        sm, smax, reasons, power, mem = [], 0.0, set(), 0.0, []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ts, line in self.rows:
            if not any(a <= ts <= b for a, b in windows):
                continue
            f = [x.strip() for x in line.split(",")]
            try:
                sm.append(float(f[0])); smax = max(smax, float(f[1])); power = max(power, float(f[2]))
            except (ValueError, IndexError):
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
            try:
                mem.append(float(f[7]))
            except (ValueError, IndexError):
                pass
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": smax or None,
                "reasons": sorted(reasons), "samples": len(sm), "power_w_max": power or None,
                "mem_mhz": float(np.median(mem)) if mem else None}


# ------------------------------------------------------------------------------------------ oracle arm
def oracle_rate(f0, fdot, x, k_sigma, sample: int):
    """Correlations/s of the fp64 CPU oracle, as it stands, on a strided sample of the bank."""
    from oracle import bege_oracle as bo
    X = np.stack([bo.segment_spectrum(xm, synth.FS, *synth.BAND) for xm in x])
    ids = np.linspace(0, f0.size - 1, sample).astype(np.int64)
    t0 = time.perf_counter()
    _, n, _, used = bo.search(X, f0[ids], fdot[ids], synth.TAU, synth.FS, k_sigma, cap=1 << 16)
    dt = time.perf_counter() - t0
    return sample * x.shape[0] / dt, used, dt, n


def run_reference(args, rank):
    if rank != 0:
        return
    f0, fdot = synth.config2_bank()
    x = synth.noise_segment(2)[None, :]
    sample = args.ref_sample
    for _ in range(args.warmup):
        oracle_rate(f0, fdot, x, 6.0, max(16, sample // 16))
    t, used = 0.0, 0
    for _ in range(args.steps):
        _, used, dt, _ = oracle_rate(f0, fdot, x, 6.0, sample)
        t += dt
    value = sample * args.steps / t
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "configs[2]: 2^20 templates (1024x1024) x 1 segment, N=2^16, k=6",
                   "sample": f"{sample} templates strided over the bank per step"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": used, "kind": "oracle",
                         "sample": f"{sample} templates strided over the 2^20 bank x 1 segment per step"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gflops_equiv": value * FFT_FLOP * 1e-9,
    }
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------ library reference point
def run_cufft(args, rank, local_rank):
    """Context only (north_star: "cuFFT used only as a timed reference point, not as the product"): the same steps
    with library kernels -- torch elementwise product, torch reductions, torch.fft.ifft (cuFFT batched C2C, N = 2^16),
    torch compare + count -- on a resident batch of template spectra produced by the product's own bank generation."""
    if rank != 0:
        return
    import torch
    from paper_1708_01609_b200 import bege
    dev = torch.device("cuda", local_rank)
    torch.cuda.set_device(dev)
    Tb = args.cufft_batch
    f0, fdot = synth.config2_bank()
    ids = np.linspace(0, f0.size - 1, Tb).astype(np.int64)
    x = synth.noise_segment(2)[None, :]
    with bege.Plan(synth.N_SEG, synth.FS, synth.BAND, device=local_rank) as plan:
        plan.bank_generate(f0[ids], fdot[ids], synth.TAU)
        plan.segment_load(x)
        H = torch.from_numpy(np.stack([plan.debug_template_spectrum(j) for j in range(Tb)])).to(dev)
        X = torch.from_numpy(plan.debug_segment_spectrum(0)).to(dev)
    k2 = 36.0
    def step():
        R = torch.conj(H) * X                                        # a3
        s2 = (R.real * R.real + R.imag * R.imag).sum(dim=1) / float(synth.N_SEG) ** 2     # a4
        z = torch.fft.ifft(R, dim=1)                                 # a5 (1/N inside)
        hit = (z.real * z.real + z.imag * z.imag) > (k2 * s2)[:, None]                   # a6
        return int(hit.sum().item())                                 # a7: count only (records not materialised)
    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize(dev)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    n = 0
    for _ in range(args.steps):
        n = step()
    e1.record()
    torch.cuda.synchronize(dev)
    ms = e0.elapsed_time(e1) / args.steps
    value = Tb / (ms * 1e-3)
    # the inverse FFT alone (the paper normalises its 65 % efficiency to the library FFT alone)
    R = torch.conj(H) * X
    torch.fft.ifft(R, dim=1)
    torch.cuda.synchronize(dev)
    e0.record()
    for _ in range(args.steps):
        torch.fft.ifft(R, dim=1)
    e1.record()
    torch.cuda.synchronize(dev)
    fft_only = Tb / (e0.elapsed_time(e1) / args.steps * 1e-3)
    print(json.dumps({"impl": "cufft", "fft_only_per_s": fft_only, "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": 1, "steps": args.steps,
                      "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "dtype": "f32",
                      "data": "synthetic", "config": {"workload": f"{Tb} templates of configs[2] x 1 segment, resident full "
                      "spectra (512 KiB each), torch elementwise + torch.fft.ifft (cuFFT) + torch reductions", "tails": n},
                      "gflops_equiv": value * FFT_FLOP * 1e-9,
                      "note": "library reference point for context; not the product, not the driver's reference arm"}),
          flush=True)


# ------------------------------------------------------------------------------------------ overlap-save bake-off
def run_ovs_probe(args, rank, local_rank):
    """the overlap-save variant's fused kernel (six 16384-point block correlations per template,
    one CTA per SM, everything in shared memory), timed on synthetic resident spectra.  A measurement for the keep-or-kill
    decision in DESIGN.md, not the product; sigma and the compaction of records are not in it (both small)."""
    if rank != 0:
        return
    from paper_1708_01609_b200 import bege
    T = args.ovs_templates
    ms, hits, _ = bege.ovs_probe(T, 6, reps=max(args.steps, 1), device=local_rank)
    value = T / (ms * 1e-3)
    print(json.dumps({"impl": "ovs_probe", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": 1, "steps": args.steps,
                      "ms_per_step": ms, "higher_is_better": True, "dtype": "f32", "data": "synthetic",
                      "config": {"workload": f"{T} resident 16384-point template spectra (128 KiB each) x 6 overlapping blocks "
                                 "of one segment; multiply + inverse transform in shared memory + threshold per block"},
                      "gflops_equiv": value * FFT_FLOP * 1e-9, "frac_of_fp32_bound": value * FFT_FLOP / FP32_PEAK,
                      "bank_bytes_2p20_templates": (1 << 20) * 16384 * 8,
                      "note": "bake-off probe (SURVEY 8(f)4); correlations/s = templates/s, six blocks each"}), flush=True)


# ------------------------------------------------------------------------------------------ our arm
def _extra_workloads(args, dev, local_rank):
    """configs[3] (segment-batched) and configs[4] (tail-heavy), measured like the headline: CUDA events around
    bege_search, wall clock around segment_load + search for the end-to-end figure.  Rank 0, N = 1 only."""
    import torch
    from paper_1708_01609_b200 import bege
    out = {}

    def timed(plan, x_host, k, cap, reps):
        rates, e2e, n = [], [], 0
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        for i in range(reps + 1):
            torch.cuda.synchronize(dev)
            t0 = time.perf_counter()
            plan.segment_load(x_host)
            e0.record()
            _t, n = plan.search(k, cap=cap, copy=False)
            e1.record()
            torch.cuda.synchronize(dev)
            t1 = time.perf_counter()
            if i:                                                    # first pass warms up
                rates.append(plan.n_templates * plan.n_segments / (e0.elapsed_time(e1) * 1e-3))
                e2e.append(plan.n_templates * plan.n_segments / (t1 - t0))
        return float(np.median(rates)), float(np.median(e2e)), int(n)

    def kernel_rate(plan, k, cap):
        plan.set_profiling(True); plan.reset_stats()
        plan.search(k, cap=cap, copy=False)
        st = plan.stats(); plan.set_profiling(False)
        return plan.n_templates * plan.n_segments / (st["fused_kernel_ms"] * 1e-3)

    # ---- configs[3]: 64 segments x 2^16 templates (the paper's M^2 block structure)
    w = synth.config3(args.batched_segments)
    x_host = torch.from_numpy(w.x).pin_memory()
    with bege.Plan(synth.N_SEG, synth.FS, synth.BAND, device=local_rank) as plan:
        t0 = time.perf_counter(); plan.bank_generate(w.f0, w.fdot, synth.TAU); gen_s = time.perf_counter() - t0
        rate, e2e, n = timed(plan, x_host, w.k_sigma, 1 << 20, args.extra_reps)
        krate = kernel_rate(plan, w.k_sigma, 1 << 20)
        # the same bank against ONE of the segments, right after (same clocks, same thermal state): like for like
        plan.segment_load(x_host[:1])
        kernel_rate(plan, w.k_sigma, 1 << 20)
        krate1 = kernel_rate(plan, w.k_sigma, 1 << 20)
    out["segment_batched"] = {
        "kernel_corr_per_s_single_segment_same_bank": krate1,
        "workload": f"configs[3]: {w.x.shape[0]} segments x {w.n_templates} templates, k = {w.k_sigma}",
        "S": int(w.x.shape[0]), "T": int(w.n_templates), "corr_per_s": rate, "kernel_corr_per_s": krate,
        "frac": rate * FFT_FLOP / FP32_PEAK, "e2e_corr_per_s": e2e, "n_tails": n,
        "h2d_bytes": int(w.x.size * 8), "d2h_bytes": 8 + 12 * n, "bank_generate_ms": 1e3 * gen_s}
    del x_host
    torch.cuda.empty_cache()

    # ---- the paper's own output forms on the configs[1]-sized bank: max projection over the
    # bank, and the dual-stream search (x = H1 + i L1, real templates: two detector correlations per complex one)
    f0g, fdg = synth.bank_grid(256, 256, 350.0, 2000.0, -400.0, 400.0)
    xd = (synth.band_limit(synth.white_noise(200)) + 1j * synth.band_limit(synth.white_noise(201))).astype(np.complex64)[None, :]
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

    def timed_call(fn, reps):
        ms = []
        for i in range(reps + 1):
            torch.cuda.synchronize(dev)
            ev0.record(); r = fn(); ev1.record()
            torch.cuda.synchronize(dev)
            if i:
                ms.append(ev0.elapsed_time(ev1))
        return float(np.median(ms)), r

    with bege.Plan(synth.N_SEG, synth.FS, synth.BAND, device=local_rank) as plan:
        plan.bank_generate(f0g, fdg, synth.TAU)
        plan.segment_load(np.ascontiguousarray(xd.real.astype(np.complex64)))
        ms, r = timed_call(lambda: plan.search_maxproj(3.5), args.extra_reps)
        out["max_projection"] = {"workload": "256x256 bank x 1 segment, k = 3.5: per sample offset the largest |z|/sigma over the "
                                 "bank and its template (PAPER.md:166-191)", "T": int(f0g.size), "corr_per_s": f0g.size / (ms * 1e-3),
                                 "n_offsets_hit": int(r[2]), "d2h_bytes": int(synth.N_SEG * 8),
                                 "note": "events around bege_search_maxproj, including the D2H of the two N-entry arrays"}
        plan.bank_generate_real(f0g, fdg, synth.TAU)
        plan.segment_load(xd)
        ms, r = timed_call(lambda: plan.search_dual(5.0, 50.0), args.extra_reps)
        out["dual_stream"] = {"workload": "256x256 bank of REAL templates x 1 segment H1 + i L1, k = 5 (PAPER.md:155, :221)",
                              "T": int(f0g.size), "corr_per_s": f0g.size / (ms * 1e-3),
                              "detector_correlations_per_s": 2 * f0g.size / (ms * 1e-3),
                              "n_simultaneous": int(r[4]), "n_coincident": int(r[5]), "d2h_bytes": int(2 * synth.N_SEG * 8),
                              "note": "events around bege_search_dual, including the D2H of the four N-entry arrays"}

    # ---- configs[4]: 2^18 templates, k = 3: ~6e7 records (0.7 GB) must cross PCIe without holding up the search
    w = synth.config4()
    x_host = torch.from_numpy(w.x).pin_memory()
    cap = args.tail_cap
    with bege.Plan(synth.N_SEG, synth.FS, synth.BAND, device=local_rank) as plan:
        t0 = time.perf_counter(); plan.bank_generate(w.f0, w.fdot, synth.TAU); gen_s = time.perf_counter() - t0
        rate, e2e, n = timed(plan, x_host, w.k_sigma, cap, args.extra_reps)
        krate = kernel_rate(plan, w.k_sigma, cap)
    out["tail_heavy"] = {
        "workload": f"configs[4]: 1 segment + 40 glitches x {w.n_templates} templates, k = {w.k_sigma}",
        "T": int(w.n_templates), "k": w.k_sigma, "corr_per_s": rate, "kernel_corr_per_s": krate,
        "frac": rate * FFT_FLOP / FP32_PEAK, "e2e_corr_per_s": e2e, "n_tails": n, "cap": cap,
        "d2h_bytes": 8 + 12 * min(n, cap), "d2h_note": "records of search slice i are copied on a side stream "
        "while slice i+1 is searched (8 slices); corr_per_s includes those copies", "bank_generate_ms": 1e3 * gen_s}
    return out


def run_ours(args, rank, world, local_rank):
    import torch
    import torch.distributed as dist
    from paper_1708_01609_b200 import bege, shard

    selftest = bool(args.selftest_launch)
    dev = None
    if not selftest:
        torch.cuda.set_device(local_rank)
        dev = torch.device("cuda", local_rank)
    T_total = args.templates
    # weak scaling: rank r owns templates [r*T, (r+1)*T) of an N-times finer fdot grid
    if world == 1 and T_total == 1 << 20:
        f0, fdot = synth.config2_bank()
    else:
        side = int(round(np.sqrt(T_total)))
        if side * side == T_total:
            f0a, fda = synth.bank_grid(side, side * world, 350.0, 2000.0, -400.0, 400.0)
        else:
            f0a, fda = synth.bank_grid(1, T_total * world, 1100.0, 1100.0, -400.0, 400.0)
        f0, fdot = f0a[rank::world].copy(), fda[rank::world].copy()
    x_np = synth.noise_segment(2)[None, :]
    x_host = torch.from_numpy(x_np) if selftest else torch.from_numpy(x_np).pin_memory()
    k_sigma, cap = 6.0, 1 << 16

    if selftest:
        # MODULE:FACTORY of a stand-in plan (tests/launch_selftest_plan.py): nothing in this file fabricates records
        import importlib
        mod, _, factory = args.selftest_launch.partition(":")
        plan = getattr(importlib.import_module(mod), factory)(rank)
        chunk = args.chunk or T_total
    else:
        plan = bege.Plan(synth.N_SEG, synth.FS, synth.BAND, device=local_rank)
        tpl_bytes = plan.stats()["hbm_bytes_per_template"]
        free, _total = torch.cuda.mem_get_info(dev)
        chunk = args.chunk or int(min(T_total, (free * 0.88) // tpl_bytes))
        chunk = max(72, chunk - chunk % 72) if chunk < T_total else T_total
        plan.alloc_workspace(chunk, 1, cap)
    tpl_bytes = plan.stats()["hbm_bytes_per_template"]
    chunks = shard.chunk_ranges(0, T_total, chunk)
    plan.segment_load(x_host)

    sampler = ClockSampler(local_rank)
    ev = None if selftest else [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in chunks]

    def barrier():
        if not selftest:
            torch.cuda.synchronize(dev)
        if world > 1:
            dist.barrier()

    last_tails = []

    def one_step(timed: bool, windows, acc):
        """generation untimed; per chunk: [segment_load from pinned host + search] = e2e, [search] = value."""
        n_tails, search_ms = 0, 0.0
        last_tails.clear()
        for ci, (a, b) in enumerate(chunks):
            g0 = time.perf_counter()
            plan.bank_generate(f0[a:b], fdot[a:b], synth.TAU)              # untimed (configs[2]); synchronous
            g1 = time.perf_counter()
            barrier()
            l0 = plan.stats()["kernel_launches"]
            t0 = time.perf_counter()
            plan.segment_load(x_host)                                        # H2D of the segment + forward FFT
            t1 = time.perf_counter()
            if ev:
                ev[ci][0].record()
            tails, n = plan.search(k_sigma, cap=cap, copy=False)             # D2H of count + records inside
            if ev:
                ev[ci][1].record()
                torch.cuda.synchronize(dev)
            t2 = time.perf_counter()
            n_tails += n
            last_tails.append(shard.globalize(np.array(tails, copy=True), a + rank * T_total))
            ms = ev[ci][0].elapsed_time(ev[ci][1]) if ev else 1e3 * (t2 - t1)
            search_ms += ms
            if timed:
                windows.append((t1, t2))
                acc["search_ms"] += ms
                acc["e2e_s"] += t2 - t0
                acc["gen_s"] += g1 - g0
                acc["load_s"] += t1 - t0
                acc["d2h"] += 8 + 12 * min(n, cap)
                acc["h2d"] += x_host.numel() * 8
                acc["launches"] += plan.stats()["kernel_launches"] - l0
        if timed:
            acc["step_ms"].append(search_ms)
        return n_tails

    sampler.start()
    acc = {"search_ms": 0.0, "e2e_s": 0.0, "gen_s": 0.0, "load_s": 0.0, "d2h": 0, "h2d": 0, "launches": 0, "step_ms": []}
    windows = []
    for _ in range(args.warmup):
        one_step(False, windows, acc)
    barrier()
    plan.reset_stats()
    n_tails = 0
    for _ in range(args.steps):
        n_tails = one_step(True, windows, acc)
    barrier()
    st = plan.stats()
    sampler.stop()

    # dominant kernel, timed alone with CUDA events on the plan's stream (each launch bracketed, synchronised)
    plan.set_profiling(True)
    plan.reset_stats()
    a, b = chunks[-1]
    plan.search(k_sigma, cap=cap, copy=False)
    pst = plan.stats()
    plan.set_profiling(False)
    kern_s = pst["fused_kernel_ms"] * 1e-3
    kern_corr = b - a

    times = torch.tensor([acc["search_ms"] * 1e-3, acc["e2e_s"], acc["e2e_s"] + acc["gen_s"]], dtype=torch.float64,
                         device=dev if dev else "cpu")
    gathered = None
    if world > 1:
        dist.all_reduce(times, op=dist.ReduceOp.MAX)
        # the only exchange of the path: the (rare) tail records of every rank's last pass, concatenated on rank 0
        mine = np.concatenate(last_tails) if last_tails else np.zeros(0, dtype=bege.TAIL_DTYPE)
        gathered = shard.gather_tails(mine)
    t_search, t_e2e, t_e2e_gen = float(times[0]), float(times[1]), float(times[2])
    total_corr = T_total * world * args.steps
    value = total_corr / t_search
    e2e = total_corr / t_e2e
    e2e_gen = total_corr / t_e2e_gen
    plan.close()
    if rank != 0:
        return

    if selftest:
        print(json.dumps({"selftest_launch": True, "metric": METRIC, "value": None, "unit": UNIT, "n_gpus": world,
                          "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_search / max(args.steps, 1),
                          "gathered_tails": int(gathered.size) if gathered is not None else None,
                          "gathered_ids_ok": bool(gathered is None or np.array_equal(
                              np.sort(np.unique(gathered["template_id"] // T_total)), np.arange(world))),
                          "config": {"workload": f"launch self-test, {T_total} templates per rank, {len(chunks)} chunks"}}),
              flush=True)
        return

    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
    rate_kernel = kern_corr / kern_s
    hbm_achieved = rate_kernel * ALG_BYTES_PER_CORR * 1e-9
    alu_achieved = rate_kernel * FFT_FLOP * 1e-12
    step_ms = np.asarray(acc["step_ms"])
    extras = {}
    if world == 1 and not args.no_extras:
        del x_host
        torch.cuda.empty_cache()
        extras = _extra_workloads(args, dev, local_rank)
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        v, used, dt, _ = oracle_rate(f0, fdot, x_np, k_sigma, args.cpu_sample)
        cpu = {"value": v, "unit": UNIT, "cores": used, "kind": "oracle",
               "sample": f"{args.cpu_sample} templates strided over the 2^20 bank x 1 segment ({dt:.1f} s)",
               "includes": "template generation + forward transform of every template inside the timed loop: the like-for-"
                           "like GPU figure is e2e_incl_generation, not value or e2e",
               "gpu_over_cpu_like_for_like": e2e_gen / v}
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * t_search / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"configs[2]: {T_total} templates x 1 segment per GPU, N=2^16, k=6, "
                               "band-limited Gaussian noise seed 2",
                   "bank_chunks": len(chunks), "chunk_templates": chunk,
                   "timed": "sum over chunks of bege_search (incl. D2H of tails); chunk generation untimed",
                   "l2": f"inputs larger than L2 (each chunk streams {chunk * tpl_bytes / 2**30:.1f} GiB of spectra)",
                   "tails_per_step": n_tails},
        "median": {"ms_per_step": float(np.median(step_ms)), "value": T_total / (float(np.median(step_ms)) * 1e-3),
                   "ms_per_step_min": float(step_ms.min()), "ms_per_step_max": float(step_ms.max())},
        "bank_generate_ms_per_step": 1e3 * acc["gen_s"] / args.steps,
        "segment_load_ms_per_step": 1e3 * acc["load_s"] / args.steps,
        "untimed_note": "bank_generate (fp64, once per chunk and pass because the 2^20-template bank exceeds HBM) is not "
                        "part of value; segment_load (H2D + forward FFT of the segment) is part of e2e only",
        "e2e": {"value": e2e, "unit": UNIT, "h2d_bytes_per_step": acc["h2d"] // args.steps,
                "d2h_bytes_per_step": acc["d2h"] // args.steps,
                "what": "per chunk: bege_segment_load from pinned host memory + bege_search into pinned host memory"},
        "e2e_incl_generation": {"value": e2e_gen, "unit": UNIT,
                                "what": "as e2e, plus bege_bank_generate of every chunk (the 2^20-template bank exceeds HBM and "
                                        "is regenerated on every pass): wall time of generation + segment_load + search"},
        "gpu_launches": int(acc["launches"]),
        "gpu_launches_note": "kernels of libbege.so launched inside the timed calls (per chunk: 3 segment-load kernels + "
                             "the persistent search kernel, up to 8 launches = slices); the untimed bank generation "
                             "launched %d more" % (int(st["kernel_launches"]) - int(acc["launches"])),
        "clocks": sampler.summary(windows),
        "gflops_equiv": value * FFT_FLOP * 1e-9,
        "roofline": {"bound": "alu", "achieved": alu_achieved, "peak": FP32_PEAK * 1e-12, "unit": "TFLOP/s",
                     "frac": alu_achieved / (FP32_PEAK * 1e-12), "traffic": NCU_DRAM_BYTES_PER_CORR * kern_corr,
                     "traffic_source": "offline", "traffic_note": "bytes per launch group = ncu dram bytes per correlation "
                     f"({NCU_SOURCE}) x correlations of the timed search; not re-measured in this run",
                     "kernel": "k_search (persistent warp-specialised search kernel), CUDA events on the plan's stream, "
                               f"{pst['fused_kernel_launches']} launches (slices of one search) over {kern_corr} correlations",
                     "peak_source": "derived: 148 SM x 128 fp32 lanes x 2 x 1.965 GHz (DESIGN.md); "
                                    "flops = 5 N log2 N per correlation (PAPER.md:134)",
                     "ncu_offline": NCU_OFFLINE,
                     "fma_pipe": {"ceiling_corr_per_s": FMA_PIPE_CEILING, "frac": rate_kernel / FMA_PIPE_CEILING,
                                  "note": "context: ~1,000 FMA-pipe cycles per 32 lags x 16 row pairs of this radix-16 arithmetic "
                                          "(packed f32x2 = 2 cycles; profiles/r2_search_kernel.md, r3_search_kernel.md); not the roofline denominator"},
                     "hbm": {"achieved": hbm_achieved, "peak": hbm_peak, "unit": "GB/s",
                             "frac": hbm_achieved / hbm_peak, "of": "measured" if peaks else "fallback",
                             "stored_bytes_per_template": tpl_bytes}},
        "cpu_baseline": cpu,
        "context": {"paper": "~8e4 correlations/s per GPU, ~1e6 on ~12 GPUs, ~65% of clFFT (AMD, OpenCL; PAPER.md:211)"},
    }
    line.update(extras)
    if gathered is not None:
        line["gathered_tails"] = int(gathered.size)
    print(json.dumps(line), flush=True)


def spawn_ranks(args):
    """`python bench.py --gpus N` with no torchrun environment: start the N ranks here (one per GPU, 127.0.0.1)."""
    import socket
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "INFO")              # communicator / rank lines on stderr (the driver counts ranks from them)
    env.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
    return subprocess.call(cmd, env=env)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference", "cufft", "ovs_probe"])
    ap.add_argument("--templates", type=int, default=1 << 20, help="templates per GPU (default: configs[2])")
    ap.add_argument("--chunk", type=int, default=0, help="bank chunk size (default: what fits HBM)")
    ap.add_argument("--cpu-sample", type=int, default=24576)
    ap.add_argument("--ref-sample", type=int, default=8192)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip the configs[3] / configs[4] blocks")
    ap.add_argument("--batched-segments", type=int, default=64)
    ap.add_argument("--extra-reps", type=int, default=2)
    ap.add_argument("--tail-cap", type=int, default=80_000_000)
    ap.add_argument("--cufft-batch", type=int, default=2048, help="templates per step of the --impl cufft reference point")
    ap.add_argument("--ovs-templates", type=int, default=147456, help="templates of the --impl ovs_probe measurement")
    ap.add_argument("--selftest-launch", default="", metavar="MODULE:FACTORY",
                    help="exercise the multi-rank plumbing only (gloo, no GPU, no search) with the stand-in plan that "
                         "FACTORY(rank) of the importable MODULE returns; used by tests/test_host_logic.py")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and args.impl == "ours":
        sys.exit(spawn_ranks(args))
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank)
        return
    if args.impl == "cufft":
        run_cufft(args, rank, local_rank)
        return
    if args.impl == "ovs_probe":
        run_ovs_probe(args, rank, local_rank)
        return
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("gloo" if args.selftest_launch else "nccl")
    try:
        run_ours(args, rank, world, local_rank)
    finally:
        if world > 1:
            import torch.distributed as dist
            dist.destroy_process_group()


if __name__ == "__main__":
    main()
