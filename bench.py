#!/usr/bin/env python
"""bench.py -- template correlations/s at N = 2^16 (C2C fp32) on B200, BASELINE.json configs[2].

One "step" = one pass of the whole 2^20-template bank (1024 x 1024 grid, 350-2000 Hz x +-400 Hz/s)
against one 16 s segment of band-limited Gaussian noise (seed 2), k = 6.  The bank (2^20 x 448 KiB of
in-band spectra) does not fit HBM, so it is processed in chunks: chunk generation (bege_bank_generate) is
untimed, as BASELINE.json configs[2] states ("template spectra are precomputed once, and the search is
timed separately from generation"); the timed region of a step is the sum over chunks of bege_search,
each bracketed by a device synchronize and CUDA events on the plan's stream.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--templates T]

N > 1 (torchrun): every rank searches its own 2^20-template shard of an N-times finer fdot grid (weak
scaling, no data-path collective); tail records are gathered on rank 0 after the timed region.
--impl reference times the fp64 CPU oracle (oracle/) on the host cores, on a bounded sample.
--impl cufft times the same steps built from library kernels (torch + cuFFT): a reference point for context only.
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
# dram__bytes_read.sum + dram__bytes_write.sum of k_search per correlation, from the ncu --set full capture summarised
# in profiles/r1g_search_kernel_final.md (36,864-template launch: 16.914 GB read + 0.365 GB written)
NCU_DRAM_BYTES_PER_CORR = (16.913879e9 + 0.365349e9) / 36864
FP32_PEAK = 148 * 128 * 2 * 1.965e9               # SMs x fp32 lanes x 2 flop x max SM clock


# ------------------------------------------------------------------------------------------ clocks
class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

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
        sm, smax, reasons, power = [], 0.0, set(), 0.0
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
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": smax or None,
                "reasons": sorted(reasons), "samples": len(sm), "power_w_max": power or None}


# ------------------------------------------------------------------------------------------ oracle arm
def oracle_rate(f0, fdot, x, k_sigma, sample: int, seconds_hint: float = 0.0):
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


# ------------------------------------------------------------------------------------------ our arm
def run_ours(args, rank, world, local_rank):
    import torch
    import torch.distributed as dist
    from paper_1708_01609_b200 import bege, shard

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
    x_host = torch.from_numpy(synth.noise_segment(2)[None, :]).pin_memory()
    k_sigma, cap = 6.0, 1 << 16

    plan = bege.Plan(synth.N_SEG, synth.FS, synth.BAND, device=local_rank)
    tpl_bytes = plan.stats()["hbm_bytes_per_template"]
    free, _total = torch.cuda.mem_get_info(dev)
    chunk = args.chunk or int(min(T_total, (free * 0.88) // tpl_bytes))
    chunk = max(72, chunk - chunk % 72) if chunk < T_total else T_total
    plan.alloc_workspace(chunk, 1, cap)
    chunks = shard.chunk_ranges(0, T_total, chunk)
    plan.segment_load(x_host)

    sampler = ClockSampler(local_rank)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in chunks]

    def barrier():
        torch.cuda.synchronize(dev)
        if world > 1:
            dist.barrier()

    def one_step(timed: bool, windows, acc):
        """generation untimed; per chunk: [segment_load from pinned host + search] = e2e, [search] = value."""
        n_tails = 0
        for ci, (a, b) in enumerate(chunks):
            plan.bank_generate(f0[a:b], fdot[a:b], synth.TAU)              # untimed (configs[2])
            barrier()
            l0 = plan.stats()["kernel_launches"]
            t0 = time.perf_counter()
            plan.segment_load(x_host)                                        # H2D of the segment + forward FFT
            t1 = time.perf_counter()
            ev[ci][0].record()
            _tails, n = plan.search(k_sigma, cap=cap, copy=False)            # D2H of count + records inside
            ev[ci][1].record()
            torch.cuda.synchronize(dev)
            t2 = time.perf_counter()
            n_tails += n
            if timed:
                windows.append((t1, t2))
                acc["search_ms"] += ev[ci][0].elapsed_time(ev[ci][1])
                acc["e2e_s"] += t2 - t0
                acc["d2h"] += 8 + 12 * min(n, cap)
                acc["h2d"] += x_host.numel() * 8
                acc["launches"] += plan.stats()["kernel_launches"] - l0
        return n_tails

    sampler.start()
    acc = {"search_ms": 0.0, "e2e_s": 0.0, "d2h": 0, "h2d": 0, "launches": 0}
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

    # dominant kernels (pass 1 + pass 2 of the search), timed alone with CUDA events on the plan's stream
    plan.set_profiling(True)
    plan.reset_stats()
    a, b = chunks[-1]
    plan.search(k_sigma, cap=cap, copy=False)
    pst = plan.stats()
    plan.set_profiling(False)
    kern_s = pst["fused_kernel_ms"] * 1e-3
    kern_corr = b - a

    search_s = torch.tensor([acc["search_ms"] * 1e-3, acc["e2e_s"]], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(search_s, op=dist.ReduceOp.MAX)
    t_search, t_e2e = float(search_s[0]), float(search_s[1])
    total_corr = T_total * world * args.steps
    value = total_corr / t_search
    e2e = total_corr / t_e2e
    if rank != 0:
        plan.close()
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
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        v, used, dt, _ = oracle_rate(f0, fdot, x_host.numpy(), k_sigma, args.cpu_sample)
        cpu = {"value": v, "unit": UNIT, "cores": used, "kind": "oracle",
               "sample": f"{args.cpu_sample} templates strided over the 2^20 bank x 1 segment ({dt:.1f} s)"}
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
        "e2e": {"value": e2e, "unit": UNIT, "h2d_bytes_per_step": acc["h2d"] // args.steps,
                "d2h_bytes_per_step": acc["d2h"] // args.steps,
                "what": "per chunk: bege_segment_load from pinned host memory + bege_search into pinned host memory"},
        "gpu_launches": int(acc["launches"]),
        "gpu_launches_note": "kernels of libbege.so launched inside the timed calls (per chunk: 2 segment-load kernels + 1 persistent search kernel); the untimed bank generation launched %d more" % (int(st["kernel_launches"]) - int(acc["launches"])),
        "clocks": sampler.summary(windows),
        "gflops_equiv": value * FFT_FLOP * 1e-9,
        "roofline": {"bound": "alu", "achieved": alu_achieved, "peak": FP32_PEAK * 1e-12, "unit": "TFLOP/s",
                     "frac": alu_achieved / (FP32_PEAK * 1e-12), "traffic": NCU_DRAM_BYTES_PER_CORR * kern_corr,
                     "traffic_note": "bytes per launch = ncu dram bytes per correlation (profiles/r1g_search_kernel_final.md) x correlations of the timed launch",
                     "kernel": "k_search (persistent warp-specialised search kernel, one launch per bank chunk), CUDA events on the plan's stream, "
                               f"{pst['fused_kernel_launches']} launch over {kern_corr} correlations",
                     "peak_source": "derived: 148 SM x 128 fp32 lanes x 2 x 1.965 GHz (DESIGN.md); "
                                    "flops = 5 N log2 N per correlation (PAPER.md:134)",
                     "hbm": {"achieved": hbm_achieved, "peak": hbm_peak, "unit": "GB/s",
                             "frac": hbm_achieved / hbm_peak, "of": "measured" if peaks else "fallback",
                             "stored_bytes_per_template": tpl_bytes}},
        "cpu_baseline": cpu,
        "context": {"paper": "~8e4 correlations/s per GPU, ~1e6 on ~12 GPUs, ~65% of clFFT (AMD, OpenCL; PAPER.md:211)"},
    }
    print(json.dumps(line), flush=True)
    plan.close()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference", "cufft"])
    ap.add_argument("--templates", type=int, default=1 << 20, help="templates per GPU (default: configs[2])")
    ap.add_argument("--chunk", type=int, default=0, help="bank chunk size (default: what fits HBM)")
    ap.add_argument("--cpu-sample", type=int, default=24576)
    ap.add_argument("--ref-sample", type=int, default=8192)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cufft-batch", type=int, default=2048, help="templates per step of the --impl cufft reference point")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank)
        return
    if args.impl == "cufft":
        run_cufft(args, rank, local_rank)
        return
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl")
    try:
        run_ours(args, rank, world, local_rank)
    finally:
        if world > 1:
            import torch.distributed as dist
            dist.destroy_process_group()


if __name__ == "__main__":
    main()
