#!/usr/bin/env python
"""bench.py — Gsamples/s flagged by the LOF hot path (arXiv 1701.08197) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--config cfg2|cfg3|cfg5]

A step = one pass of the whole hot path (statistics -> thresholds -> SumThreshold freq -> SumThreshold
time -> bit-pack + row sums [-> history flagger when the config has one]) over one block of synthetic
input already resident in HBM.  Workload at N = 1: BASELINE.json configs[1], the LOFAR-like
pre-correlation block (96 streams x 64 channels x 768 samples per subband-second), batched over 64
subbands (6144 streams, 1.2 GB: larger than L2, so no flush is needed between steps).
Prints ONE JSON line (rank 0).  `--impl reference` times the CPU oracle instead (rank 0 only).
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

ALGO_BYTES_PER_SAMPLE = 4.0 + 1.0 / 8.0     # one read of the power + the flag bit


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, device copy)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def measured_traffic(config):
    """DRAM bytes per launch of the dominant kernel from the committed ncu --set full capture, or None."""
    import csv
    p = os.path.join(ROOT, "profiles", "r01_fused_traffic.csv")
    if os.path.exists(p):
        for r in csv.DictReader(open(p)):
            if r["config"] == config:
                return float(r["dram_bytes_read"]) + float(r["dram_bytes_write"]), r["kernel"], \
                    float(r.get("thread_instr_per_sample") or 0) or None
    return None, None, None


def make_workload(name, seed=0):
    """Returns (power float32 [S][C][T] numpy, dict of Flagger kwargs, description, block seconds)."""
    from paper_1701_08197_b200 import workloads as wl
    if name == "cfg2":
        w = wl.config2(seed, n_subbands=64, want_truth=False)
        return w.power, dict(max_window=64), "cfg2 LOFAR-like pre-correlation 48st x 2pol x 64ch x 768t, x64 subbands", 64.0
    if name == "cfg2x8":
        w = wl.config2(seed, n_subbands=8, want_truth=False)
        return w.power, dict(max_window=64), "cfg2 LOFAR-like pre-correlation, x8 subbands", 8.0
    if name == "cfg3":
        w = wl.config3(seed, want_truth=False)
        return w.power, dict(max_window=64), "cfg3 visibility-shaped 1891 baselines x 4 pol x 16ch x 768t", 1.0
    if name == "cfg5":
        g = wl.Config5Stream(seed, want_truth=False)
        w = g.next_block()
        return w.power, dict(max_window=64, history_length=300, history_min_fill=2), \
            "cfg5 beam-formed 488 subbands x 16ch x 12208t + history flagger", 1.0
    if name == "cfg4":
        # cut to 12 stations (24 streams, 600 MB of complex int16) so that generation stays within a minute
        w = wl.config4(seed, n_stations=12)
        return w.volt, dict(max_window=256), "cfg4 raw-voltage 12 of 48 stations x 2 pol x 32 subbands x 195312 t, ci16", 0.25
    if name == "cfg1":
        w = wl.config1(seed)
        return w.power, dict(max_window=32), "cfg1 tiny 1 x 16 x 256", 1.0
    raise SystemExit(f"unknown config {name}")


class ClockSampler(threading.Thread):
    """Samples nvidia-smi clocks and throttle reasons during the timed region."""
    Q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.rows, self.stop_flag = index, [], False

    def run(self):
        while not self.stop_flag:
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5).stdout
                f = [x.strip() for x in out.strip().split(",")]
                if len(f) >= 6:
                    self.rows.append(f)
            except Exception:
                pass
            time.sleep(0.05)

    def summary(self):
        if not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unsampled"]}
        sm = sorted(float(r[0]) for r in self.rows)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(r[2 + i].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(self.rows[0][1]), "reasons": reasons,
                "samples": len(self.rows)}


def oracle_rate(power, kw, target_seconds=12.0):
    """Times the oracle as it stands on a bounded sample of whole streams, on all host cores
    (one thread per group of streams, the paper's CPU decomposition)."""
    from oracle import lofo
    lofo.build()
    S, C, T = power.shape[:3]
    cores = os.cpu_count() or 1
    okw = dict(kw)
    n = min(S, max(cores, 2 * cores))

    def run(m):
        prm = lofo.make_params(m, C, T, **okw)
        x = power[:m]
        if x.dtype == np.int16:                        # raw voltages: the oracle forms the power first
            x = lofo.power_from_ci16(x)
        lofo.flag_block_threads(prm, x, cores)

    t0 = time.perf_counter()
    run(n)
    dt = time.perf_counter() - t0
    rate = n * C * T / dt
    n2 = int(min(S, max(n, rate * target_seconds / (C * T))))
    if n2 > n:
        t0 = time.perf_counter()
        run(n2)
        dt = time.perf_counter() - t0
        n = n2
    return n * C * T / dt, cores, f"first {n} of {S} streams of the same block, {cores} threads over whole streams, {dt:.1f} s"


def run_reference(args):
    """--impl reference: the CPU oracle, as it stands, on a bounded sample per step (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    power, kw, desc, block_s = make_workload(args.config)
    S, C, T = power.shape[:3]
    from oracle import lofo
    lofo.build()
    cores = os.cpu_count() or 1
    n = min(S, 4 * cores)                      # a few streams per thread: each step is seconds, not minutes
    okw = {k: v for k, v in kw.items()}
    prm = lofo.make_params(n, C, T, **okw)

    def one_step():
        x = power[:n]
        if x.dtype == np.int16:
            x = lofo.power_from_ci16(x)
        lofo.flag_block_threads(prm, x, cores)

    for _ in range(args.warmup):
        one_step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        one_step()
    dt = time.perf_counter() - t0
    val = n * C * T * args.steps / dt / 1e9
    line = {"impl": "reference", "metric": "Gsamples/s flagged", "value": val, "unit": "Gsamples/s",
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": desc, "S": S, "C": C, "T": T, **kw},
            "cpu_baseline": {"value": val, "unit": "Gsamples/s", "cores": cores, "kind": "oracle",
                             "sample": f"first {n} of {S} streams per step, {cores} threads over whole streams"},
            "e2e": {"value": val, "unit": "Gsamples/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def run_gpu(args):
    import torch
    from paper_1701_08197_b200 import build, lof
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device — the LOF path has no CPU fallback")
    build.build_lib()
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    power, kw, desc, block_s = make_workload(args.config, seed=rank)   # each rank flags its own subbands
    S, C, T = power.shape[:3]
    n_samples = S * C * T
    f = lof.Flagger(S, C, T, device=local, **kw)
    has_hist = kw.get("history_length", 0) > 0
    # two resident input buffers (the second a time-rolled copy) used alternately; each exceeds L2
    xs = [torch.from_numpy(power).cuda(), None]
    xs[1] = torch.roll(xs[0], 37, dims=2).contiguous() if n_samples * 4 < (8 << 30) else xs[0]
    flags, stats = f.new_flags(), f.new_stats()
    stream = torch.cuda.current_stream()

    def step(i):
        f.flag_block(xs[i & 1], flags, stats, stream)
        if has_hist:
            f.history_update(flags, None, stream)

    for i in range(max(args.warmup, 3)):
        step(i)
    torch.cuda.synchronize()
    if dist:
        dist.barrier()
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.2)
    l0 = f.launch_count()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    torch.cuda.synchronize()
    ev[0].record(stream)
    for i in range(args.steps):
        step(i)
        ev[i + 1].record(stream)
    torch.cuda.synchronize()
    launches = f.launch_count() - l0
    if dist:
        dist.barrier()
    total_ms = ev[0].elapsed_time(ev[-1])
    sampler.stop_flag = True
    sampler.join()
    per = sorted(ev[i].elapsed_time(ev[i + 1]) for i in range(args.steps))
    from paper_1701_08197_b200 import sharding
    total_ms = sharding.max_over_ranks(total_ms, device="cuda")
    value = sharding.aggregate_rate(n_samples, args.steps, total_ms, world) / 1e9

    # end to end through the C-ABI host entry point: pinned host input -> flags + stats on the host
    hp = torch.from_numpy(power).pin_memory()
    hf = torch.empty((S, C, f.W), dtype=torch.int32).pin_memory()
    hs = torch.empty((S, 32), dtype=torch.uint8).pin_memory()
    f.flag_block_host(hp, hf, hs)
    e2e_steps = max(2, min(args.steps, 5))
    torch.cuda.synchronize()
    if dist:
        dist.barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        f.flag_block_host(hp, hf, hs)
    e2e_s = time.perf_counter() - t0
    e2e_s = sharding.max_over_ranks(e2e_s, device="cuda")
    e2e_val = sharding.aggregate_rate(n_samples, e2e_steps, e2e_s * 1e3, world) / 1e9

    if rank != 0:
        return
    peak, peak_src = measured_peaks()
    ms_step = total_ms / args.steps
    achieved = n_samples * ALGO_BYTES_PER_SAMPLE / (ms_step * 1e-3) / 1e9
    traffic, kname, tips = measured_traffic(args.config)
    one_kernel = launches in (args.steps, 3 * args.steps)     # fused: 1 launch per step (+2 history kernels)
    cpu_val, cores, sample = oracle_rate(power, kw)
    line = {
        "metric": "Gsamples/s flagged", "value": value, "unit": "Gsamples/s", "n_gpus": world,
        "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "ms_per_step_min": per[0],
        "ms_per_step_median": per[len(per) // 2],
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "real_time_factor": world * block_s * args.steps / (total_ms * 1e-3),
        "config": {"workload": desc, "S": S, "C": C, "T": T, **kw, "input_bytes": n_samples * 4,
                   "l2": "input larger than L2 (126 MB), two buffers alternated, no flush"},
        "gpu_launches": int(launches),
        "clocks": sampler.summary(),
        "e2e": {"value": e2e_val, "unit": "Gsamples/s", "h2d_bytes_per_step": n_samples * 4,
                "d2h_bytes_per_step": S * C * f.W * 4 + S * 32, "steps": e2e_steps},
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "traffic": traffic, "peak_source": peak_src, "frac_of_8TBs": achieved / 8000.0,
                     "kernel": (kname or "lof_k_fused") + " (one launch per step)" if one_kernel
                     else "whole step (all kernels of lof_flag_block, generic path)",
                     "algorithmic_bytes_per_launch": n_samples * ALGO_BYTES_PER_SAMPLE,
                     "algorithmic_bytes_per_sample": ALGO_BYTES_PER_SAMPLE},
        "cpu_baseline": {"value": cpu_val / 1e9, "unit": "Gsamples/s", "cores": cores, "kind": "oracle", "sample": sample},
    }
    if tips:
        # the roof this kernel is actually pressed against: instruction issue.  Executed
        # thread-instructions per sample from the committed ncu capture x the live rate, against
        # SMs x 4 schedulers x 32 lanes x the SM clock sampled during the run
        import torch
        sms = torch.cuda.get_device_properties(0).multi_processor_count
        mhz = line["clocks"].get("sm_mhz") or line["clocks"].get("sm_max_mhz") or 1965.0
        peak_i = sms * 4 * 32 * mhz * 1e6
        line["roofline"]["issue"] = {"thread_instr_per_sample": tips, "achieved": value * 1e9 * tips / world,
                                     "peak": peak_i, "unit": "thread-instr/s",
                                     "frac": value * 1e9 * tips / world / peak_i}
    print(json.dumps(line))
    f.close()
    if dist:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="lof", choices=["lof", "reference"])
    ap.add_argument("--config", default="cfg2")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
