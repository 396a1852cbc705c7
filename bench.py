#!/usr/bin/env python
"""bench.py — Gsamples/s flagged by the LOF hot path (arXiv 1701.08197) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--config cfg2|cfg3|cfg4|cfg5] [--quick]

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


def kernel_source_hash():
    """sha1 of the CUDA sources: stamps an ncu capture so that a stale one is recognised (profiles/*.csv)."""
    import hashlib
    h = hashlib.sha1()
    d = os.path.join(ROOT, "paper_1701_08197_b200", "csrc")
    for f in sorted(os.listdir(d)):
        h.update(open(os.path.join(d, f), "rb").read())
    return h.hexdigest()[:12]


def measured_traffic(config):
    """DRAM bytes per launch of the dominant kernel from the newest committed `ncu --set full` capture
    (profiles/r*_traffic.csv, one row per config, stamped with the hash of the sources it was taken on).
    Returns (bytes or None, kernel, thread-instr/sample or None, source note)."""
    import csv
    import glob
    for p in sorted(glob.glob(os.path.join(ROOT, "profiles", "r*_traffic.csv")), reverse=True):
        for r in csv.DictReader(open(p)):
            if r["config"] != config:
                continue
            stamp = r.get("csrc_sha1", "")
            fresh = stamp == kernel_source_hash()
            note = f"ncu capture {os.path.basename(p)} (sources {stamp or 'unstamped'}" + \
                   (", same as this build)" if fresh else ", OLDER than this build: stale)")
            tips = float(r.get("thread_instr_per_sample") or 0) or None
            return float(r["dram_bytes_read"]) + float(r["dram_bytes_write"]), r["kernel"], tips, note
    return None, None, None, "no capture committed"


_CFG2 = {}


def make_workload(name, seed=0):
    """Returns (power float32 [S][C][T] numpy, dict of Flagger kwargs, description, block seconds)."""
    from paper_1701_08197_b200 import workloads as wl
    if name in ("cfg2", "cfg2x8", "cfg2x16", "cfg2x32"):
        if seed not in _CFG2:                   # generated once per run: 64 subband-seconds of 96 streams
            _CFG2.clear()
            _CFG2[seed] = wl.config2(seed, n_subbands=64, want_truth=False).power
        nsub = 64 if name == "cfg2" else int(name[5:])
        return _CFG2[seed][:96 * nsub], dict(max_window=64), \
            f"cfg2 LOFAR-like pre-correlation 48st x 2pol x 64ch x 768t, x{nsub} subbands", float(nsub)
    if name == "cfg3":
        w = wl.config3(seed, want_truth=False)
        return w.power, dict(max_window=64), "cfg3 visibility-shaped 1891 baselines x 4 pol x 16ch x 768t", 1.0
    if name == "cfg5":
        g = wl.Config5Stream(seed, want_truth=False)
        w = g.next_block()
        return w.power, dict(max_window=64, history_length=300, history_min_fill=2), \
            "cfg5 beam-formed 488 subbands x 16ch x 12208t + history flagger", 1.0
    if name == "cfg4":
        w = wl.config4(seed)                   # full size: 96 streams x 32 subbands x 195 312 complex int16, 2.4 GB
        return w.volt, dict(max_window=256), "cfg4 raw-voltage 48 stations x 2 pol x 32 subbands x 195312 t, ci16", 1.0
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
    """Times the oracle as it stands on a bounded sample of whole streams: on all host cores (one thread per group
    of streams, the paper's CPU decomposition) and on a single thread.
    Returns (samples/s all cores, cores, sample note, samples/s one thread)."""
    from oracle import lofo
    lofo.build()
    S, C, T = power.shape[:3]
    cores = os.cpu_count() or 1
    okw = dict(kw)
    n = min(S, max(cores, 2 * cores))

    def run(m, threads):
        prm = lofo.make_params(m, C, T, **okw)
        x = power[:m]
        if x.dtype == np.int16:                        # raw voltages: the oracle forms the power first
            x = lofo.power_from_ci16(x)
        lofo.flag_block_threads(prm, x, threads)

    t0 = time.perf_counter()
    run(n, cores)
    dt = time.perf_counter() - t0
    rate = n * C * T / dt
    n2 = int(min(S, max(n, rate * target_seconds / (C * T))))
    if n2 > n:
        t0 = time.perf_counter()
        run(n2, cores)
        dt = time.perf_counter() - t0
        n = n2
    n1 = max(1, min(S, int(rate / cores * 3.0 / (C * T))))    # about 3 s of one core
    t0 = time.perf_counter()
    run(n1, 1)
    dt1 = time.perf_counter() - t0
    return n * C * T / dt, cores, f"first {n} of {S} streams of the same block, {cores} threads over whole streams, " \
        f"{dt:.1f} s; one thread: first {n1} streams, {dt1:.1f} s", n1 * C * T / dt1


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
            "config": {"workload": desc, "S": S, "C": C, "T": T, **kw, "input_bytes": S * C * T * 4,
                       "l2": "input larger than L2 (126 MB), two buffers alternated, no flush",
                       "preheat": "1.5 s of untimed steps before the timed ones (sustained clocks)"},
            "cpu_baseline": {"value": val, "unit": "Gsamples/s", "cores": cores, "kind": "oracle",
                             "sample": f"first {n} of {S} streams per step, {cores} threads over whole streams"},
            "e2e": {"value": val, "unit": "Gsamples/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


PATH_NAMES = {0: "none", 1: "fused", 2: "long-row (segments)", 3: "long-row (cooperative tiles)", 4: "generic"}


def time_config(lof, name, steps, warmup, local, seed=0, preheat_s=1.5, sampler=None, mode="block", **extra_kw):
    """Device-timed steps of one configuration with inputs resident in HBM.  A step = one pass of the whole hot
    path over the block (+ lof_history_update when the config has a history).  `preheat_s` seconds of untimed
    steps come first, so that the clocks are the sustained ones and the clock sampler sees the load.
    mode: "block" = lof_flag_block, "integrated" = lof_flag_block_integrated."""
    import torch
    power, kw, desc, block_s = make_workload(name, seed=seed)
    kw = dict(kw, **extra_kw)
    S, C, T = power.shape[:3]
    n_samples = S * C * T
    f = lof.Flagger(S, C, T, device=local, **kw)
    has_hist = kw.get("history_length", 0) > 0 and mode == "block"
    # two resident input buffers (the second a time-rolled copy) used alternately; each exceeds L2
    xs = [torch.from_numpy(power).cuda(), None]
    xs[1] = torch.roll(xs[0], 37, dims=2).contiguous() if power.nbytes < (2 << 30) else xs[0]
    flags, stats, stats2 = f.new_flags(), f.new_stats(), f.new_stats()
    stream = torch.cuda.current_stream()

    def step(i):
        if mode == "integrated":
            f.flag_block_integrated(xs[i & 1], flags, stats, stats2, stream)
        else:
            f.flag_block(xs[i & 1], flags, stats, stream)
            if has_hist:
                f.history_update(flags, None, stream)

    for i in range(max(warmup, 3)):
        step(i)
    torch.cuda.synchronize()
    if sampler is not None and not sampler.is_alive():
        sampler.start()
    t0 = time.perf_counter()
    i = 0
    while time.perf_counter() - t0 < preheat_s:            # untimed: sustained clocks, ring of the two buffers
        for _ in range(8):
            step(i); i += 1
        torch.cuda.synchronize()
    l0 = f.launch_count()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
    torch.cuda.synchronize()
    ev[0].record(stream)
    for i in range(steps):
        step(i)
        ev[i + 1].record(stream)
    torch.cuda.synchronize()
    launches = f.launch_count() - l0
    total_ms = ev[0].elapsed_time(ev[-1])
    per = sorted(ev[i].elapsed_time(ev[i + 1]) for i in range(steps))
    return dict(f=f, power=power, kw=kw, desc=desc, block_s=block_s, S=S, C=C, T=T, n_samples=n_samples,
                total_ms=total_ms, per=per, launches=int(launches), path=PATH_NAMES.get(f.path_used(), "?"),
                flags=flags, stats=stats)


def run_gpu(args):
    import torch
    from paper_1701_08197_b200 import build, lof, sharding
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
    peak, peak_src = measured_peaks()
    sampler = ClockSampler(local)
    if dist:
        dist.barrier()
    # ---- headline: BASELINE.json configs[1] batched over 64 subbands (each rank flags its own subbands)
    # --row: one of SURVEY.md §8(f)'s rows instead of the plain block (for profiling; use with --quick)
    row_kw = {"sir": dict(sir_eta=0.2), "mad": dict(stats_mode=1)}.get(args.row, {})
    r = time_config(lof, args.config, args.steps, args.warmup, local, seed=rank, sampler=sampler,
                    mode="integrated" if args.row == "integrated" else "block", **row_kw)
    if dist:
        dist.barrier()
    sampler.stop_flag = True
    sampler.join()
    f, power, kw = r["f"], r["power"], r["kw"]
    S, C, T, n_samples = r["S"], r["C"], r["T"], r["n_samples"]
    total_ms = sharding.max_over_ranks(r["total_ms"], device="cuda")
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
    del hp, hf, hs
    f.close()
    del r["f"], r["flags"], r["stats"]

    if rank != 0:
        if dist:
            dist.destroy_process_group()
        return
    ms_step = total_ms / args.steps
    achieved = n_samples * ALGO_BYTES_PER_SAMPLE / (ms_step * 1e-3) / 1e9
    traffic, kname, tips, traffic_src = measured_traffic(args.config)
    one_kernel = r["launches"] in (args.steps, 3 * args.steps)  # fused: 1 launch per step (+2 history kernels)
    line = {
        "metric": "Gsamples/s flagged", "value": value, "unit": "Gsamples/s", "n_gpus": world,
        "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "ms_per_step_min": r["per"][0],
        "ms_per_step_median": r["per"][len(r["per"]) // 2],
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "real_time_factor": world * r["block_s"] * args.steps / (total_ms * 1e-3),
        "config": {"workload": r["desc"], "row": args.row, "S": S, "C": C, "T": T, **kw, "input_bytes": n_samples * 4,
                   "l2": "input larger than L2 (126 MB), two buffers alternated, no flush",
                   "preheat": "1.5 s of untimed steps before the timed ones (sustained clocks)"},
        "gpu_launches": r["launches"], "path": r["path"],
        "clocks": sampler.summary(),
        "e2e": {"value": e2e_val, "unit": "Gsamples/s", "h2d_bytes_per_step": n_samples * 4,
                "d2h_bytes_per_step": S * C * ((T + 31) // 32) * 4 + S * 32, "steps": e2e_steps},
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "traffic": traffic, "traffic_source": traffic_src, "peak_source": peak_src,
                     "frac_of_8TBs": achieved / 8000.0,
                     "kernel": (kname or "lof_k_fused") + " (one launch per step)" if one_kernel
                     else "whole step (all kernels of lof_flag_block)",
                     "algorithmic_bytes_per_launch": n_samples * ALGO_BYTES_PER_SAMPLE,
                     "algorithmic_bytes_per_sample": ALGO_BYTES_PER_SAMPLE},
    }
    if tips:
        # the roof this kernel is actually pressed against: instruction issue.  Executed
        # thread-instructions per sample from the stamped ncu capture x the live rate, against
        # SMs x 4 schedulers x 32 lanes x the SM clock sampled during the run
        sms = torch.cuda.get_device_properties(0).multi_processor_count
        mhz = line["clocks"].get("sm_mhz") or line["clocks"].get("sm_max_mhz") or 1965.0
        peak_i = sms * 4 * 32 * mhz * 1e6
        line["roofline"]["issue"] = {"thread_instr_per_sample": tips, "achieved": value * 1e9 * tips / world,
                                     "peak": peak_i, "unit": "thread-instr/s",
                                     "frac": value * 1e9 * tips / world / peak_i}
    cpu_val, cores, sample, cpu_1 = oracle_rate(power, kw)
    line["cpu_baseline"] = {"value": cpu_val / 1e9, "unit": "Gsamples/s", "cores": cores, "kind": "oracle",
                            "sample": sample, "value_1thread": cpu_1 / 1e9}
    del power
    if args.config == "cfg2" and not args.quick and world == 1:
        line["per_config"] = per_config_lines(lof, local, peak)
        line["linearity"] = linearity_check(lof, local)
        line["next_rows"] = next_rows(lof, local, peak, ms_step)
    print(json.dumps(line))
    if dist:
        dist.destroy_process_group()


def per_config_lines(lof, local, peak):
    """The other three LOFAR-shaped configs at the sizes BASELINE.json states, each 10 device-timed steps after
    3 warm-up steps and a 1 s pre-heat (same protocol as the headline)."""
    out = {}
    for name in ("cfg3", "cfg4", "cfg5"):
        t0 = time.perf_counter()
        smp = ClockSampler(local)
        r = time_config(lof, name, 10, 3, local, preheat_s=1.0, sampler=smp)
        smp.stop_flag = True
        smp.join()
        ms = r["total_ms"] / 10
        gb = r["n_samples"] * ALGO_BYTES_PER_SAMPLE / (ms * 1e-3) / 1e9
        out[name] = {"workload": r["desc"], "S": r["S"], "C": r["C"], "T": r["T"], **r["kw"],
                     "gsamples_s": r["n_samples"] / (ms * 1e-3) / 1e9, "ms_per_step": ms,
                     "ms_per_step_min": r["per"][0], "real_time_factor": r["block_s"] / (ms * 1e-3),
                     "achieved_GBs": gb, "roofline_frac": gb / peak, "gpu_launches": r["launches"],
                     "path": r["path"], "clocks": smp.summary(), "wall_s": None}
        r["f"].close()
        del r
        import torch
        torch.cuda.empty_cache()
        out[name]["wall_s"] = round(time.perf_counter() - t0, 1)
    return out


def linearity_check(lof, local):
    """run time linear in the number of samples.  Config 2 at 16, 32 and 64 subbands (S = 1536,
    3072, 6144 streams, all far above the number of SMs): ms per step and its deviation from the line through
    the origin fitted to the three points."""
    import torch
    pts = []
    for nsub in (16, 32, 64):
        power = make_workload("cfg2" if nsub == 64 else f"cfg2x{nsub}")[0]
        S, C, T = power.shape
        f = lof.Flagger(S, C, T, device=local, max_window=64)
        x = torch.from_numpy(power).cuda()
        fl, st = f.new_flags(), f.new_stats()
        for _ in range(5):
            f.flag_block(x, fl, st)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for _ in range(20):
            f.flag_block(x, fl, st)
        e1.record()
        torch.cuda.synchronize()
        pts.append((S, e0.elapsed_time(e1) / 20))
        f.close()
        del x
    slope = sum(s * m for s, m in pts) / sum(s * s for s, m in pts)
    return {"S": [p[0] for p in pts], "ms_per_step": [p[1] for p in pts], "ms_per_stream_fit": slope,
            "max_rel_deviation_from_line": max(abs(m - slope * s) / (slope * s) for s, m in pts)}


def next_rows(lof, local, peak, ms_plain):
    """SURVEY.md §8(f) rows on the headline workload: SIR operator (cost relative to the plain block), fully
    integrated mode (HBM-bound: GB/s against the measured peak), MAD scale (multi-kernel path)."""
    out = {}
    r = time_config(lof, "cfg2", 10, 3, local, preheat_s=0.5, sir_eta=0.2)
    ms = r["total_ms"] / 10
    out["sir_eta_0.2"] = {"ms_per_step": ms, "gsamples_s": r["n_samples"] / (ms * 1e-3) / 1e9,
                          "cost_vs_plain_block": ms / ms_plain - 1.0, "gpu_launches": r["launches"]}
    r["f"].close(); del r
    r = time_config(lof, "cfg2", 10, 3, local, preheat_s=0.5, mode="integrated")
    ms = r["total_ms"] / 10
    gb = r["n_samples"] * ALGO_BYTES_PER_SAMPLE / (ms * 1e-3) / 1e9
    out["integrated_mode"] = {"ms_per_step": ms, "gsamples_s": r["n_samples"] / (ms * 1e-3) / 1e9,
                              "achieved_GBs": gb, "roofline_frac": gb / peak, "gpu_launches": r["launches"]}
    r["f"].close(); del r
    r = time_config(lof, "cfg2x8", 10, 3, local, preheat_s=0.5, stats_mode=1)
    ms = r["total_ms"] / 10
    out["stats_mode_mad_x8_subbands"] = {"ms_per_step": ms, "gsamples_s": r["n_samples"] / (ms * 1e-3) / 1e9,
                                         "gpu_launches": r["launches"], "path": r["path"]}
    r["f"].close(); del r
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="lof", choices=["lof", "reference"])
    ap.add_argument("--config", default="cfg2")
    ap.add_argument("--row", default="block", choices=["block", "sir", "integrated", "mad"],
                    help="time the plain block (default) or a §8(f) row: SIR operator, integrated mode, MAD scale")
    ap.add_argument("--quick", action="store_true", help="headline only: no per_config / linearity / next_rows")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
