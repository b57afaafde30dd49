#!/usr/bin/env python
"""bench.py -- throughput of the reduced-basis hierarchical matched filter hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config paper|small|large|...] [--impl ours|reference]

A "step" is one rbmf_filter call: all of steps a1-a6 (include/rbmf.h) on one strain segment.  `value` is template-
seconds of strain filtered per second = T * (N / fs) / t_step (the paper's own throughput definition),
with inputs resident in HBM; `e2e` is the same through rbmf_filter_host (pinned host strain in, host triggers out,
copies inside the timed region).  One JSON line on stdout (rank 0).  See DESIGN.md "Measurement".
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "template_seconds_filtered_per_second"
UNIT = "template-seconds/s"

# DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum) from the `ncu --set full` captures summarised
# under profiles/ (r01_launches.md); known only for the configuration that was profiled, else reported as null.
NCU_TRAFFIC = {("paper", 8, "screen", "gemm"): 359.5e6 + 2.5e6, ("paper", 8, "screen", "fft"): 542.8e6 + 1181.2e6,
               ("paper", 8, "screen", "stage2"): 186.0e6 + 3.9e6}


# ------------------------------------------------------------------------------------------------- clocks
class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled while the timed region runs (B200_PROFILING.md recipe)."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.samples = []
        self.proc = None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(gpu_index), "--query-gpu=" + self.FIELDS, "--format=csv,noheader,nounits",
                 "-lms", "50"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.samples.append((time.time(), line.strip()))

    def stop(self):
        if self.proc is not None:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except Exception:
                self.proc.kill()

    def summary(self, t0: float, t1: float) -> dict:
        sm, smax, reasons, power = [], [], set(), []
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for ts, line in self.samples:
            if ts < t0 or ts > t1 + 0.05:
                continue
            parts = [p.strip() for p in line.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); smax.append(float(parts[1])); power.append(float(parts[2]))
            except ValueError:
                continue
            for name, val in zip(names, parts[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w": statistics.median(power) if power else None, "reasons": sorted(reasons),
                "samples": len(sm)}


# ------------------------------------------------------------------------------------------- oracle legs
def oracle_throughput(wl, templates_per_step, steps, warmup, time_budget_s):
    """Times oracle.rbmf_oracle.oracle_filter, as it stands, on `templates_per_step` templates per step (work is
    independent per template).  Returns (template-seconds/s, ms per step, threads, description)."""
    from oracle import rbmf_oracle as orc
    cfg = wl["config"]
    try:
        from threadpoolctl import threadpool_info
        threads = max([int(i.get("num_threads", 1)) for i in threadpool_info()] + [1])
    except Exception:
        threads = 1
    rng = np.random.default_rng(99)
    times = []
    t_begin = time.time()
    for s in range(warmup + steps):
        ids = np.sort(rng.choice(cfg.T, size=min(templates_per_step, cfg.T), replace=False))
        t0 = time.perf_counter()
        orc.oracle_filter(wl["strain"], wl["basis"], wl["coeffs"], wl["sigma"], cfg.N, cfg.fs, cfg.f_low, cfg.w,
                          cfg.thr1, cfg.thr2, templates=ids, keep_margins=False)
        dt = time.perf_counter() - t0
        if s >= warmup:
            times.append(dt)
        if time.time() - t_begin > time_budget_s and len(times) >= 1:
            break
    ms = 1e3 * sum(times) / len(times)
    n_t = min(templates_per_step, cfg.T)
    value = n_t * (cfg.N / cfg.fs) / (ms * 1e-3)
    sample = ("%d of %d templates per step (seeded random subset), full segment, numpy fp64 oracle_filter "
              "(FFT single-threaded, BLAS %d threads), %d timed steps" % (n_t, cfg.T, threads, len(times)))
    return value, ms, threads, sample


def oracle_templates_per_step(cfg):
    # ~1-3 s of CPU work per step: cost per template ~ bins * k * 8 flops (h' build) + an N-point fp64 FFT
    per_template = cfg.bins * cfg.k * 8 / 2.0e10 + cfg.N * 6.0e-8
    return int(max(4, min(cfg.T, 2.0 / per_template)))


# ---------------------------------------------------------------------------------------------------- main
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", default="paper")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--w", type=int, default=None, help="override the averaging window")
    ap.add_argument("--gemm", default="screen", choices=["screen", "bf16x3"],
                    help="stage-1 kernel: fp16 screen + fp32 confirm (library default) or bf16x3")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    import torch
    from paper_2110_13115_b200 import dist as rdist, workloads

    rank, local_rank, world = rdist.env_world()
    cfg = workloads.CONFIGS[args.config]
    if args.w is not None:
        cfg = cfg.replace(w=args.w)
    config_desc = {"workload": "%s: N=%d fs=%g f_low=%g k=%d T=%d w=%d thr=%g/%g injections=%d" % (
        cfg.name, cfg.N, cfg.fs, cfg.f_low, cfg.k, cfg.T, cfg.w, cfg.thr1, cfg.thr2, cfg.n_inj),
        "N": cfg.N, "k": cfg.k, "T": cfg.T, "w": cfg.w, "segment_seconds": cfg.N / cfg.fs,
        "parallelism": "replicas x%d (one strain segment per GPU, no collective)" % world,
        "l2": "working set (basis %.0f MB + beta %.0f MB) exceeds the 126 MB L2; no flush needed" % (
            cfg.N / 2 * cfg.k * 8 / 1e6, cfg.N * cfg.k * 8 / 1e6)}

    # ------------------------------------------------------------------ reference arm: the oracle, on host cores
    if args.impl == "reference":
        if rank != 0:
            return 0
        dev = "cuda" if torch.cuda.is_available() else "cpu"
        wl = workloads.make_workload(cfg, device=dev)
        tps = oracle_templates_per_step(cfg)
        value, ms, threads, sample = oracle_throughput(wl, tps, args.steps, args.warmup, time_budget_s=150.0)
        line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
                "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": config_desc,
                "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
                "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
                "gpu_launches": 0}
        print(json.dumps(line))
        return 0

    # --------------------------------------------------------------------------------------------- our arm
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    rank, local_rank, world = rdist.init()
    torch.cuda.set_device(local_rank)
    device = torch.device("cuda", local_rank)
    from paper_2110_13115_b200 import rbmf

    wl = workloads.make_workload(cfg, device=str(device))
    seg = rdist.segment_index(rank, 0, world)
    strain_np, _ = workloads.make_strain(wl, seg)
    stream = torch.cuda.Stream(device=device)
    with torch.cuda.stream(stream):
        impls = {"screen": rbmf.RBMF_GEMM_SCREEN, "bf16x3": rbmf.RBMF_GEMM_TCGEN05}
        strain_dev = torch.from_numpy(strain_np).to(device)
        strain_pinned = torch.from_numpy(strain_np).pin_memory()
        capacity = 1 << 22
        while True:
            # list capacities grow until one warm-up pass fits (dense banks give 1e6-1e7 records)
            plan = rbmf.Plan(cfg.N, cfg.fs, cfg.f_low, cfg.k, cfg.T, w=cfg.w, device=str(device), stream=stream,
                             max_candidates=capacity, max_triggers=capacity)
            plan.set_gemm_impl(impls[args.gemm])
            plan.set_basis(torch.from_numpy(wl["basis"]))
            plan.set_coeffs(torch.from_numpy(wl["coeffs"]), torch.from_numpy(wl["sigma"]))
            torch.cuda.empty_cache()
            for _ in range(args.warmup):
                plan.filter_async(strain_dev, cfg.thr1, cfg.thr2)
            stream.synchronize()
            nc, nt, st = plan.counts(allow_overflow=True)
            if st != rbmf.RBMF_ERR_OVERFLOW or capacity >= (1 << 26):
                break
            plan.close()
            capacity <<= 2
        # pinned host array for the trigger list (the end-to-end leg copies into it every step)
        out_pinned = torch.empty(plan.max_triggers * 4, dtype=torch.int32).pin_memory()
        out_host = out_pinned.numpy().view(rbmf.TRIGGER_DTYPE)
        plan.set_timing(True)
        sampler = ClockSampler(local_rank if "CUDA_VISIBLE_DEVICES" not in os.environ else
                               int(os.environ["CUDA_VISIBLE_DEVICES"].split(",")[local_rank]))
        rdist.barrier(device)
        torch.cuda.synchronize(device)
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        stage = {"fft": [], "gemm": [], "stage2": [], "total": []}
        t_wall0 = time.time()
        ev0.record(stream)
        for _ in range(args.steps):                   # the timed region: K steps back to back, no host sync inside
            plan.filter_async(strain_dev, cfg.thr1, cfg.thr2)
        ev1.record(stream)
        torch.cuda.synchronize(device)
        rdist.barrier(device)
        elapsed_ms = rdist.max_over_ranks(ev0.elapsed_time(ev1), device)
        # per-kernel durations: the same K steps again, reading the library's CUDA events after every step (this
        # costs a host round trip per step, which is why it is not done inside the region `value` comes from)
        for _ in range(args.steps):
            plan.filter_async(strain_dev, cfg.thr1, cfg.thr2)
            ms = plan.stage_ms()                      # waits for this step's last event, reads the stage events
            for key in stage:
                stage[key].append(ms[key])
        t_wall1 = time.time()
        clocks = sampler.summary(t_wall0, t_wall1)

        # ---- end-to-end leg: host strain in, host triggers out, every step
        for _ in range(2):
            plan.filter_host(strain_pinned.numpy(), cfg.thr1, cfg.thr2, out_host)
        rdist.barrier(device)
        torch.cuda.synchronize(device)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        n_e2e = 0
        for _ in range(args.steps):
            _, n_e2e = plan.filter_host(strain_pinned.numpy(), cfg.thr1, cfg.thr2, out_host)
        e1.record(stream)
        torch.cuda.synchronize(device)
        e2e_ms = rdist.max_over_ranks(e0.elapsed_time(e1), device)
        sampler.stop()

        # ---- the other tensor-core mode, per-stage only (context for `stages`; not part of `value`)
        other = {"screen": "bf16x3", "bf16x3": "screen"}.get(args.gemm)
        other_stage = None
        if other is not None:
            plan.set_gemm_impl(impls[other])
            acc = {"fft": [], "gemm": [], "stage2": [], "total": []}
            for i in range(3 + min(args.steps, 20)):
                plan.filter_async(strain_dev, cfg.thr1, cfg.thr2)
                ms = plan.stage_ms()
                if i >= 3:
                    for key in acc:
                        acc[key].append(ms[key])
            other_stage = {key + "_ms": statistics.mean(v) for key, v in acc.items()}
            plan.set_gemm_impl(impls[args.gemm])

    seg_seconds = cfg.N / cfg.fs
    ms_per_step = elapsed_ms / args.steps
    value = world * cfg.T * seg_seconds / (ms_per_step * 1e-3)
    e2e_value = world * cfg.T * seg_seconds / (e2e_ms / args.steps * 1e-3)

    if rank != 0:
        rdist.finalize()
        return 0

    # ---- rooflines: dominant kernel = the stage-1 GEMM
    peaks_path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(peaks_path):
        peaks = json.load(open(peaks_path))
        hbm_peak, tensor_peak, peak_src = peaks["hbm_gbs"], peaks["bf16_tflops_sustained"], "measured (sustained bf16)"
    else:
        hbm_peak, tensor_peak, peak_src = 6650.0, 1400.0, "fallback"
    gemm_ms = statistics.mean(stage["gemm"])
    fft_ms = statistics.mean(stage["fft"])
    s2_ms = statistics.mean(stage["stage2"])
    M = cfg.N // cfg.w
    useful_flops = 8.0 * cfg.T * cfg.k * M
    products = 1.0 if args.gemm == "screen" else 3.0         # tensor-core products executed per useful one
    executed_flops = products * useful_flops
    gemm_tflops = executed_flops / (gemm_ms * 1e-3) / 1e12
    band = cfg.N // 2 - cfg.j_low
    fft_alg_bytes = cfg.k * band * 8 + (cfg.N // 2 + 1) * 8 + cfg.k * cfg.N * 8 + cfg.k * M * 8
    fft_gbs = fft_alg_bytes / (fft_ms * 1e-3) / 1e9
    roofline = {"kernel": ("gemm_screen_pair_kernel" if args.gemm == "screen" else "gemm_tcgen05_kernel") + " (a4-a5)", "bound": "tensor", "achieved": gemm_tflops,
                "peak": tensor_peak, "unit": "TFLOP/s", "frac": gemm_tflops / tensor_peak,
                "traffic": NCU_TRAFFIC.get((args.config, cfg.w, args.gemm, "gemm")),
                "peak_source": peak_src, "flops_counted": "executed 16-bit MMA flops = %d x 8 T k N/w (%s)" % (
                    int(products), "one fp16 product: rigorous-bound screen, fp32 confirm in kernel 3"
                    if args.gemm == "screen" else "bf16x3 split precision"),
                "useful_tflops": useful_flops / (gemm_ms * 1e-3) / 1e12, "avg_kernel_ms": gemm_ms}
    stages = {"fft_ms": fft_ms, "gemm_ms": gemm_ms, "stage2_ms": s2_ms, "total_ms": statistics.mean(stage["total"]),
              "fft": {"bound": "hbm", "algorithmic_GBps": fft_gbs, "peak": hbm_peak, "frac": fft_gbs / hbm_peak,
                      "algorithmic_bytes": fft_alg_bytes,
                      "traffic": NCU_TRAFFIC.get((args.config, cfg.w, args.gemm, "fft"))},
              "n_candidates": nc, "n_triggers": nt, "gemm_mode": args.gemm, "list_capacity": capacity,
              "lists_overflowed": bool(nc > capacity or nt > capacity)}
    if other_stage is not None:
        stages["other_mode"] = dict(other_stage, gemm_mode=other)

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": ("f16 tensor-core screen with a rigorous error bound + f32 confirm/re-score + f32 FFT"
                      if args.gemm == "screen" else "bf16x3 (fp32-equivalent split bf16 on tensor cores) + f32"),
            "data": "synthetic", "config": config_desc, "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": (cfg.N // 2 + 1) * 8,
                    "d2h_bytes_per_step": 16 + int(min(n_e2e, plan.max_triggers)) * 16,
                    "ms_per_step": e2e_ms / args.steps},
            "gpu_launches": plan.launches_per_filter() * args.steps, "roofline": roofline, "stages": stages}

    if world == 1 and not args.no_cpu_baseline:
        tps = oracle_templates_per_step(cfg)
        v, ms, threads, sample = oracle_throughput(wl, tps, steps=6, warmup=1, time_budget_s=25.0)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample,
                                "ms_per_step": ms}
    print(json.dumps(line))
    plan.close()
    rdist.finalize()
    return 0


if __name__ == "__main__":
    sys.exit(main())
