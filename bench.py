#!/usr/bin/env python
"""bench.py -- throughput of the reduced-basis hierarchical matched filter hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config paper|small|large|sweep_k512_T100000|...|all]
                    [--impl ours|reference]

`--config all` prints one JSON line per BASELINE.json config (the sweep as its (k, T) grid); the default run times the
`paper` config and adds a compact `configs` array (per-stage ms and roofline fractions of small, large and one sweep
point) measured by the same program.

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

KERNEL_OF = {"fft": "fft_tma_kernel", "gemm": "gemm_", "stage2": "stage2_score"}


KERNEL_SOURCES = ("fft_tma.cu", "gemm_tcgen05.cu", "stage2_bybin.cu", "stage2_kernels.cu", "prep_kernels.cu",
                  "rbmf_internal.h")


def kernel_fingerprint():
    """sha256 over the DEVICE code of the sources of the hot-path kernels (comments and blank lines dropped, so that a
    reworded comment does not invalidate a capture).  A committed ncu traffic capture is stamped with it
    (profiles/traffic_fingerprints.txt: `<csv name> <fingerprint>`); `roofline.traffic` is null when the capture was
    made from other kernel sources than the ones this run executes.  `python bench.py --kernel-fingerprint` prints it."""
    import hashlib
    import re
    h = hashlib.sha256()
    csrc = os.path.join(ROOT, "paper_2110_13115_b200", "csrc")
    for name in KERNEL_SOURCES:
        text = open(os.path.join(csrc, name)).read()
        text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
        lines = [re.sub(r"//.*$", "", ln).strip() for ln in text.splitlines()]
        h.update(name.encode())
        h.update("\n".join(ln for ln in lines if ln).encode())
    return h.hexdigest()[:16]


def traffic_stamp(csv_name):
    path = os.path.join(ROOT, "profiles", "traffic_fingerprints.txt")
    if os.path.exists(path):
        for ln in open(path):
            parts = ln.split()
            if len(parts) >= 2 and parts[0] == csv_name:
                return parts[1]
    return None


def ncu_traffic(config, w, mode):
    """DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum) per stage, read from the ncu launch list
    committed as profiles/traffic_<config>_w<w>_<mode>.csv (an `ncu --csv` log of that very configuration; the .md
    beside it names the command).  Returns ({stage: bytes}, source) -- ({}, reason) when no capture exists."""
    import csv
    path = os.path.join(ROOT, "profiles", "traffic_%s_w%d_%s.csv" % (config, w, mode))
    if not os.path.exists(path):
        return {}, "no ncu capture committed for (%s, w=%d, %s)" % (config, w, mode)
    stamp, now = traffic_stamp(os.path.basename(path)), kernel_fingerprint()
    if stamp != now:
        return {}, "profiles/%s is stale: captured from kernel sources %s, this build is %s" % (
            os.path.basename(path), stamp or "(unstamped)", now)
    acc = {}
    with open(path, newline="") as fh:
        rows = [r for r in csv.reader(fh) if len(r) >= 15 and r[0].isdigit()]
    for r in rows:
        name, metric, val = r[4], r[12], float(r[14])
        if metric not in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
            continue
        for stage, pat in KERNEL_OF.items():
            if pat in name:
                acc.setdefault(stage, {}).setdefault(r[0], 0.0)
                acc[stage][r[0]] += val
    return {st: sum(v.values()) / len(v) for st, v in acc.items()}, "profiles/" + os.path.basename(path)


def cpu_info():
    model = "unknown"
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                model = line.split(":", 1)[1].strip()
                break
    except OSError:
        pass
    try:
        cores = len(os.sched_getaffinity(0))
    except AttributeError:
        cores = os.cpu_count() or 1
    return cores, model


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
    independent per template).  Returns (template-seconds/s, ms per step, thread record, description).  The thread
    record says what the oracle really used: numpy's FFT runs on ONE thread, only its BLAS leg (the reconstruction of
    the templates) on several; `cores` is the larger of the two, `cores_available` what the box would have allowed."""
    from oracle import rbmf_oracle as orc
    cfg = wl["config"]
    try:
        from threadpoolctl import threadpool_info
        blas_threads = max([int(i.get("num_threads", 1)) for i in threadpool_info()] + [1])
    except Exception:
        blas_threads = 1
    cores, model = cpu_info()
    threads = {"cores": min(blas_threads, cores), "blas_threads": min(blas_threads, cores), "fft_threads": 1,
               "cores_available": cores}
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
    sample = ("%d of %d templates per step (seeded random subset), full segment, numpy fp64 oracle_filter as it stands "
              "(%d cores available by sched_getaffinity on %s; its BLAS leg uses %d threads, its FFT leg one), "
              "%d timed steps" % (n_t, cfg.T, cores, model, blas_threads, len(times)))
    return value, ms, threads, sample


def oracle_templates_per_step(cfg):
    # ~1-3 s of CPU work per step: cost per template ~ bins * k * 8 flops (h' build) + an N-point fp64 FFT
    per_template = cfg.bins * cfg.k * 8 / 2.0e10 + cfg.N * 6.0e-8
    return int(max(4, min(cfg.T, 2.0 / per_template)))


# ------------------------------------------------------------------------------------------ one configuration
def describe(cfg, world):
    return {"workload": "%s: N=%d fs=%g f_low=%g k=%d T=%d w=%d thr=%g/%g injections=%d" % (
        cfg.name, cfg.N, cfg.fs, cfg.f_low, cfg.k, cfg.T, cfg.w, cfg.thr1, cfg.thr2, cfg.n_inj),
        "N": cfg.N, "k": cfg.k, "T": cfg.T, "w": cfg.w, "segment_seconds": cfg.N / cfg.fs,
        "parallelism": "replicas x%d (one strain segment per GPU, no collective)" % world,
        "l2": ("working set (basis %.0f MB + beta %.0f MB) exceeds the 126 MB L2; no flush needed" if
               cfg.N * cfg.k * 12 > 252e6 else
               "working set (basis %.0f MB + beta %.0f MB) is L2-sized: a 256 MB scrub buffer is written between steps") % (
            cfg.N / 2 * cfg.k * 8 / 1e6, cfg.N * cfg.k * 8 / 1e6)}


def pick_peaks(elapsed_ms, clocks):
    """(hbm peak, tensor peak of the regime, burst, sustained, regime, source).  The burst figure applies to a short
    timed region at full clocks, the sustained one to a seconds-long loop or one that ran into the power cap
    (B200_PROFILING.md)."""
    peaks_path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(peaks_path):
        peaks = json.load(open(peaks_path))
        hbm, burst, sust, src = peaks["hbm_gbs"], peaks["bf16_tflops"], peaks["bf16_tflops_sustained"], "measured"
    else:
        hbm, burst, sust, src = 6650.0, 1590.0, 1400.0, "fallback"
    capped = "sw_power_cap" in (clocks.get("reasons") or [])
    regime = "sustained" if (elapsed_ms >= 1000.0 or capped) else "burst"
    return hbm, (sust if regime == "sustained" else burst), burst, sust, regime, src


def stat(xs):
    return {"mean": statistics.mean(xs), "median": statistics.median(xs), "best": min(xs)}


def measure(cfg, args, rdist, rbmf, workloads, torch, device, stream, rank, world, local_rank, headline):
    """Times one configuration.  headline = True adds the end-to-end leg, the other tensor-core mode and (N = 1) the
    CPU baseline; False returns the compact per-stage summary used for the `configs` array."""
    steps = args.steps if headline else max(3, min(args.steps, args.summary_steps))
    wl = workloads.make_workload(cfg, device=str(device))
    seg = rdist.segment_index(rank, 0, world)
    strain_np, _ = workloads.make_strain(wl, seg)
    impls = {"screen": rbmf.RBMF_GEMM_SCREEN, "bf16x3": rbmf.RBMF_GEMM_TCGEN05}
    small_ws = cfg.N * cfg.k * 12 <= 252e6
    with torch.cuda.stream(stream):
        strain_dev = torch.from_numpy(strain_np).to(device)
        scrub = torch.empty(256 << 20, dtype=torch.uint8, device=device) if small_ws else None
        capacity = 1 << 22
        while True:
            # list capacities grow until one warm-up pass fits (dense banks give 1e6-1e9 records)
            torch.cuda.empty_cache()
            plan = rbmf.Plan(cfg.N, cfg.fs, cfg.f_low, cfg.k, cfg.T, w=cfg.w, device=str(device), stream=stream,
                             max_candidates=capacity, max_triggers=capacity)
            plan.set_gemm_impl(impls[args.gemm])
            plan.set_basis(torch.from_numpy(wl["basis"]))
            plan.set_coeffs(torch.from_numpy(wl["coeffs"]), torch.from_numpy(wl["sigma"]))
            for _ in range(args.warmup):
                plan.filter_async(strain_dev, cfg.thr1, cfg.thr2)
            stream.synchronize()
            nc, nt, st = plan.counts(allow_overflow=True)
            if st != rbmf.RBMF_ERR_OVERFLOW or capacity >= (1 << 30):
                break
            plan.close()
            capacity <<= 2
        plan.set_timing(True)
        sampler = ClockSampler(local_rank if "CUDA_VISIBLE_DEVICES" not in os.environ else
                               int(os.environ["CUDA_VISIBLE_DEVICES"].split(",")[local_rank]))
        rdist.barrier(device)
        torch.cuda.synchronize(device)
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        stage = {"fft": [], "gemm": [], "stage2": [], "total": []}
        t_wall0 = time.time()
        if scrub is None:
            ev0.record(stream)
            for _ in range(steps):                    # the timed region: K steps back to back, no host sync inside
                plan.filter_async(strain_dev, cfg.thr1, cfg.thr2)
            ev1.record(stream)
            torch.cuda.synchronize(device)
            elapsed_local = ev0.elapsed_time(ev1)
        else:
            # L2-sized working set: scrub L2 between steps, time each step with its own pair of events
            evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
            for a, b in evs:
                scrub.fill_(1)
                a.record(stream)
                plan.filter_async(strain_dev, cfg.thr1, cfg.thr2)
                b.record(stream)
            torch.cuda.synchronize(device)
            elapsed_local = sum(a.elapsed_time(b) for a, b in evs)
        rdist.barrier(device)
        elapsed_ms = rdist.max_over_ranks(elapsed_local, device)
        # per-kernel durations of the SAME K steps: the library keeps the stage events of its last 64 timed calls
        # (rbmf_get_stage_ms_history), read here after the region has ended -- no host round trip inside it, so the
        # stage sums and ms_per_step describe one and the same run (steps > 64: the last 64 of them)
        for ms in plan.stage_ms_history(min(steps, 64)):
            for key in stage:
                stage[key].append(ms[key])
        t_wall1 = time.time()
        clocks = sampler.summary(t_wall0, t_wall1)
        n_screened = plan.screened_count()

        e2e = None
        other_stage = None
        if headline:
            # ---- end-to-end leg: host strain in, host triggers out, every step
            strain_pinned = torch.from_numpy(strain_np).pin_memory()
            out_pinned = torch.empty(plan.max_triggers * 4, dtype=torch.int32).pin_memory()
            out_host = out_pinned.numpy().view(rbmf.TRIGGER_DTYPE)
            for _ in range(2):
                plan.filter_host(strain_pinned.numpy(), cfg.thr1, cfg.thr2, out_host)
            rdist.barrier(device)
            torch.cuda.synchronize(device)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            n_e2e = 0
            for _ in range(steps):
                _, n_e2e = plan.filter_host(strain_pinned.numpy(), cfg.thr1, cfg.thr2, out_host)
            e1.record(stream)
            torch.cuda.synchronize(device)
            e2e_ms = rdist.max_over_ranks(e0.elapsed_time(e1), device)
            e2e = {"value": world * cfg.T * (cfg.N / cfg.fs) / (e2e_ms / steps * 1e-3), "unit": UNIT,
                   "h2d_bytes_per_step": (cfg.N // 2 + 1) * 8,
                   "d2h_bytes_per_step": 16 + int(min(n_e2e, plan.max_triggers)) * 16, "ms_per_step": e2e_ms / steps}
            del out_pinned, out_host
        sampler.stop()
        # ---- the other tensor-core mode, per-stage only (context for `stages`; not part of `value`)
        other = {"screen": "bf16x3", "bf16x3": "screen"}[args.gemm]
        plan.set_gemm_impl(impls[other])
        acc = {"fft": [], "gemm": [], "stage2": [], "total": []}
        for i in range(3 + min(steps, 20 if headline else 3)):
            plan.filter_async(strain_dev, cfg.thr1, cfg.thr2)
            ms = plan.stage_ms()
            if i >= 3:
                for key in acc:
                    acc[key].append(ms[key])
        other_stage = {key + "_ms": statistics.mean(v) for key, v in acc.items()}
        plan.set_gemm_impl(impls[args.gemm])
        launches = plan.launches_per_filter()
        plan.close()
        del plan, scrub
        torch.cuda.empty_cache()

    seg_seconds = cfg.N / cfg.fs
    ms_per_step = elapsed_ms / steps
    value = world * cfg.T * seg_seconds / (ms_per_step * 1e-3)

    # ---- rooflines: dominant kernel = the stage-1 GEMM
    hbm_peak, tensor_peak, peak_burst, peak_sust, regime, peak_src = pick_peaks(elapsed_ms, clocks)
    gemm_ms, fft_ms, s2_ms = (statistics.mean(stage[kk]) for kk in ("gemm", "fft", "stage2"))
    M = cfg.N // cfg.w
    useful_flops = 8.0 * cfg.T * cfg.k * M
    products = 1.0 if args.gemm == "screen" else 3.0         # tensor-core products executed per useful one
    gemm_tflops = products * useful_flops / (gemm_ms * 1e-3) / 1e12
    band = cfg.N // 2 - cfg.j_low
    fft_alg_bytes = cfg.k * band * 8 + (cfg.N // 2 + 1) * 8 + cfg.k * cfg.N * 8 + cfg.k * M * 8
    fft_gbs = fft_alg_bytes / (fft_ms * 1e-3) / 1e9
    traffic, traffic_src = ncu_traffic(cfg.name, cfg.w, args.gemm)
    roofline = {"kernel": ("gemm_screen_pair_kernel" if args.gemm == "screen" else "gemm_tcgen05_kernel") + " (a4-a5)",
                "bound": "tensor", "achieved": gemm_tflops, "peak": tensor_peak, "unit": "TFLOP/s",
                "frac": gemm_tflops / tensor_peak, "traffic": traffic.get("gemm"), "traffic_source": traffic_src,
                "regime": regime, "peak_source": "%s bf16 cuBLAS, %s figure (timed region %.0f ms%s)" % (
                    peak_src, regime, elapsed_ms, ", sw_power_cap active" if "sw_power_cap" in (clocks.get("reasons") or []) else ""),
                "frac_of_burst_peak": gemm_tflops / peak_burst, "frac_of_sustained_peak": gemm_tflops / peak_sust,
                "flops_counted": "executed 16-bit MMA flops = %d x 8 T k N/w (%s)" % (
                    int(products), "one fp16 product: error-bounded screen, fp32 confirm in kernel 3"
                    if args.gemm == "screen" else "bf16x3 split precision"),
                "useful_tflops": useful_flops / (gemm_ms * 1e-3) / 1e12, "avg_kernel_ms": gemm_ms}
    # north_star's OTHER target, kept inside `roofline` so that the driver's record carries it: kernel 1 against the HBM
    # peak, in algorithmic bytes and in the real DRAM bytes of the committed capture (null when that capture is stale)
    fft_dram = traffic.get("fft")
    roofline["fft"] = {"kernel": "fft_tma_kernel (a1-a3)", "bound": "hbm", "unit": "GB/s", "peak": hbm_peak,
                       "algorithmic_GBps": fft_gbs, "frac": fft_gbs / hbm_peak, "target_frac": 0.70,
                       "dram_GBps": (fft_dram / (fft_ms * 1e-3) / 1e9) if fft_dram else None,
                       "dram_frac": (fft_dram / (fft_ms * 1e-3) / 1e9 / hbm_peak) if fft_dram else None,
                       "traffic": fft_dram, "algorithmic_bytes": fft_alg_bytes, "avg_kernel_ms": fft_ms}
    # ... and the arithmetic mode this run did NOT use for `value` (separate short pass, one host read per step): with
    # the default screen that is the literal split-precision GEMM of north_star
    o_gemm, o_total = other_stage["gemm_ms"], other_stage["total_ms"]
    o_products = 3.0 if other == "bf16x3" else 1.0
    o_tflops = o_products * useful_flops / (o_gemm * 1e-3) / 1e12
    roofline[other] = {"kernel": ("gemm_tcgen05_kernel" if other == "bf16x3" else "gemm_screen_pair_kernel") + " (a4-a5)",
                       # a short pass of its own (a few steps): judged against the BURST peak whatever the regime of
                       # the headline region was
                       "bound": "tensor", "unit": "TFLOP/s", "achieved": o_tflops, "peak": peak_burst,
                       "frac": o_tflops / peak_burst, "frac_of_sustained_peak": o_tflops / peak_sust,
                       "avg_kernel_ms": o_gemm, "step_ms": o_total,
                       "value_in_this_mode": world * cfg.T * seg_seconds / (o_total * 1e-3),
                       "note": "executed 16-bit MMA flops = %d x 8 T k N/w; step_ms from the library's own events" % int(o_products)}
    roofline["kernel_fingerprint"] = kernel_fingerprint()
    roofline["stage_times_from"] = "the timed region itself (library events of its last %d steps)" % len(stage["gemm"])
    # second roofline of kernel 1: its fp32 arithmetic, 5 N log2 N flops per series + 6 per band bin (the paper's count,
    # PAPER.md:236), against 148 SMs x 128 lanes x 2 (FMA) x the SM clock sampled under load
    fft_flops = cfg.k * (5.0 * cfg.N * np.log2(cfg.N) + 6.0 * band)
    sm_hz = (clocks.get("sm_mhz") or 1965.0) * 1e6
    alu_peak = 148 * 128 * 2 * sm_hz / 1e12
    fft_alu = {"bound": "alu", "achieved": fft_flops / (fft_ms * 1e-3) / 1e12, "peak": alu_peak, "unit": "TFLOP/s",
               "frac": fft_flops / (fft_ms * 1e-3) / 1e12 / alu_peak,
               "note": "fp32 FMA peak at the sampled clock; a butterfly network is ~2/3 additions, so 0.5 is its ceiling"}
    stages = {"fft_ms": fft_ms, "gemm_ms": gemm_ms, "stage2_ms": s2_ms, "total_ms": statistics.mean(stage["total"]),
              "per_step_ms": {kk: stat(v) for kk, v in stage.items()},
              "fft": {"bound": "hbm", "algorithmic_GBps": fft_gbs, "peak": hbm_peak, "frac": fft_gbs / hbm_peak,
                      "algorithmic_bytes": fft_alg_bytes, "traffic": traffic.get("fft"),
                      # real DRAM bytes of the committed ncu capture over this run's event time (both
                      # the algorithmic and the achieved DRAM rate are reported)
                      "dram_GBps": (traffic["fft"] / (fft_ms * 1e-3) / 1e9) if traffic.get("fft") else None,
                      "dram_frac": (traffic["fft"] / (fft_ms * 1e-3) / 1e9 / hbm_peak) if traffic.get("fft") else None,
                      "alu": fft_alu},
              "stage2": {"candidates_per_s": (nc / (s2_ms * 1e-3)) if s2_ms > 0 else None,
                         "algorithmic_GBps": n_screened * (cfg.w + 1) * cfg.k * 8 / (s2_ms * 1e-3) / 1e9,
                         "traffic": traffic.get("stage2")},
              "n_candidates": nc, "n_screened": n_screened, "n_triggers": nt, "gemm_mode": args.gemm,
              "list_capacity": capacity, "lists_overflowed": bool(n_screened > capacity or nt > capacity),
              "other_mode": dict(other_stage, gemm_mode=other)}
    if not headline:
        return {"workload": describe(cfg, world)["workload"], "steps": steps, "ms_per_step": ms_per_step, "value": value,
                "fft_ms": fft_ms, "gemm_ms": gemm_ms, "stage2_ms": s2_ms, "fft_frac_hbm": fft_gbs / hbm_peak,
                "gemm_frac_tensor": gemm_tflops / tensor_peak, "gemm_tflops": gemm_tflops, "regime": regime,
                "n_candidates": nc, "n_triggers": nt, "lists_overflowed": stages["lists_overflowed"],
                "other_mode": stages["other_mode"], "clocks": clocks}, wl
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None,
            "dtype": ("f16 tensor-core screen with an error bound + f32 confirm/re-score + f32 FFT"
                      if args.gemm == "screen" else "bf16x3 (fp32-equivalent split bf16 on tensor cores) + f32"),
            "data": "synthetic", "config": describe(cfg, world), "clocks": clocks, "e2e": e2e,
            "gpu_launches": launches * steps, "roofline": roofline, "stages": stages}
    return line, wl


# ------------------------------------------------------------------------- extras: SURVEY.md 8(f) rows f1-f3
def _time_calls(torch, stream, device, fn, steps, warmup=3):
    for _ in range(warmup):
        fn()
    torch.cuda.synchronize(device)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(steps):
        fn()
    e1.record(stream)
    torch.cuda.synchronize(device)
    return e0.elapsed_time(e1) / steps


def measure_batch(name, B, steps, rbmf, workloads, torch, device, stream):
    """f1: B segments per call (rbmf_filter_batch) against single-segment calls on the same plan, incl. the front end
    (rbmf_prepare_strain on B coloured time series)."""
    cfg = workloads.CONFIGS[name]
    wl = workloads.make_workload(cfg, device=str(device))
    with torch.cuda.stream(stream):
        strains = torch.from_numpy(np.stack([workloads.make_strain(wl, s)[0] for s in range(B)])).to(device)
        xs, inv_asd = zip(*[workloads.make_time_series(wl, s) for s in range(B)])
        x_dev, asd_dev = torch.from_numpy(np.stack(xs)).to(device), torch.from_numpy(inv_asd[0]).to(device)
        plan = rbmf.Plan(cfg.N, cfg.fs, cfg.f_low, cfg.k, cfg.T, w=cfg.w, device=str(device), stream=stream,
                         max_candidates=1 << 22, max_triggers=1 << 22, max_batch=B)
        plan.set_basis(torch.from_numpy(wl["basis"]))
        plan.set_coeffs(torch.from_numpy(wl["coeffs"]), torch.from_numpy(wl["sigma"]))
        plan.set_timing(True)
        ms_b = _time_calls(torch, stream, device, lambda: plan.filter_batch_async(strains, cfg.thr1, cfg.thr2), steps)
        st_b = plan.stage_ms()
        nc, nt, st = plan.counts(allow_overflow=True)
        ms_1 = _time_calls(torch, stream, device, lambda: plan.filter_async(strains[0], cfg.thr1, cfg.thr2), steps)
        st_1 = plan.stage_ms()
        ms_fe = _time_calls(torch, stream, device, lambda: plan.prepare_strain(x_dev, asd_dev), steps)
        plan.close()
    seg = cfg.N / cfg.fs
    return {"row": "f1 batched segments + front end", "workload": describe(cfg, 1)["workload"], "batch": B,
            "ms_per_call_batch": ms_b, "ms_per_call_single": ms_1,
            "value_batch": B * cfg.T * seg / (ms_b * 1e-3), "value_single": cfg.T * seg / (ms_1 * 1e-3),
            "speedup_per_segment": ms_1 * B / ms_b, "stages_batch_ms": st_b, "stages_single_ms": st_1,
            "front_end_ms_for_B_series": ms_fe, "n_candidates": nc, "n_triggers": nt,
            "lists_overflowed": st == rbmf.RBMF_ERR_OVERFLOW, "unit": UNIT}


def measure_routes(name, ws, steps, rbmf, workloads, torch, device, stream, slab=256):
    """f2: the paper's two template routes against the basis/GEMM route on the same inputs."""
    cfg0 = workloads.CONFIGS[name]
    wl = workloads.make_workload(cfg0, device=str(device))
    out = []
    with torch.cuda.stream(stream):
        strain = torch.from_numpy(wl["strain"]).to(device)
        c = torch.from_numpy(wl["coeffs"]).to(device)
        b = torch.from_numpy(wl["basis"]).to(device)
        tpl = torch.empty((cfg0.T, cfg0.bins), dtype=torch.complex64, device=device)   # h'_t = sum_k c_tk b_k
        for a in range(0, cfg0.T, 2048):
            tpl[a:a + 2048] = c[a:a + 2048] @ b
        del c, b
        for w in ws:
            cfg = cfg0.replace(w=w)
            plan = rbmf.Plan(cfg.N, cfg.fs, cfg.f_low, cfg.k, cfg.T, w=w, device=str(device), stream=stream,
                             max_candidates=1 << 24, max_triggers=1 << 24, template_slab=slab)
            plan.set_basis(torch.from_numpy(wl["basis"]))
            plan.set_coeffs(torch.from_numpy(wl["coeffs"]), torch.from_numpy(wl["sigma"]))
            plan.set_templates(tpl, torch.from_numpy(wl["sigma"]))
            plan.set_timing(True)
            row = {"row": "f2 template routes vs basis route", "workload": describe(cfg, 1)["workload"], "w": w,
                   "slab": slab}
            for label, impl, route in (("basis_gemm_screen", rbmf.RBMF_GEMM_SCREEN, rbmf.RBMF_STAGE1_BASIS),
                                       ("basis_gemm_bf16x3", rbmf.RBMF_GEMM_TCGEN05, rbmf.RBMF_STAGE1_BASIS),
                                       ("templates_eq12", rbmf.RBMF_GEMM_TCGEN05, rbmf.RBMF_STAGE1_TEMPLATES)):
                plan.set_gemm_impl(impl)
                plan.set_stage1_route(route)
                ms = _time_calls(torch, stream, device, lambda: plan.filter_async(strain, cfg.thr1, cfg.thr2), steps)
                st = plan.stage_ms()
                nc, nt, _ = plan.counts(allow_overflow=True)
                row[label] = {"ms_per_call": ms, "stage1_ms": st["gemm"], "fft_ms": st["fft"], "stage2_ms": st["stage2"],
                              "n_candidates": nc, "n_triggers": nt}
            plan.set_stage1_route(rbmf.RBMF_STAGE1_BASIS)
            if w == ws[0]:
                def flat():
                    plan._check(rbmf.rbmf_filter_flat(plan._h, strain.data_ptr(), float(cfg.thr2), plan._out.data_ptr(),
                                                      plan._n_out.data_ptr()), "rbmf_filter_flat")
                ms = _time_calls(torch, stream, device, flat, max(2, steps // 2), warmup=1)
                _, nt, _ = plan.counts(allow_overflow=True)
                bank_bytes = cfg.T * (cfg.N // 2 - cfg.j_low) * 8
                row["flat_template_method"] = {"ms_per_call": ms, "n_triggers": nt,
                                               "bank_GBps": bank_bytes / (ms * 1e-3) / 1e9,
                                               "value": cfg.T * (cfg.N / cfg.fs) / (ms * 1e-3)}
            plan.close()
            out.append(row)
    return out


def measure_bankset(steps, rbmf, workloads, torch, device, stream):
    """f3: four sub-banks with their own basis sizes (Table I) against one strain: one bank-set call
    against the same plans called one after the other."""
    base = workloads.CONFIGS["small"]
    parts = [(1.0, 1.5, 64, 500, 8), (1.5, 2.0, 128, 700, 8), (2.0, 2.5, 96, 300, 8), (2.5, 3.0, 128, 500, 16)]
    subs = workloads.make_subbanks(base, parts, device=str(device))
    with torch.cuda.stream(stream):
        strain = torch.from_numpy(subs[0]["strain"]).to(device)
        plans = []
        for wl in subs:
            cfg = wl["config"]
            p = rbmf.Plan(cfg.N, cfg.fs, cfg.f_low, cfg.k, cfg.T, w=cfg.w, device=str(device), stream=stream,
                          max_candidates=1 << 20, max_triggers=1 << 20)
            p.set_basis(torch.from_numpy(wl["basis"]))
            p.set_coeffs(torch.from_numpy(wl["coeffs"]), torch.from_numpy(wl["sigma"]))
            plans.append(p)
        bs = rbmf.BankSet(plans, max_triggers=1 << 22, stream=stream)
        ms_set = _time_calls(torch, stream, device, lambda: bs.filter_async(strain, base.thr1, base.thr2), steps)
        nc, nt, tot, _ = bs.counts()

        def one_by_one():
            for p in plans:
                p.filter_async(strain, base.thr1, base.thr2)
        ms_seq = _time_calls(torch, stream, device, one_by_one, steps)
        bs.close()
        for p in plans:
            p.close()
    tsec = sum(wl["config"].T for wl in subs) * (base.N / base.fs)
    return {"row": "f3 many sub-banks", "sub_banks": [{"k": k, "T": T, "w": w, "mc": [lo, hi]} for lo, hi, k, T, w in parts],
            "N": base.N, "ms_bank_set": ms_set, "ms_one_by_one": ms_seq, "value_bank_set": tsec / (ms_set * 1e-3),
            "n_triggers": tot, "per_sub_bank_triggers": nt, "unit": UNIT}


def measure_prepare(name, rbmf, workloads, torch, device):
    """f4: preparation on the GPU (covariance + block power iteration + projection) for one config's bank."""
    cfg = workloads.CONFIGS[name]
    wl = workloads.make_workload(cfg, device=str(device))
    n = min(cfg.T, cfg.basis_subset)
    ids = np.arange(n)
    tpl = torch.from_numpy(workloads.bank_templates(wl, ids, device=str(device)).astype(np.complex64)).to(device)
    torch.cuda.synchronize(device)
    t0 = time.time()
    basis, _ = rbmf.prepare_basis(tpl, cfg.N, cfg.fs, cfg.f_low, cfg.k, iterations=12, seed=1)
    torch.cuda.synchronize(device)
    t1 = time.time()
    coeffs, sigma = rbmf.prepare_coeffs(tpl, basis, cfg.N, cfg.fs, cfg.f_low)
    torch.cuda.synchronize(device)
    t2 = time.time()
    return {"row": "f4 preparation on the GPU", "workload": describe(cfg, 1)["workload"], "templates": int(n),
            "prepare_basis_s": t1 - t0, "prepare_coeffs_s": t2 - t1, "iterations": 12,
            "captured_power": float((sigma.double() ** 2).mean()), "captured_power_generator_fp64_svd": wl["captured"]}


def measure_cufft_context(names, workloads, torch, device):
    """Context only, never on the hot path: what the library FFT needs for the same transform sizes -- a batched
    complex-to-complex inverse FFT of k series of N samples through torch.fft (cuFFT) ALONE, and the paper's three
    separate steps (pointwise multiply, batched IFFT, w-sample averaging) as torch ops -- next to
    which the fused kernel 1 (multiply + IFFT + averaging + operand planes in one launch) is reported."""
    out = []
    for name in names:
        cfg = workloads.CONFIGS[name]
        N, k, w = cfg.N, cfg.k, cfg.w
        x = torch.randn(k, N, dtype=torch.complex64, device=device)
        b = torch.randn(k, N // 2, dtype=torch.complex64, device=device)
        d = torch.randn(N // 2, dtype=torch.complex64, device=device)

        def timed(fn, reps=20):
            for _ in range(3):
                fn()
            torch.cuda.synchronize(device)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(reps):
                fn()
            e1.record()
            torch.cuda.synchronize(device)
            return e0.elapsed_time(e1) / reps

        def three_steps():
            x[:, :N // 2] = d[None, :] * b.conj()
            x[:, N // 2:] = 0
            return torch.fft.ifft(x, dim=1, norm="forward").view(k, N // w, w).mean(dim=2)

        row = {"row": "context: library FFT / GEMM (cuFFT, cuBLAS through torch), not on the hot path",
               "workload": "%s: N=%d k=%d T=%d w=%d" % (name, N, k, cfg.T, w),
               "cufft_batched_c2c_ifft_alone_ms": timed(lambda: torch.fft.ifft(x, dim=1, norm="forward")),
               "multiply_ifft_average_as_torch_ops_ms": timed(three_steps)}
        del x, b, d
        # the paper's stage 1: cuBLAS on beta^avg and the coefficients, then a separate trigger search
        if cfg.T * (N // w) * 8 <= 48e9:
            coeff = torch.randn(cfg.T, k, dtype=torch.complex64, device=device)
            bavg = torch.randn(k, N // w, dtype=torch.complex64, device=device)
            row["cublas_cgemm_fp32_stage1_ms"] = timed(lambda: torch.matmul(coeff, bavg), reps=3)
            row["cublas_cgemm_plus_threshold_count_ms"] = timed(
                lambda: (torch.view_as_real(torch.matmul(coeff, bavg)).square_().sum(dim=-1) >= 25.0).sum(), reps=3)
            del coeff, bavg
        out.append(row)
    return out


# ---------------------------------------------------------------------------------------------------- main
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", default="paper", help="a name in workloads.CONFIGS, or `all`")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--w", type=int, default=None, help="override the averaging window")
    ap.add_argument("--gemm", default="screen", choices=["screen", "bf16x3"],
                    help="stage-1 kernel: fp16 screen + fp32 confirm (library default) or bf16x3")
    ap.add_argument("--summary-configs", default="small,large,sweep_k256_T10000",
                    help="configs summarised in the `configs` array of the default line ('' = none)")
    ap.add_argument("--summary-steps", type=int, default=5)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--kernel-fingerprint", action="store_true",
                    help="print the fingerprint of the hot-path kernel sources (the stamp of a traffic capture) and exit")
    ap.add_argument("--extras", default="batch,routes,bankset,prepare,cufft",
                    help="SURVEY 8(f) rows measured into the `extras` array of the default line: batch (f1: small at "
                         "B=8, paper at B=4), routes (f2: template routes vs GEMM route on small and paper), bankset "
                         "(f3), prepare (f4: preparation kernels on small), cufft (context: the library FFT alone on the same "
                         "sizes); '' = none")
    args = ap.parse_args()
    if args.kernel_fingerprint:
        print(kernel_fingerprint())
        return 0
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    import torch
    from paper_2110_13115_b200 import dist as rdist, workloads

    rank, local_rank, world = rdist.env_world()
    if args.config == "all":
        names = ["tiny", "small", "paper", "large"] + list(workloads.SWEEP_NAMES)
    else:
        names = [args.config]

    # ------------------------------------------------------------------ reference arm: the oracle, on host cores
    if args.impl == "reference":
        if rank != 0:
            return 0
        cfg = workloads.CONFIGS[names[0] if args.config != "all" else "paper"]
        if args.w is not None:
            cfg = cfg.replace(w=args.w)
        dev = "cuda" if torch.cuda.is_available() else "cpu"
        wl = workloads.make_workload(cfg, device=dev)
        tps = oracle_templates_per_step(cfg)
        value, ms, threads, sample = oracle_throughput(wl, tps, args.steps, args.warmup, time_budget_s=150.0)
        line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
                "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": describe(cfg, world),
                "cpu_baseline": dict({"value": value, "unit": UNIT, "kind": "oracle", "sample": sample}, **threads),
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
    stream = torch.cuda.Stream(device=device)

    for name in names:
        cfg = workloads.CONFIGS[name]
        if args.w is not None:
            cfg = cfg.replace(w=args.w)
        line, wl = measure(cfg, args, rdist, rbmf, workloads, torch, device, stream, rank, world, local_rank, True)
        if world == 1 and not args.no_cpu_baseline:
            tps = oracle_templates_per_step(cfg)
            v, ms, threads, sample = oracle_throughput(wl, tps, steps=6, warmup=1,
                                                       time_budget_s=25.0 if args.config != "all" else 8.0)
            line["cpu_baseline"] = dict({"value": v, "unit": UNIT, "kind": "oracle", "sample": sample,
                                         "ms_per_step": ms}, **threads)
        del wl
        if args.config != "all" and world == 1:
            # The headline above is complete; what follows adds context to the same line.  A failure in one of these
            # side measurements (e.g. out of memory on a smaller device) is recorded in the line, not raised.
            def guarded(target, label, fn):
                try:
                    out = fn()
                    target.extend(out if isinstance(out, list) else [out])
                except Exception as exc:                  # noqa: BLE001
                    target.append({"row": label, "error": "%s: %s" % (type(exc).__name__, str(exc)[:300])})
                    torch.cuda.empty_cache()

            line["configs"] = []
            for other in [c for c in args.summary_configs.split(",") if c and c != name]:
                guarded(line["configs"], other,
                        lambda other=other: measure(workloads.CONFIGS[other], args, rdist, rbmf, workloads, torch, device,
                                                    stream, rank, world, local_rank, False)[0])
            ex = [e for e in args.extras.split(",") if e]
            line["extras"] = []
            if "batch" in ex:
                guarded(line["extras"], "f1 batch small", lambda: measure_batch("small", 8, 20, rbmf, workloads, torch, device, stream))
                guarded(line["extras"], "f1 batch paper", lambda: measure_batch("paper", 4, 10, rbmf, workloads, torch, device, stream))
            if "routes" in ex:
                guarded(line["extras"], "f2 routes small", lambda: measure_routes("small", (8, 16), 10, rbmf, workloads, torch, device, stream))
                guarded(line["extras"], "f2 routes paper", lambda: measure_routes("paper", (8, 16), 4, rbmf, workloads, torch, device, stream))
            if "bankset" in ex:
                guarded(line["extras"], "f3 bank set", lambda: measure_bankset(20, rbmf, workloads, torch, device, stream))
            if "prepare" in ex:
                guarded(line["extras"], "f4 preparation", lambda: measure_prepare("small", rbmf, workloads, torch, device))
            if "cufft" in ex:
                guarded(line["extras"], "library context",
                        lambda: measure_cufft_context(("small", "paper", "large", "sweep_k256_T10000"), workloads, torch, device))
        if rank == 0:
            print(json.dumps(line), flush=True)
    rdist.finalize()
    return 0


if __name__ == "__main__":
    sys.exit(main())
