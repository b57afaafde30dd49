"""The (w, rho_I) tuning study of the paper on the GPU path.

For averaging windows w and first-stage thresholds rho_I this measures, on the caller's strain segments,

  f(w, rho_I)        first-stage triggers per template and per second of data (Fig. 5),
  n_final(rho_II)    hierarchical triggers with |rho| >= rho_II, against n_flat(rho_II) of the flat search (w = 1),
  rho_target         Eq. 16: the smallest rho_II from which the hierarchical search keeps >= `ratio` of the flat triggers
                     (Fig. 6),
  cost               Eq. 15 normalised by Eq. 13 with the measured f (Fig. 7; log base 2, reading R19), next to the
                     measured milliseconds per call of this library,

All filtering runs in the library's kernels (`rbmf.Plan`); this module only counts the triggers they return (torch /
numpy on the lists) and evaluates the paper's closed-form cost model.  It does not import the oracle.
"""
from __future__ import annotations

import math

import numpy as np


def _counts_at_least(mods, grid):
    """number of entries of the device tensor `mods` that are >= each grid value (ascending grid) -> numpy int64"""
    import torch
    if mods.numel() == 0:
        return np.zeros(len(grid), dtype=np.int64)
    srt = torch.sort(mods).values
    g = torch.as_tensor(np.asarray(grid, dtype=np.float32), device=mods.device)
    return (srt.numel() - torch.searchsorted(srt, g, right=False)).cpu().numpy().astype(np.int64)


def rho_target(n_final, n_flat, grid, ratio=0.99):
    """Eq. 16 on the cumulative counts n_final[i], n_flat[i] = triggers with |rho| >= grid[i]
    (ascending grid): the smallest threshold with flat triggers above which the hierarchical search keeps at least
    `ratio` of the flat triggers at EVERY grid value -- a threshold that passes below one that fails does not count.
    None if there is no such threshold."""
    kept = np.asarray(n_final, dtype=np.float64)
    flat = np.asarray(n_flat, dtype=np.float64)
    lost_too_many = np.flatnonzero(kept < ratio * flat)
    first = int(lost_too_many[-1]) + 1 if lost_too_many.size else 0     # the condition holds on grid[first:]
    populated = np.flatnonzero(flat[first:] > 0)
    return float(grid[first + int(populated[0])]) if populated.size else None


def cost_ratio(N, T, w, p, f_per_template):
    """Eq. 15 / Eq. 13: total operations of the hierarchical scheme with the first stage by
    templates, f first-stage triggers per template and segment, over those of the flat template method."""
    z_basic = N * T * (5.0 * math.log2(N) + 6.0)
    z_first = N * T * (5.0 / w * math.log2(N / w) + 6.0 + 2.0 / w)
    z_total = z_first + 4.0 * p * w * f_per_template * T + N * p * (5.0 * math.log2(N) + 6.0)
    return z_total / z_basic, z_first / z_basic


def tune(rbmf, N, fs, f_low, basis, coeffs, sigma, strains, ws=(2, 4, 8, 16), thr1_grid=(3.0, 3.5, 4.0, 4.5, 5.0),
         rho2_grid=None, ratio=0.99, capacity=1 << 24, device="cuda:0", gemm_impl=None):
    """Run the study.  basis (k, N/2+1), coeffs (T, k), sigma (T,), strains (S, N/2+1): numpy or torch arrays.
    Returns {"grid", "n_flat", "flat_ms", "rows": [{w, rho_I, f_per_template_second, n_final, rho_target,
    cost_over_flat, first_stage_cost_over_flat, ms_per_segment, ...}]}."""
    import torch
    if rho2_grid is None:
        rho2_grid = np.round(np.arange(min(thr1_grid), 8.0001, 0.1), 6)
    rho2_grid = np.asarray(rho2_grid, dtype=np.float64)
    thr2 = float(rho2_grid[0])
    basis_t, coeffs_t, sigma_t = torch.as_tensor(basis), torch.as_tensor(coeffs), torch.as_tensor(sigma)
    k, T = basis_t.shape[0], coeffs_t.shape[0]
    S = len(strains)
    seconds = S * N / fs
    strains_dev = torch.as_tensor(np.asarray(strains)).to(device)

    def run(w, thr1):
        """sum over segments of the counts on the grid, candidates, and the mean ms per segment"""
        counts, n_cand, ms = np.zeros(len(rho2_grid), dtype=np.int64), 0, 0.0
        for s in range(S):
            plan.filter_async(strains_dev[s], thr1, thr2)
            nc, nt, st = plan.counts(allow_overflow=True)
            if st != rbmf.RBMF_OK:
                raise RuntimeError("tuning: list capacity %d exceeded (w=%d, rho_I=%g)" % (capacity, w, thr1))
            rows = plan.triggers_device()
            mods = torch.hypot(rows[:, 2].view(torch.float32), rows[:, 3].view(torch.float32))
            counts += _counts_at_least(mods, rho2_grid)
            n_cand += nc
            ms += plan.stage_ms()["total"]
        return counts, n_cand, ms / S

    def make_plan(w):
        p = rbmf.Plan(N, fs, f_low, k, T, w=w, max_candidates=capacity, max_triggers=capacity, device=device)
        if gemm_impl is not None:
            p.set_gemm_impl(gemm_impl)
        p.set_basis(basis_t)
        p.set_coeffs(coeffs_t, sigma_t)
        p.set_timing(True)
        return p

    plan = make_plan(1)                                   # the flat search: every sample is its own bin
    n_flat, _, flat_ms = run(1, thr2)
    plan.close()
    out = {"grid": rho2_grid.tolist(), "n_flat": n_flat.tolist(), "flat_ms_per_segment": flat_ms, "ratio": ratio,
           "segments": S, "seconds": seconds, "rows": []}
    for w in ws:
        plan = make_plan(w)
        for thr1 in thr1_grid:
            n_final, n_cand, ms = run(w, float(thr1))
            f_seg = n_cand / (T * S)                      # first-stage triggers per template and segment
            total, first = cost_ratio(N, T, w, k, f_seg)
            out["rows"].append({"w": int(w), "rho_I": float(thr1), "n_first_stage": int(n_cand),
                                "f_per_template_second": n_cand / (T * seconds), "n_final": n_final.tolist(),
                                "rho_target": rho_target(n_final, n_flat, rho2_grid, ratio),
                                "cost_over_flat": total, "first_stage_cost_over_flat": first,
                                "ms_per_segment": ms, "ms_over_flat_search": ms / flat_ms})
        plan.close()
    return out


def main(argv=None):
    """python -m paper_2110_13115_b200.tuning [--config small] [--segments 8] [--ws 2,4,8,16] [--thr1 3.0,3.5,...]
    Runs the study on noise-only segments of a synthetic config (paper_2110_13115_b200.workloads) and prints one JSON
    document (the rows of Fig. 5-7: f(w, rho_I), rho_target, Eq. 15 / Eq. 13, measured ms)."""
    import argparse
    import json

    import torch

    from . import rbmf, workloads
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", default="small")
    ap.add_argument("--segments", type=int, default=8)
    ap.add_argument("--ws", default="2,4,8,16")
    ap.add_argument("--thr1", default="3.0,3.5,4.0,4.5,5.0,5.5")
    ap.add_argument("--ratio", type=float, default=0.99)
    args = ap.parse_args(argv)
    cfg = workloads.CONFIGS[args.config].replace(n_inj=0)          # Gaussian noise only, as PAPER.md:296
    wl = workloads.make_workload(cfg, device="cuda" if torch.cuda.is_available() else "cpu")
    strains = np.stack([workloads.make_strain(wl, s)[0] for s in range(args.segments)])
    thr1 = [float(x) for x in args.thr1.split(",")]
    res = tune(rbmf, cfg.N, cfg.fs, cfg.f_low, wl["basis"], wl["coeffs"], wl["sigma"], strains,
               ws=[int(x) for x in args.ws.split(",")], thr1_grid=thr1,
               rho2_grid=np.round(np.arange(min(thr1), 7.0001, 0.1), 6), ratio=args.ratio)
    res["config"] = "%s (noise only): N=%d fs=%g k=%d T=%d, %d segments" % (cfg.name, cfg.N, cfg.fs, cfg.k, cfg.T,
                                                                          args.segments)
    print(json.dumps(res))
    return 0


if __name__ == "__main__":
    import sys
    sys.exit(main())
