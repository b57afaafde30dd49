"""Comparison rule between a trigger list under test and the fp64 oracle's result (test infrastructure).

"Identical trigger sets" across an fp32 GPU path and an fp64 oracle is decidable only away from the thresholds, so
("comparison rule") with tau = 1e-3, the metric's own SNR tolerance:

  mandatory set M = oracle triggers with |rho_bar|/thr1 - 1 >  tau  and  |rho|/thr2 - 1 >  tau
  allowed   set A = oracle samples  with |rho_bar|/thr1 - 1 > -tau  and  |rho|/thr2 - 1 > -tau
  pass  iff  M  subset-of  GOT  subset-of  A,  and for every trigger in GOT
             | |rho_got| - |rho_or| | <= 1e-3 |rho_or|   and   |arg(rho_got conj(rho_or))| <= 1e-3 rad.

This module imports nothing from the CUDA path.
"""
from __future__ import annotations

import numpy as np

TAU = 1e-3


def _keys(templates, times, N):
    return np.asarray(templates, dtype=np.int64) * int(N) + np.asarray(times, dtype=np.int64)


def compare_triggers(got, oracle_result, N, thr1, thr2, tau=TAU, snr_rtol=1e-3, phase_atol=1e-3):
    """got: structured array with fields template, time, re, im.  oracle_result: dict from oracle_filter
    (keep_margins=True).  Returns a report dict; report['ok'] is the verdict."""
    near = oracle_result["near"]
    trig = oracle_result["triggers"]
    mod_near = np.hypot(near["re"], near["im"])
    allowed = near[(near["avg_abs"] / thr1 - 1.0 > -tau) & (mod_near / thr2 - 1.0 > -tau)]
    mod_trig = np.hypot(trig["re"], trig["im"])
    mandatory = trig[(trig["avg_abs"] / thr1 - 1.0 > tau) & (mod_trig / thr2 - 1.0 > tau)]

    k_got = _keys(got["template"], got["time"], N)
    k_all = _keys(allowed["template"], allowed["time"], N)
    k_man = _keys(mandatory["template"], mandatory["time"], N)
    dup = len(k_got) - len(np.unique(k_got))
    missing = np.setdiff1d(k_man, k_got)
    extra = np.setdiff1d(k_got, k_all)

    # per-trigger values against the oracle's value at the same (template, time)
    max_rel, max_phase, bad_val = _match_values(k_got, got["re"], got["im"], k_all, allowed["re"], allowed["im"],
                                                snr_rtol, phase_atol)
    ok = dup == 0 and len(missing) == 0 and len(extra) == 0 and bad_val == 0
    return {
        "ok": bool(ok), "n_got": int(len(k_got)), "n_oracle": int(len(trig)), "n_mandatory": int(len(k_man)),
        "n_allowed": int(len(k_all)), "n_missing": int(len(missing)), "n_extra": int(len(extra)),
        "n_duplicates": int(dup), "n_bad_values": bad_val, "max_rel_snr_err": max_rel, "max_phase_err": max_phase,
        "tie_band": int(len(k_all) - len(k_man)),
    }


def _match_values(k_got, got_re, got_im, k_ref, ref_re, ref_im, snr_rtol, phase_atol):
    """For every got key present in k_ref: relative modulus error and phase error against the reference value."""
    if len(k_ref) == 0 or len(k_got) == 0:
        return 0.0, 0.0, 0
    order = np.argsort(k_ref)
    pos = np.clip(np.searchsorted(k_ref[order], k_got), 0, len(k_ref) - 1)
    idx = order[pos]
    hit = k_ref[idx] == k_got
    ref = np.asarray(ref_re)[idx[hit]] + 1j * np.asarray(ref_im)[idx[hit]]
    val = np.asarray(got_re)[hit].astype(np.float64) + 1j * np.asarray(got_im)[hit].astype(np.float64)
    if len(ref) == 0:
        return 0.0, 0.0, 0
    rel = np.abs(np.abs(val) - np.abs(ref)) / np.abs(ref)
    ph = np.abs(np.angle(val * np.conj(ref)))
    return float(rel.max()), float(ph.max()), int(((rel > snr_rtol) | (ph > phase_atol)).sum())


def compare_candidates(got, oracle_result, n_bins, thr1, tau=TAU, snr_rtol=1e-3, phase_atol=1e-3):
    """First-stage candidate sets, two-sided and value-checked, same rule as the triggers:
      mandatory M = oracle bins with |rho_bar|/thr1 - 1 >  tau   (from oracle_result['candidates'])
      allowed   A = oracle bins with |rho_bar|/thr1 - 1 > -tau   (from oracle_result['cand_near'])
      pass iff M subset-of GOT subset-of A, no duplicates, and every reported averaged SNR is within 1e-3 (relative
      modulus) and 1e-3 rad of the oracle's rho_bar of that bin.
    `got` has fields template, bin, re, im."""
    cand = oracle_result["candidates"]
    near = oracle_result["cand_near"]
    man = cand[np.hypot(cand["re"], cand["im"]) / thr1 - 1.0 > tau]
    allowed = near[np.hypot(near["re"], near["im"]) / thr1 - 1.0 > -tau]
    k_got = _keys(got["template"], got["bin"], n_bins)
    k_man = _keys(man["template"], man["bin"], n_bins)
    k_all = _keys(allowed["template"], allowed["bin"], n_bins)
    dup = len(k_got) - len(np.unique(k_got))
    missing = np.setdiff1d(k_man, k_got)
    extra = np.setdiff1d(k_got, k_all)
    max_rel, max_phase, bad_val = _match_values(k_got, got["re"], got["im"], k_all, allowed["re"], allowed["im"],
                                                snr_rtol, phase_atol)
    ok = dup == 0 and len(missing) == 0 and len(extra) == 0 and bad_val == 0
    return {"ok": bool(ok), "n_got": int(len(k_got)), "n_oracle": int(len(cand)), "n_mandatory": int(len(k_man)),
            "n_allowed": int(len(k_all)), "n_missing": int(len(missing)), "n_extra": int(len(extra)),
            "n_duplicates": int(dup), "n_bad_values": bad_val, "max_rel_err": max_rel, "max_phase_err": max_phase}
