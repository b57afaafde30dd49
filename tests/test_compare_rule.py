"""CPU pins of the comparison rule every parity verdict rests on (oracle/compare.py; SURVEY.md 8(c) "comparison rule";
sets of PAPER.md:191, averaging of Eq. 9).

The rule is exercised on the oracle's own result for a small workload: it must accept that result, and it must reject
each single defect a broken GPU path could produce (a dropped mandatory trigger, a trigger outside the allowed band, a
duplicate, a value off by 2e-3, a phase off by 2e-3 rad), while tolerating exactly the tie-band differences.  The
`near` / `cand_near` supersets, which ARE the allowed sets, are pinned against a pure-Python enumeration.
"""
import numpy as np
import pytest

from oracle import compare
from oracle import rbmf_oracle as orc
from paper_2110_13115_b200 import workloads as wlm

TRIG_DT = np.dtype([("template", np.int32), ("time", np.int32), ("re", np.float32), ("im", np.float32)])
CAND_DT = np.dtype([("template", np.int32), ("bin", np.int32), ("re", np.float32), ("im", np.float32)])


@pytest.fixture(scope="module")
def micro():
    cfg = wlm.WorkloadConfig("micro", 31, 256, 256.0, 20.0, 8, 8, 4, 1.0, 1.3, 1, 9.0, 9.0, thr1=2.0, thr2=2.5)
    return wlm.make_workload(cfg)


def run_oracle(wl, thr1=None, thr2=None):
    cfg = wl["config"]
    thr1 = cfg.thr1 if thr1 is None else thr1
    thr2 = cfg.thr2 if thr2 is None else thr2
    return orc.oracle_filter(wl["strain"], wl["basis"], wl["coeffs"], wl["sigma"], cfg.N, cfg.fs, cfg.f_low, cfg.w,
                             thr1, thr2), thr1, thr2


def as_got(trig):
    g = np.empty(len(trig), dtype=TRIG_DT)
    for f in ("template", "time", "re", "im"):
        g[f] = trig[f]
    return g


def as_got_cand(cand):
    g = np.empty(len(cand), dtype=CAND_DT)
    for f in ("template", "bin", "re", "im"):
        g[f] = cand[f]
    return g


def mandatory_mask(trig, thr1, thr2, tau=compare.TAU):
    return (trig["avg_abs"] / thr1 - 1 > tau) & (np.hypot(trig["re"], trig["im"]) / thr2 - 1 > tau)


# ------------------------------------------------------------------------------------------------ triggers
def test_oracle_list_passes_and_order_is_free(micro):
    ref, thr1, thr2 = run_oracle(micro)
    N = micro["config"].N
    got = as_got(ref["triggers"])
    assert len(got) > 10
    rep = compare.compare_triggers(got, ref, N, thr1, thr2)
    assert rep["ok"] and rep["n_got"] == len(got) and rep["n_missing"] == rep["n_extra"] == 0, rep
    assert rep["max_rel_snr_err"] < 1e-6 and rep["max_phase_err"] < 1e-6      # float32 rounding of the copy only
    perm = np.random.default_rng(0).permutation(len(got))
    assert compare.compare_triggers(got[perm], ref, N, thr1, thr2)["ok"]       # unordered set
    assert compare.compare_triggers(got[:0], ref, N, 50.0, 50.0)["ok"]         # empty against empty


def test_dropped_mandatory_trigger_fails(micro):
    ref, thr1, thr2 = run_oracle(micro)
    N = micro["config"].N
    man = np.nonzero(mandatory_mask(ref["triggers"], thr1, thr2))[0]
    assert len(man) > 0
    got = as_got(np.delete(ref["triggers"], man[len(man) // 2]))
    rep = compare.compare_triggers(got, ref, N, thr1, thr2)
    assert not rep["ok"] and rep["n_missing"] == 1 and rep["n_extra"] == 0


def test_trigger_outside_allowed_band_fails(micro):
    ref, thr1, thr2 = run_oracle(micro)
    cfg = micro["config"]
    near_keys = set(zip(ref["near"]["template"].tolist(), ref["near"]["time"].tolist()))
    t, n = next((t, n) for t in range(cfg.T) for n in range(cfg.N) if (t, n) not in near_keys)
    got = as_got(ref["triggers"])
    extra = np.array([(t, n, thr2 * 1.5, 0.0)], dtype=TRIG_DT)
    rep = compare.compare_triggers(np.concatenate([got, extra]), ref, cfg.N, thr1, thr2)
    assert not rep["ok"] and rep["n_extra"] == 1 and rep["n_missing"] == 0
    # a sample just OUTSIDE the band (margin slightly below -tau) is an extra; just inside it is tolerated
    trig = ref["triggers"]
    i = int(np.argmin(np.hypot(trig["re"], trig["im"])))
    mod = float(np.hypot(trig["re"][i], trig["im"][i]))
    for factor, ok in ((1.0 + 1.5e-3, False), (1.0 + 5e-4, True)):
        ref2, _, thr2b = run_oracle(micro, thr2=mod * factor)     # the sample now lies below the threshold
        rep = compare.compare_triggers(as_got(trig[i:i + 1]), ref2, cfg.N, thr1, thr2b)
        assert (rep["n_extra"] == 0) == ok, (factor, rep)


def test_duplicate_fails(micro):
    ref, thr1, thr2 = run_oracle(micro)
    got = as_got(ref["triggers"])
    rep = compare.compare_triggers(np.concatenate([got, got[3:4]]), ref, micro["config"].N, thr1, thr2)
    assert not rep["ok"] and rep["n_duplicates"] == 1


@pytest.mark.parametrize("scale,rot,ok", [(1 + 2e-3, 0.0, False), (1 - 2e-3, 0.0, False), (1.0, 2e-3, False),
                                          (1.0, -2e-3, False), (1 + 5e-4, 5e-4, True)])
def test_value_tolerances(micro, scale, rot, ok):
    ref, thr1, thr2 = run_oracle(micro)
    got = as_got(ref["triggers"])
    i = len(got) // 3
    v = complex(got["re"][i], got["im"][i]) * scale * np.exp(1j * rot)
    got["re"][i], got["im"][i] = v.real, v.imag
    rep = compare.compare_triggers(got, ref, micro["config"].N, thr1, thr2)
    assert rep["ok"] == ok and (rep["n_bad_values"] == 0) == ok, rep


def test_values_are_matched_to_the_right_record(micro):
    """Swapping the values of two triggers (keys untouched) must be caught: the searchsorted pairing is by key."""
    ref, thr1, thr2 = run_oracle(micro)
    got = as_got(ref["triggers"])
    mods = np.hypot(got["re"], got["im"])
    i, j = int(np.argmax(mods)), int(np.argmin(mods))
    assert mods[i] / mods[j] > 1.01
    for f in ("re", "im"):
        got[f][i], got[f][j] = got[f][j], got[f][i]
    rep = compare.compare_triggers(got[::-1], ref, micro["config"].N, thr1, thr2)
    assert not rep["ok"] and rep["n_bad_values"] == 2


def test_tie_band_members_may_come_and_go(micro):
    cfg = micro["config"]
    base, thr1, _ = run_oracle(micro)
    trig = base["triggers"]
    i = int(np.argsort(np.hypot(trig["re"], trig["im"]))[len(trig) // 2])
    mod = float(np.hypot(trig["re"][i], trig["im"][i]))
    key = (int(trig["template"][i]), int(trig["time"][i]))
    # threshold just ABOVE the sample: not an oracle trigger, but allowed -> reporting it is fine
    ref, _, thr2 = run_oracle(micro, thr2=mod * (1 + 5e-4))
    keys = list(zip(ref["triggers"]["template"].tolist(), ref["triggers"]["time"].tolist()))
    assert key not in keys
    got = np.concatenate([as_got(ref["triggers"]), as_got(trig[i:i + 1])])
    rep = compare.compare_triggers(got, ref, cfg.N, thr1, thr2)
    assert rep["ok"] and rep["tie_band"] >= 1, rep
    # threshold just BELOW the sample: an oracle trigger, but not mandatory -> dropping it is fine
    ref, _, thr2 = run_oracle(micro, thr2=mod * (1 - 5e-4))
    keys = list(zip(ref["triggers"]["template"].tolist(), ref["triggers"]["time"].tolist()))
    assert key in keys
    got = as_got(np.delete(ref["triggers"], keys.index(key)))
    rep = compare.compare_triggers(got, ref, cfg.N, thr1, thr2)
    assert rep["ok"] and rep["n_got"] == rep["n_oracle"] - 1, rep
    # the same for the first-stage margin: thr1 just above / below that trigger's bin average
    avg = float(trig["avg_abs"][i])
    ref, thr1b, thr2 = run_oracle(micro, thr1=avg * (1 + 5e-4))
    got = np.concatenate([as_got(ref["triggers"]), as_got(trig[i:i + 1])])
    assert compare.compare_triggers(got, ref, cfg.N, thr1b, thr2)["ok"]
    ref, thr1b, thr2 = run_oracle(micro, thr1=avg * (1 + 3e-3))
    got = np.concatenate([as_got(ref["triggers"]), as_got(trig[i:i + 1])])
    assert not compare.compare_triggers(got, ref, cfg.N, thr1b, thr2)["ok"]


# ---------------------------------------------------------------- the supersets, against a plain enumeration
def test_near_sets_against_python_enumeration(micro):
    cfg = micro["config"]
    N, w = cfg.N, cfg.w
    ref, thr1, thr2 = run_oracle(micro)
    hp = orc.reconstructed_templates(micro["coeffs"], micro["basis"])
    exp_near, exp_cnear = [], []
    for t in range(cfg.T):
        rho = orc.snr_series_direct(micro["strain"], hp[t], micro["sigma"][t], N, cfg.j_low)
        for i in range(N // w):
            mean = sum(rho[i * w + r] for r in range(w)) / w
            if abs(mean) >= thr1 * (1 - 2e-3):
                exp_cnear.append((t, i, mean))
                for r in range(w):
                    if abs(rho[i * w + r]) >= thr2 * (1 - 2e-3):
                        exp_near.append((t, i * w + r, rho[i * w + r], abs(mean)))
    near, cnear = ref["near"], ref["cand_near"]
    assert [(int(a), int(b)) for a, b in zip(near["template"], near["time"])] == [(t, n) for t, n, _, _ in exp_near]
    assert np.allclose(near["re"] + 1j * near["im"], [v for _, _, v, _ in exp_near], rtol=0, atol=1e-11)
    assert np.allclose(near["avg_abs"], [a for _, _, _, a in exp_near], rtol=0, atol=1e-11)
    assert [(int(a), int(b)) for a, b in zip(cnear["template"], cnear["bin"])] == [(t, i) for t, i, _ in exp_cnear]
    assert np.allclose(cnear["re"] + 1j * cnear["im"], [v for _, _, v in exp_cnear], rtol=0, atol=1e-11)
    assert len(near) >= len(ref["triggers"]) and len(cnear) >= len(ref["candidates"])
    # the allowed sets of the rule (margin > -tau = -1e-3) lie inside these supersets (cut at -2e-3) by construction;
    # every trigger / candidate is a member
    tk = set(zip(ref["triggers"]["template"].tolist(), ref["triggers"]["time"].tolist()))
    assert tk <= set(zip(near["template"].tolist(), near["time"].tolist()))
    ck = set(zip(ref["candidates"]["template"].tolist(), ref["candidates"]["bin"].tolist()))
    assert ck <= set(zip(cnear["template"].tolist(), cnear["bin"].tolist()))


# ---------------------------------------------------------------------------------------------- candidates
def test_candidate_rule(micro):
    cfg = micro["config"]
    ref, thr1, thr2 = run_oracle(micro)
    nb = cfg.N // cfg.w
    cand = ref["candidates"]
    got = as_got_cand(cand)
    rep = compare.compare_candidates(got, ref, nb, thr1)
    assert rep["ok"] and rep["n_got"] == len(cand) > 5, rep
    mod = np.hypot(cand["re"], cand["im"])
    man = np.nonzero(mod / thr1 - 1 > compare.TAU)[0]
    rep = compare.compare_candidates(as_got_cand(np.delete(cand, man[0])), ref, nb, thr1)
    assert not rep["ok"] and rep["n_missing"] == 1
    # an over-full list: a bin whose averaged SNR is far below thr1
    ckeys = set(zip(ref["cand_near"]["template"].tolist(), ref["cand_near"]["bin"].tolist()))
    t, i = next((t, i) for t in range(cfg.T) for i in range(nb) if (t, i) not in ckeys)
    extra = np.array([(t, i, thr1 * 1.2, 0.0)], dtype=CAND_DT)
    rep = compare.compare_candidates(np.concatenate([got, extra]), ref, nb, thr1)
    assert not rep["ok"] and rep["n_extra"] == 1
    rep = compare.compare_candidates(np.concatenate([got, got[:1]]), ref, nb, thr1)
    assert not rep["ok"] and rep["n_duplicates"] == 1
    # a wrong averaged value
    bad = got.copy()
    bad["re"][2] *= 1 + 3e-3
    bad["im"][2] *= 1 + 3e-3
    rep = compare.compare_candidates(bad, ref, nb, thr1)
    assert not rep["ok"] and rep["n_bad_values"] == 1
    bad = got.copy()
    v = complex(bad["re"][2], bad["im"][2]) * np.exp(2e-3j)
    bad["re"][2], bad["im"][2] = v.real, v.imag
    assert not compare.compare_candidates(bad, ref, nb, thr1)["ok"]
    # tie band: thr1 just above one candidate's modulus -> it may still be reported; 3e-3 above -> it may not
    j = int(np.argsort(mod)[len(mod) // 2])
    for factor, ok in ((1 + 5e-4, True), (1 + 3e-3, False)):
        ref2, thr1b, _ = run_oracle(micro, thr1=float(mod[j]) * factor)
        got2 = np.concatenate([as_got_cand(ref2["candidates"]), got[j:j + 1]])
        assert compare.compare_candidates(got2, ref2, nb, thr1b)["ok"] == ok
