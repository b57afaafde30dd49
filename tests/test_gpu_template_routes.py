"""The paper's template routes on the GPU against the fp64 oracle: the flat template method
(Eq. 13) and the fast first stage by templates (Eq. 10-12) feeding the unchanged second stage."""
import numpy as np
import pytest

from oracle import compare
from oracle import rbmf_oracle as orc
from paper_2110_13115_b200 import workloads as wlm

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def rbmf(built_library):
    from paper_2110_13115_b200 import rbmf as mod
    return mod


_WL = {}


def workload(name):
    if name not in _WL:
        _WL[name] = wlm.make_workload(wlm.CONFIGS[name], device="cuda")
    return _WL[name]


def reconstructed(wl):
    import torch
    c = torch.from_numpy(wl["coeffs"]).cuda().to(torch.complex128)
    b = torch.from_numpy(wl["basis"]).cuda().to(torch.complex128)
    return (c @ b).to(torch.complex64).contiguous()       # input synthesis only: h'_t = sum_k c_tk b_k as complex64


def make_plan(rbmf, wl, w, slab, cap=1 << 20):
    import torch
    cfg = wl["config"]
    plan = rbmf.Plan(cfg.N, cfg.fs, cfg.f_low, cfg.k, cfg.T, w=w, max_candidates=cap, max_triggers=cap,
                     template_slab=slab)
    plan.set_basis(torch.from_numpy(wl["basis"]))
    plan.set_coeffs(torch.from_numpy(wl["coeffs"]), torch.from_numpy(wl["sigma"]))
    return plan


@pytest.mark.parametrize("name,w,slab,thr", [("tiny", 4, 24, 3.5), ("tiny", 2, 64, 3.5), ("mini", 8, 128, 4.0)])
def test_flat_template_method_bank_templates(rbmf, name, w, slab, thr):
    """Bank templates u_t, sigma = 1 (the paper's literal convention): every sample of every template."""
    import torch
    wl = workload(name)
    cfg = wl["config"]
    bank = wlm.bank_templates(wl, np.arange(cfg.T), device="cuda").astype(np.complex64)
    plan = make_plan(rbmf, wl, w, slab)
    tpl = torch.from_numpy(bank).cuda()
    plan.set_templates(tpl, None)
    got = plan.filter_flat(torch.from_numpy(wl["strain"]), thr)
    ref = orc.template_method_triggers(wl["strain"], bank, None, cfg.N, cfg.fs, cfg.f_low, thr)
    rep = compare.compare_triggers(got, ref, cfg.N, 1.0, thr)
    plan.close()
    assert rep["ok"] and rep["n_mandatory"] > 100, rep
    # the injected template peaks at its injected SNR at the injected sample (R22)
    inj = wl["injections"][0]
    sel = got[(got["template"] == inj["template"]) & (got["time"] == inj["n0"])]
    assert len(sel) == 1 and abs(np.hypot(sel["re"][0], sel["im"][0]) - inj["snr"]) < 3.5


@pytest.mark.parametrize("name,w,slab,thr", [("tiny", 4, 16, (3.0, 4.0)), ("mini", 2, 64, (3.5, 4.0)),
                                             ("mini", 8, 300, (3.0, 4.0)), ("mini", 16, 128, (1.5, 3.5))])
def test_first_stage_by_templates_then_second_stage(rbmf, name, w, slab, thr):
    import torch
    wl = workload(name)
    cfg = wl["config"]
    plan = make_plan(rbmf, wl, w, slab)
    tpl = reconstructed(wl)
    plan.set_templates(tpl, torch.from_numpy(wl["sigma"]))
    ref = orc.oracle_filter(wl["strain"], wl["basis"], wl["coeffs"], wl["sigma"], cfg.N, cfg.fs, cfg.f_low, w, *thr)
    # the hierarchical search with the first stage by templates ...
    plan.set_stage1_route(rbmf.RBMF_STAGE1_TEMPLATES)
    got = plan.filter(torch.from_numpy(wl["strain"]), *thr)
    cand = plan.candidates()
    rep = compare.compare_triggers(got, ref, cfg.N, *thr)
    crep = compare.compare_candidates(cand, ref, cfg.N // w, thr[0])
    assert rep["ok"] and rep["n_mandatory"] > 50, rep
    assert crep["ok"] and crep["n_mandatory"] > 50, crep
    # ... its candidates against the oracle's own Eq. 12 route on a template sample ...
    ids = np.arange(0, cfg.T, max(1, cfg.T // 16))
    ref12 = orc.first_stage_by_templates(wl["strain"], tpl[ids].cpu().numpy(), wl["sigma"][ids], cfg.N, cfg.fs, cfg.f_low,
                                         w, thr[0])
    for key in ("candidates", "cand_near"):
        ref12[key]["template"] = ids[ref12[key]["template"]]
    sub = cand[np.isin(cand["template"], ids)]
    crep12 = compare.compare_candidates(sub, ref12, cfg.N // w, thr[0])
    assert crep12["ok"] and crep12["n_got"] > 0, crep12
    # ... and the same call by the basis route gives the same sets (tie band aside)
    plan.set_stage1_route(rbmf.RBMF_STAGE1_BASIS)
    got_b = plan.filter(torch.from_numpy(wl["strain"]), *thr)
    ka = got["template"].astype(np.int64) * cfg.N + got["time"]
    kb = got_b["template"].astype(np.int64) * cfg.N + got_b["time"]
    assert len(np.setxor1d(ka, kb)) <= max(2, rep["tie_band"])
    # flat method with the reconstructed templates = the oracle's flat set, of which the hierarchical set is a subset
    flat = plan.filter_flat(torch.from_numpy(wl["strain"]), thr[1])
    ref_flat = orc.template_method_triggers(wl["strain"], tpl.cpu().numpy(), wl["sigma"], cfg.N, cfg.fs, cfg.f_low, thr[1])
    frep = compare.compare_triggers(flat, ref_flat, cfg.N, 1.0, thr[1])
    assert frep["ok"], frep
    kf = flat["template"].astype(np.int64) * cfg.N + flat["time"]
    assert len(np.setdiff1d(ka, kf)) <= rep["tie_band"] and len(kf) >= len(ka)
    plan.close()


def test_small_config_both_template_routes(rbmf):
    import torch
    wl = workload("small")
    cfg = wl["config"]
    plan = make_plan(rbmf, wl, cfg.w, 256, cap=1 << 22)
    tpl = reconstructed(wl)
    plan.set_templates(tpl, torch.from_numpy(wl["sigma"]))
    plan.set_stage1_route(rbmf.RBMF_STAGE1_TEMPLATES)
    got = plan.filter(torch.from_numpy(wl["strain"]), cfg.thr1, cfg.thr2)
    cand = plan.candidates()
    ref = orc.oracle_filter(wl["strain"], wl["basis"], wl["coeffs"], wl["sigma"], cfg.N, cfg.fs, cfg.f_low, cfg.w,
                            cfg.thr1, cfg.thr2)
    rep = compare.compare_triggers(got, ref, cfg.N, cfg.thr1, cfg.thr2)
    crep = compare.compare_candidates(cand, ref, cfg.N // cfg.w, cfg.thr1)
    assert rep["ok"] and rep["n_mandatory"] > 1000, rep
    assert crep["ok"], crep
    flat = plan.filter_flat(torch.from_numpy(wl["strain"]), cfg.thr2)
    plan.close()
    assert len(flat) == ref["n_flat"] or abs(len(flat) - ref["n_flat"]) <= 200      # tie band of the flat set
    ids = np.unique(flat["template"])[:40]
    ref_flat = orc.template_method_triggers(wl["strain"], tpl[ids].cpu().numpy(), wl["sigma"][ids], cfg.N, cfg.fs,
                                            cfg.f_low, cfg.thr2)
    for key in ("triggers", "near"):
        ref_flat[key]["template"] = ids[ref_flat[key]["template"]]
    frep = compare.compare_triggers(flat[np.isin(flat["template"], ids)], ref_flat, cfg.N, 1.0, cfg.thr2)
    assert frep["ok"] and frep["n_mandatory"] > 50, frep


def test_template_routes_argument_checks(rbmf):
    import ctypes
    b = rbmf
    h = ctypes.c_void_p()
    assert b.rbmf_plan_create(ctypes.byref(h), 4096, 1024.0, 30.0, 16, 64) == b.RBMF_OK
    assert b.rbmf_plan_set_stage1_route(h, b.RBMF_STAGE1_TEMPLATES) == b.RBMF_ERR_STATE     # not enabled
    assert b.rbmf_plan_enable_template_routes(h, 6) == b.RBMF_ERR_ARG
    assert b.rbmf_plan_set_window(h, 1) == b.RBMF_OK
    assert b.rbmf_plan_enable_template_routes(h, 64) == b.RBMF_ERR_UNSUPPORTED              # w = 1 is the flat method
    assert b.rbmf_plan_set_window(h, 4) == b.RBMF_OK
    assert b.rbmf_plan_enable_template_routes(h, 64) == b.RBMF_OK
    assert b.rbmf_plan_set_stage1_route(h, b.RBMF_STAGE1_TEMPLATES) == b.RBMF_OK
    assert b.rbmf_plan_set_stage1_route(h, 5) == b.RBMF_ERR_ARG
    dummy = ctypes.c_void_p(1024)
    assert b.rbmf_filter_flat(h, dummy, 5.0, dummy, dummy) == b.RBMF_ERR_STATE
    assert b.rbmf_set_templates(h, dummy, None) == b.RBMF_ERR_STATE
    b.rbmf_plan_destroy(h)


def test_refused_template_route_call_launches_nothing(rbmf):
    """rbmf_filter with RBMF_STAGE1_TEMPLATES selected but no templates set is a call-order error.  It must be refused
    BEFORE the first launch (it used to be noticed after the FFT kernel had been enqueued): beta of the previous,
    successful call is still there byte for byte although the refused call was given a different strain, and the
    previous call's lists are still readable."""
    import torch
    wl = workload("tiny")
    cfg = wl["config"]
    plan = make_plan(rbmf, wl, 4, 16)
    first = plan.filter(torch.from_numpy(wl["strain"]), 3.0, 4.0)
    beta = plan.internal("beta").tobytes()
    plan.set_stage1_route(rbmf.RBMF_STAGE1_TEMPLATES)
    other = torch.from_numpy(np.ascontiguousarray(wl["strain"][::-1] * 2.0))
    with pytest.raises(rbmf.RbmfError) as info:
        plan.filter(other, 3.0, 4.0)
    assert info.value.status == rbmf.RBMF_ERR_STATE
    torch.cuda.synchronize()
    assert plan.internal("beta").tobytes() == beta
    assert np.array_equal(np.sort(plan.triggers(), order=("template", "time")),
                          np.sort(first, order=("template", "time")))
    plan.close()
