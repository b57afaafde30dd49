"""Parity of the CUDA path (through the C ABI) with the fp64 oracle, element by element on the same seeded inputs.

Bars (BASELINE.json north_star): trigger sets identical under the tau = 1e-3 tie band,
per-trigger |SNR| within 1e-3 relative and phase within 1e-3 rad; beta within 1e-5 absolute of the oracle's fp64
series (output rms 1.41); beta^avg within 1e-5 + 2^-16 |value| (bf16 hi+lo storage keeps 16 mantissa bits).
"""
import numpy as np
import pytest

from oracle import compare
from oracle import rbmf_oracle as orc
from paper_2110_13115_b200 import workloads as wlm

pytestmark = pytest.mark.gpu

BETA_ATOL = 1e-5


X3, SCREEN = 0, 2                # rbmf_gemm_impl (include/rbmf.h); SCREEN is the library default
SIMT = "fp32-check"              # test-only: bf16x3 operands through the plain fp32 CUDA-core kernel (rbmf_diag_set)


def beta_avg_close(got, ref, impl=X3):
    """bf16 hi + lo keeps 16 mantissa bits: 2^-17 relative per stored value, on top of the FFT's own error.
    The screen's single fp16 plane keeps 11: 2^-11 relative per component."""
    rel = 2.0 ** -16 if impl != SCREEN else 2.0 ** -10.4
    return np.all(np.abs(got - ref) <= 1e-5 + rel * np.abs(ref))


@pytest.fixture(scope="module")
def rbmf(built_library):
    from paper_2110_13115_b200 import rbmf as mod
    return mod


_WL = {}


def workload(name, **kw):
    key = (name, tuple(sorted(kw.items())))
    if key not in _WL:
        cfg = wlm.CONFIGS[name]
        if kw:
            cfg = cfg.replace(**kw)
        _WL[key] = wlm.make_workload(cfg, device="cuda")
    return _WL[key]


def set_impl(rbmf, plan, impl):
    if impl is None:
        return
    plan.diag_set(rbmf.RBMF_DIAG_STAGE1_FP32_CHECK, 1 if impl == SIMT else 0)
    plan.set_gemm_impl(X3 if impl == SIMT else impl)


def make_plan(rbmf, wl, w=None, impl=None, **kw):
    import torch
    cfg = wl["config"]
    plan = rbmf.Plan(cfg.N, cfg.fs, cfg.f_low, cfg.k, cfg.T, w=cfg.w if w is None else w,
                     max_candidates=kw.pop("max_candidates", 1 << 20), max_triggers=kw.pop("max_triggers", 1 << 20))
    set_impl(rbmf, plan, impl)
    plan.set_basis(torch.from_numpy(wl["basis"]))
    plan.set_coeffs(torch.from_numpy(wl["coeffs"]), torch.from_numpy(wl["sigma"]))
    return plan


def oracle(wl, w, thr1, thr2, templates=None):
    cfg = wl["config"]
    return orc.oracle_filter(wl["strain"], wl["basis"], wl["coeffs"], wl["sigma"], cfg.N, cfg.fs, cfg.f_low, w,
                             thr1, thr2, templates=templates)


def check(rbmf, wl, w, thr1, thr2, impl=SCREEN, expect_triggers=True, single_cta=False):
    import torch
    cfg = wl["config"]
    plan = make_plan(rbmf, wl, w=w, impl=impl)
    if single_cta:
        plan.diag_set(rbmf.RBMF_DIAG_SINGLE_CTA_SCREEN, 1)
    got = plan.filter(torch.from_numpy(wl["strain"]), thr1, thr2)
    ref = oracle(wl, w, thr1, thr2)
    rep = compare.compare_triggers(got, ref, cfg.N, thr1, thr2)
    cand = plan.candidates()
    crep = compare.compare_candidates(cand, ref, cfg.N // w, thr1)
    plan.close()
    assert rep["ok"], rep
    assert crep["ok"], crep
    if expect_triggers:
        assert rep["n_got"] > 0 and rep["n_mandatory"] > 0
    return rep, crep


# ------------------------------------------------------------------------------------------ kernel 1
@pytest.mark.parametrize("name", ["tiny", "mini"])
def test_beta_matches_oracle_series(rbmf, name):
    import torch
    wl = workload(name)
    cfg = wl["config"]
    plan = make_plan(rbmf, wl, impl=X3)
    plan.filter(torch.from_numpy(wl["strain"]), 50.0, 50.0)
    beta = plan.internal("beta")                       # (N, k)
    bavg = plan.internal("beta_avg")                   # (N/w, k)
    set_impl(rbmf, plan, SCREEN)
    plan.filter(torch.from_numpy(wl["strain"]), 50.0, 50.0)
    bavg16 = plan.internal("beta_avg")                 # the screen's single fp16 plane
    plan.close()
    ref = orc.basis_series(wl["strain"], wl["basis"], cfg.N, cfg.j_low)   # (k, N) fp64
    assert 1.2 < np.sqrt((np.abs(ref) ** 2).mean()) < 2.0                 # ~unit-variance quadratures (+ injection)
    err = np.abs(beta.T.astype(np.complex128) - ref).max()
    assert err < BETA_ATOL, err
    ref_avg = orc.bin_average(ref, cfg.w)
    assert beta_avg_close(bavg.T.astype(np.complex128), ref_avg)
    assert beta_avg_close(bavg16.T.astype(np.complex128), ref_avg, SCREEN)


@pytest.mark.parametrize("N,w", [(1024, 1), (2048, 2), (8192, 4), (32768, 16), (65536, 32)])
def test_beta_all_fft_lengths(rbmf, N, w):
    """Every pass length the dispatcher can pick (L = 32 .. 1024 appear over these sizes, incl. the folded transform)."""
    import torch
    wl = workload("tiny", N=N, T=16, n_inj=0, index=50 + w)
    cfg = wl["config"]
    plan = make_plan(rbmf, wl, w=w, impl=X3)
    plan.filter(torch.from_numpy(wl["strain"]), 50.0, 50.0)
    beta, bavg = plan.internal("beta"), plan.internal("beta_avg")
    plan.close()
    ref = orc.basis_series(wl["strain"], wl["basis"], cfg.N, cfg.j_low)
    assert np.abs(beta.T.astype(np.complex128) - ref).max() < BETA_ATOL
    assert beta_avg_close(bavg.T.astype(np.complex128), orc.bin_average(ref, w))


def test_beta_largest_length_sampled(rbmf):
    """N = 2^20 (1024 x 1024 passes): sampled columns against the oracle's fp64 series."""
    import torch
    wl = workload("tiny", N=1 << 20, fs=4096.0, f_low=20.0, T=16, n_inj=0, index=60)
    cfg = wl["config"]
    plan = make_plan(rbmf, wl, w=8, impl=X3)
    plan.filter(torch.from_numpy(wl["strain"]), 50.0, 50.0)
    beta, bavg = plan.internal("beta"), plan.internal("beta_avg")
    plan.close()
    cols = [0, 7, 15]
    ref = orc.basis_series(wl["strain"], wl["basis"][cols], cfg.N, cfg.j_low)
    assert np.abs(beta[:, cols].T.astype(np.complex128) - ref).max() < BETA_ATOL
    assert beta_avg_close(bavg[:, cols].T.astype(np.complex128), orc.bin_average(ref, 8))


# ------------------------------------------------------------------------------- whole path, exhaustive
@pytest.mark.parametrize("impl", [X3, SIMT, SCREEN])
@pytest.mark.parametrize("thr", [(3.0, 4.0), (5.0, 6.0)])
def test_tiny_exhaustive(rbmf, impl, thr):
    check(rbmf, workload("tiny"), 4, thr[0], thr[1], impl=impl)


def test_tiny_narrow_exhaustive(rbmf):
    rep, _ = check(rbmf, workload("tiny_narrow"), 4, 5.0, 6.0)
    assert rep["n_got"] > 0


@pytest.mark.parametrize("impl", [X3, SCREEN])
@pytest.mark.parametrize("w", [1, 2, 4, 8, 16])
def test_mini_all_windows(rbmf, w, impl):
    """N = 16384, k = 32, T = 300 (ragged against the 128-template tile), 3 injections."""
    # fs = 1024 Hz: a 16-sample average washes the peaks out, so the coarse threshold drops with w
    thr1 = {1: 4.0, 2: 4.0, 4: 4.0, 8: 3.5, 16: 2.5}[w]
    check(rbmf, workload("mini"), w, thr1, 5.0, impl=impl)


def test_mini_largest_window(rbmf):
    # w = 32 at fs = 1024 Hz averages every peak away: the point is the two-slot row layout of kernel 3
    check(rbmf, workload("mini"), 32, 0.4, 3.0, impl=SCREEN, expect_triggers=False)


def test_screen_single_cta_kernel(rbmf):
    """The screen's fallback kernel (no thread-block clusters) gives the same lists as the 2-CTA one."""
    check(rbmf, workload("mini"), 8, 3.5, 5.0, impl=SCREEN, single_cta=True)


def test_single_bin_block(rbmf):
    """N/w = 128: one time-bin block.  The 2-CTA screen kernel then has a partner CTA whose block lies entirely
    past the end (TMA zero fill + bin mask)."""
    wl = workload("tiny", N=1024, T=40, n_inj=1, index=71)
    for impl in (SCREEN, X3):
        check(rbmf, wl, 8, 1.5, 3.0, impl=impl, expect_triggers=False)


@pytest.mark.parametrize("impl", [X3, SCREEN])
def test_non_integer_band_edge_and_out_of_band_values_ignored(rbmf, impl):
    """f_low N / fs = 121.2: the band starts at bin 122 (ceil).  Basis and strain carry garbage below the band and in
    the Nyquist bin; the library must ignore it exactly as the oracle's definition does (include/rbmf.h, rbmf_set_basis)."""
    wl = dict(workload("tiny", f_low=30.3, index=72))
    cfg = wl["config"]
    assert cfg.j_low == 122 and orc.band(cfg.N, cfg.fs, cfg.f_low) == (122, cfg.N // 2)
    rng = np.random.default_rng(3)
    basis, strain = wl["basis"].copy(), wl["strain"].copy()
    basis[:, :122] = (rng.standard_normal((cfg.k, 122)) + 1j * rng.standard_normal((cfg.k, 122))).astype(np.complex64)
    basis[:, cfg.N // 2] = 7.0
    strain[:122] = strain[:122] * 3 + 50.0
    strain[cfg.N // 2] = 1000.0
    wl["basis"], wl["strain"] = basis, strain
    check(rbmf, wl, 4, 3.0, 4.0, impl=impl)


def test_mini_simt_and_tensor_core_candidates_agree(rbmf):
    """The three stage-1 implementations give the same candidate list (threshold ties aside), and the screen's
    superset really contains it with a modest overhead."""
    import torch
    wl = workload("mini")
    cfg = wl["config"]
    sets, trig = [], []
    for impl in (X3, SIMT, SCREEN):
        plan = make_plan(rbmf, wl, impl=impl)
        trig.append(plan.filter(torch.from_numpy(wl["strain"]), 2.5, 4.5))
        sets.append(plan.candidates())
        plan.close()
    a = sets[0]
    ka = a["template"].astype(np.int64) * cfg.N + a["bin"]
    assert len(ka) > 1000
    for b in sets[1:]:
        kb = b["template"].astype(np.int64) * cfg.N + b["bin"]
        sym = np.setxor1d(ka, kb)
        assert len(sym) <= max(2, len(ka) // 2000)          # only threshold ties may differ
        common, ia, ib = np.intersect1d(ka, kb, return_indices=True)
        assert np.abs(a["re"][ia] - b["re"][ib]).max() < 2e-4 and np.abs(a["im"][ia] - b["im"][ib]).max() < 2e-4
    # final triggers: identical sets between bf16x3 and screen + fp32 confirm, up to ties at thr1
    ta = trig[0]["template"].astype(np.int64) * cfg.N + trig[0]["time"]
    tc = trig[2]["template"].astype(np.int64) * cfg.N + trig[2]["time"]
    assert len(np.setxor1d(ta, tc)) <= max(2, len(ta) // 500)


def test_screen_superset_is_tight(rbmf):
    """How many (template, bin) pairs the fp16 screen passes relative to the confirmed candidates: the rigorous
    error bound must cost only a modest surplus (it is O(2^-10 ||beta^avg||) ~ 0.01-0.03 in SNR)."""
    import torch
    wl = workload("small")
    cfg = wl["config"]
    plan = make_plan(rbmf, wl, impl=SCREEN)
    plan.filter(torch.from_numpy(wl["strain"]), cfg.thr1, cfg.thr2)
    n_conf = plan.counts()[0]
    set_impl(rbmf, plan, X3)
    plan.filter(torch.from_numpy(wl["strain"]), cfg.thr1 - 0.05, cfg.thr2)
    n_loose = plan.counts()[0]
    plan.filter(torch.from_numpy(wl["strain"]), cfg.thr1, cfg.thr2)
    n_x3 = plan.counts()[0]
    plan.close()
    assert abs(n_conf - n_x3) <= max(3, n_x3 // 500)
    assert n_conf <= n_loose                       # sanity of the scale: thr1 - 0.05 already admits more


@pytest.mark.parametrize("impl", [X3, SCREEN])
def test_small_config_exhaustive(rbmf, impl):
    """BASELINE.json configs[1]: N = 131072, k = 128, T = 2000, w = 8, thresholds 5.0 / 6.0, 10 injections."""
    rep, crep = check(rbmf, workload("small"), 8, 5.0, 6.0, impl=impl)
    assert rep["n_got"] > 100


def test_small_narrow_recovers_injections(rbmf):
    """Narrow-Mc bank (truncation tolerance holds): every injection is recovered near its injected SNR."""
    import torch
    wl = workload("small_narrow")
    cfg = wl["config"]
    assert 1.0 - wl["captured"] < 1e-4
    plan = make_plan(rbmf, wl)
    got = plan.filter(torch.from_numpy(wl["strain"]), 5.0, 6.0)
    plan.close()
    ref = oracle(wl, 8, 5.0, 6.0, templates=sorted({i["template"] for i in wl["injections"]}))
    sub = got[np.isin(got["template"], ref["triggers"]["template"])]
    rep = compare.compare_triggers(sub, ref, cfg.N, 5.0, 6.0)
    assert rep["ok"], rep
    for inj in wl["injections"]:
        if inj["snr"] < 8.0:
            continue
        m = (got["template"] == inj["template"]) & (np.abs(got["time"] - inj["n0"]) <= 1)
        assert m.any(), inj
        peak = np.hypot(got["re"][m], got["im"][m]).max()
        assert abs(peak - inj["snr"]) < 3.5, (peak, inj)          # injected SNR +- noise


# ----------------------------------------------------------------------------------------- edge cases
def test_no_triggers_and_repeatability(rbmf):
    import torch
    wl = workload("tiny")
    plan = make_plan(rbmf, wl)
    s = torch.from_numpy(wl["strain"])
    assert len(plan.filter(s, 40.0, 40.0)) == 0
    assert plan.counts()[:2] == (0, 0)
    a = plan.filter(s, 3.0, 4.0)
    b = plan.filter(s, 3.0, 4.0)
    assert len(a) > 0 and np.array_equal(a, b)           # set content is deterministic
    plan.close()


def test_zero_strain_gives_nothing(rbmf):
    import torch
    wl = workload("tiny")
    plan = make_plan(rbmf, wl)
    assert len(plan.filter(torch.zeros(wl["config"].bins, dtype=torch.complex64), 1.0, 1.0)) == 0
    plan.close()


def test_overflow_is_reported_and_bounded(rbmf):
    import torch
    wl = workload("tiny")
    plan = make_plan(rbmf, wl, impl=SCREEN, max_candidates=64, max_triggers=1 << 16)
    plan.filter_async(torch.from_numpy(wl["strain"]).cuda(), 2.0, 2.0)
    nc, nt, st = plan.counts(allow_overflow=True)
    assert st == rbmf.RBMF_ERR_OVERFLOW and nc <= 64      # screened list overflowed; confirmed <= processed
    plan.close()
    plan = make_plan(rbmf, wl, impl=X3, max_candidates=64, max_triggers=16)
    plan.filter_async(torch.from_numpy(wl["strain"]).cuda(), 2.0, 2.0)
    nc, nt, st = plan.counts(allow_overflow=True)
    assert st == rbmf.RBMF_ERR_OVERFLOW and nc > 64
    trig = plan.triggers(allow_overflow=True)
    assert len(trig) <= 16
    with pytest.raises(rbmf.RbmfError):
        plan.counts()
    plan.close()
    # triggers-only overflow: candidate list large enough, trigger list too small
    plan = make_plan(rbmf, wl, max_candidates=1 << 18, max_triggers=16)
    plan.filter_async(torch.from_numpy(wl["strain"]).cuda(), 2.0, 2.0)
    nc, nt, st = plan.counts(allow_overflow=True)
    ref = oracle(wl, 4, 2.0, 2.0)
    assert st == rbmf.RBMF_ERR_OVERFLOW and abs(nt - len(ref["triggers"])) <= max(5, len(ref["near"]) - len(ref["triggers"]))
    plan.close()


def test_sigma_null_uses_coefficient_norm(rbmf):
    import torch
    wl = workload("tiny")
    cfg = wl["config"]
    plan = rbmf.Plan(cfg.N, cfg.fs, cfg.f_low, cfg.k, cfg.T, w=cfg.w, max_candidates=1 << 18, max_triggers=1 << 18)
    plan.set_basis(torch.from_numpy(wl["basis"]))
    plan.set_coeffs(torch.from_numpy(wl["coeffs"]), None)
    got = plan.filter(torch.from_numpy(wl["strain"]), 3.0, 4.0)
    plan.close()
    sig = np.linalg.norm(wl["coeffs"].astype(np.complex128), axis=1).astype(np.float32)
    ref = orc.oracle_filter(wl["strain"], wl["basis"], wl["coeffs"], sig, cfg.N, cfg.fs, cfg.f_low, cfg.w, 3.0, 4.0)
    assert compare.compare_triggers(got, ref, cfg.N, 3.0, 4.0)["ok"]


def test_unit_sigma_is_the_papers_convention(rbmf):
    """sigma_t = 1 (templates 'normalized to unity'): SNRs scale by ||c_t||."""
    import torch
    wl = workload("tiny")
    cfg = wl["config"]
    ones = np.ones(cfg.T, dtype=np.float32)
    plan = rbmf.Plan(cfg.N, cfg.fs, cfg.f_low, cfg.k, cfg.T, w=cfg.w, max_candidates=1 << 18, max_triggers=1 << 18)
    plan.set_basis(torch.from_numpy(wl["basis"]))
    plan.set_coeffs(torch.from_numpy(wl["coeffs"]), torch.from_numpy(ones))
    got = plan.filter(torch.from_numpy(wl["strain"]), 2.0, 2.5)
    plan.close()
    ref = orc.oracle_filter(wl["strain"], wl["basis"], wl["coeffs"], ones, cfg.N, cfg.fs, cfg.f_low, cfg.w, 2.0, 2.5)
    rep = compare.compare_triggers(got, ref, cfg.N, 2.0, 2.5)
    assert rep["ok"] and rep["n_got"] > 0, rep


def test_filter_host_matches_device_call(rbmf):
    import torch
    wl = workload("tiny")
    plan = make_plan(rbmf, wl, max_candidates=1 << 16, max_triggers=1 << 16)
    a = plan.filter(torch.from_numpy(wl["strain"]), 3.0, 4.0)
    pinned = torch.from_numpy(wl["strain"]).pin_memory()
    out, n = plan.filter_host(pinned.numpy(), 3.0, 4.0)
    plan.close()
    assert n == len(a)
    assert np.array_equal(np.sort(out, order=("template", "time")), a)


def test_non_default_stream(rbmf):
    import torch
    wl = workload("tiny")
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        plan = make_plan(rbmf, wl)
        a = plan.filter(torch.from_numpy(wl["strain"]), 3.0, 4.0)
        plan.close()
    ref = oracle(wl, 4, 3.0, 4.0)
    assert compare.compare_triggers(a, ref, wl["config"].N, 3.0, 4.0)["ok"]


def test_explicit_stream_without_entering_it(rbmf):
    """Plan(stream=s) while torch's current stream is another one: the binding's staging copies and read-backs run on
    the plan's stream and inputs produced on the current stream are ordered before their use."""
    import torch
    wl = workload("mini")
    cfg = wl["config"]
    st = torch.cuda.Stream()
    plan = rbmf.Plan(cfg.N, cfg.fs, cfg.f_low, cfg.k, cfg.T, w=cfg.w, max_candidates=1 << 20, max_triggers=1 << 20,
                     stream=st)
    assert torch.cuda.current_stream().cuda_stream != st.cuda_stream
    plan.set_basis(torch.from_numpy(wl["basis"]))
    plan.set_coeffs(torch.from_numpy(wl["coeffs"]), torch.from_numpy(wl["sigma"]))
    # the strain is produced by a kernel on the CURRENT stream right before the call (after a long-running fill)
    big = torch.empty(1 << 28, dtype=torch.float32, device="cuda").normal_()
    s = torch.from_numpy(wl["strain"]).cuda() * (1.0 + 0.0 * big[:1].sum())
    plan.filter_async(s, 3.5, 5.0)
    a = plan.triggers()
    st2 = torch.cuda.Stream()
    plan.set_stream(st2)                                   # ordered after the work on the old stream
    b = plan.filter(torch.from_numpy(wl["strain"]), 3.5, 5.0)
    plan.close()
    ref = oracle(wl, cfg.w, 3.5, 5.0)
    assert compare.compare_triggers(a, ref, cfg.N, 3.5, 5.0)["ok"]
    assert np.array_equal(a, b)
