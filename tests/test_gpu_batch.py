"""Batched segments and the by-bin stage 2 against the fp64 oracle, plus guard-zone
and repeatability checks that stand in for compute-sanitizer (closed on this pool, profiles/r02_sanitizer.md)."""
import numpy as np
import pytest

from oracle import compare
from oracle import rbmf_oracle as orc
from paper_2110_13115_b200 import workloads as wlm

pytestmark = pytest.mark.gpu

X3, SCREEN = 0, 2


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


def strains_of(wl, n):
    return np.stack([wlm.make_strain(wl, s)[0] for s in range(n)])


def make_plan(rbmf, wl, w=None, impl=SCREEN, max_batch=1, cap=1 << 20):
    import torch
    cfg = wl["config"]
    plan = rbmf.Plan(cfg.N, cfg.fs, cfg.f_low, cfg.k, cfg.T, w=cfg.w if w is None else w, max_candidates=cap,
                     max_triggers=cap, max_batch=max_batch)
    plan.set_gemm_impl(impl)
    plan.set_basis(torch.from_numpy(wl["basis"]))
    plan.set_coeffs(torch.from_numpy(wl["coeffs"]), torch.from_numpy(wl["sigma"]))
    return plan


def batch_oracle(wl, strains, w, thr1, thr2):
    cfg = wl["config"]
    return orc.oracle_filter_batch(strains, wl["basis"], wl["coeffs"], wl["sigma"], cfg.N, cfg.fs, cfg.f_low, w,
                                   thr1, thr2)


@pytest.mark.parametrize("impl", [SCREEN, X3])
@pytest.mark.parametrize("name,nb,max_batch,w,thr", [("tiny", 3, 3, 4, (3.0, 4.0)), ("mini", 3, 4, 8, (3.0, 4.0)),
                                                      ("mini", 2, 2, 1, (4.0, 4.5)), ("mini", 5, 5, 32, (0.5, 3.5))])
def test_batch_against_oracle(rbmf, name, nb, max_batch, w, thr, impl):
    import torch
    wl = workload(name)
    cfg = wl["config"]
    strains = strains_of(wl, nb)
    plan = make_plan(rbmf, wl, w=w, impl=impl, max_batch=max_batch)
    got = plan.filter_batch(torch.from_numpy(strains), *thr)
    cand = plan.candidates()
    ref = batch_oracle(wl, strains, w, *thr)
    rep = compare.compare_triggers(got, ref, nb * cfg.N, *thr)
    crep = compare.compare_candidates(cand, ref, nb * cfg.N // w, thr[0])
    assert rep["ok"] and rep["n_mandatory"] > 0, rep
    assert crep["ok"], crep
    assert len(np.unique(got["time"] // cfg.N)) >= min(nb, 2)   # more than one segment produced triggers
    # beta / beta^avg of the last segment against the oracle's series of that strain alone
    beta = plan.internal("beta", segment=nb - 1)
    ref_beta = orc.basis_series(strains[nb - 1], wl["basis"], cfg.N, cfg.j_low).T
    assert np.abs(beta - ref_beta).max() <= 1e-5
    # a single-segment call on the same plan afterwards reproduces segment 0 of the batch
    one = plan.filter(torch.from_numpy(strains[0]), *thr)
    seg0 = got[got["time"] < cfg.N]
    assert np.array_equal(np.sort(one, order=("template", "time"))[["template", "time"]], seg0[["template", "time"]])
    plan.close()


def test_batch_small_config_two_segments(rbmf):
    import torch
    wl = workload("small")
    cfg = wl["config"]
    strains = strains_of(wl, 2)
    plan = make_plan(rbmf, wl, max_batch=2)
    got = plan.filter_batch(torch.from_numpy(strains), cfg.thr1, cfg.thr2)
    ref = batch_oracle(wl, strains, cfg.w, cfg.thr1, cfg.thr2)
    rep = compare.compare_triggers(got, ref, 2 * cfg.N, cfg.thr1, cfg.thr2)
    crep = compare.compare_candidates(plan.candidates(), ref, 2 * cfg.N // cfg.w, cfg.thr1)
    host, n_host = plan.filter_batch_host(strains, cfg.thr1, cfg.thr2)
    plan.close()
    assert rep["ok"] and rep["n_mandatory"] > 100, rep
    assert crep["ok"], crep
    assert n_host == len(got)
    assert np.array_equal(np.sort(host, order=("template", "time")), got)


@pytest.mark.parametrize("w", [1, 2, 4, 8, 16, 32])
def test_stage2_by_bin_and_per_candidate_kernels_agree(rbmf, w):
    """Both stage-2 kernels pass the oracle comparison on the same call and report the same sets."""
    import torch
    wl = workload("mini")
    cfg = wl["config"]
    thr = ({16: 1.5, 32: 0.5}.get(w, 2.5), 3.5)     # wide windows attenuate the averaged SNR
    ref = orc.oracle_filter(wl["strain"], wl["basis"], wl["coeffs"], wl["sigma"], cfg.N, cfg.fs, cfg.f_low, w, *thr)
    res = []
    for per_cand in (0, 1):
        plan = make_plan(rbmf, wl, w=w)
        plan.diag_set(rbmf.RBMF_DIAG_STAGE2_PER_CANDIDATE, per_cand)
        got = plan.filter(torch.from_numpy(wl["strain"]), *thr)
        rep = compare.compare_triggers(got, ref, cfg.N, *thr)
        crep = compare.compare_candidates(plan.candidates(), ref, cfg.N // w, thr[0])
        assert rep["ok"] and rep["n_mandatory"] > 500, rep
        assert crep["ok"], crep
        res.append(got)
        plan.close()
    a, b = res
    ka, kb = a["template"].astype(np.int64) * cfg.N + a["time"], b["template"].astype(np.int64) * cfg.N + b["time"]
    assert len(np.setxor1d(ka, kb)) <= max(2, rep["tie_band"])      # they may differ only inside the tie band
    common = np.intersect1d(ka, kb, return_indices=True)
    assert np.abs(a["re"][common[1]] - b["re"][common[2]]).max() < 1e-5


def test_dense_bin_with_more_candidates_than_one_work_item(rbmf):
    """thr1 so low that every (template, bin) is a candidate: bins hold T = 300 > 128 candidates (several work items
    per bin, a ragged last one), and the list is exactly T * N/w long."""
    import torch
    wl = workload("mini")
    cfg = wl["config"]
    w, thr = 32, (1e-6, 4.0)
    plan = make_plan(rbmf, wl, w=w, cap=1 << 19)
    got = plan.filter(torch.from_numpy(wl["strain"]), *thr)
    nc, nt, _ = plan.counts()
    assert nc == cfg.T * (cfg.N // w)
    ref = orc.oracle_filter(wl["strain"], wl["basis"], wl["coeffs"], wl["sigma"], cfg.N, cfg.fs, cfg.f_low, w, *thr)
    rep = compare.compare_triggers(got, ref, cfg.N, *thr)
    plan.close()
    assert rep["ok"] and rep["n_got"] == nt and rep["n_mandatory"] > 50, rep


# ------------------------------------------------------------------------------------- guard zones, repeatability
GUARD = 1 << 20


def _guarded_plan(rbmf, wl, **kw):
    """A Plan whose workspace, trigger array and count sit between guard zones of a known pattern."""
    import ctypes
    import torch
    cfg = wl["config"]
    plan = make_plan(rbmf, wl, **kw)
    torch.cuda.synchronize()
    nbytes = plan.workspace_bytes
    big = torch.full((nbytes + 2 * GUARD + 2048,), 0xA5, dtype=torch.uint8, device="cuda")
    base = (big.data_ptr() + GUARD + 1023) // 1024 * 1024
    off = base - big.data_ptr()
    # re-point the plan at the guarded block (invalidates basis / coefficients: set them again)
    st = rbmf.rbmf_plan_set_workspace(plan._h, ctypes.c_void_p(base), nbytes)
    assert st == rbmf.RBMF_OK
    plan._ws = big
    plan.set_basis(torch.from_numpy(wl["basis"]))
    plan.set_coeffs(torch.from_numpy(wl["coeffs"]), torch.from_numpy(wl["sigma"]))
    out = torch.full((plan.max_triggers * 4 + 2 * GUARD // 4,), 0x5A5A5A5A, dtype=torch.int32, device="cuda")
    plan._out = out[GUARD // 4: GUARD // 4 + plan.max_triggers * 4]
    plan._out_guarded = out
    cnt = torch.full((1 + 2 * 1024,), 0x0123456789ABCDEF, dtype=torch.int64, device="cuda")
    plan._n_out = cnt[1024:1025]
    plan._cnt_guarded = cnt
    return plan, big, off, nbytes


def _guards_intact(plan, big, off, nbytes):
    import torch
    torch.cuda.synchronize()
    assert bool((big[:off] == 0xA5).all()) and bool((big[off + nbytes:] == 0xA5).all()), "workspace guard overwritten"
    out = plan._out_guarded
    assert bool((out[: GUARD // 4] == 0x5A5A5A5A).all()) and bool((out[GUARD // 4 + plan.max_triggers * 4:] == 0x5A5A5A5A).all())
    cnt = plan._cnt_guarded
    assert bool((cnt[:1024] == 0x0123456789ABCDEF).all()) and bool((cnt[1025:] == 0x0123456789ABCDEF).all())


@pytest.mark.parametrize("name,w,impl,nb,thr,cap", [
    ("tiny", 4, SCREEN, 1, (3.0, 4.0), 1 << 16), ("tiny", 4, X3, 1, (3.0, 4.0), 1 << 16),
    ("mini", 8, SCREEN, 3, (3.0, 4.0), 1 << 18), ("mini", 1, X3, 2, (4.0, 4.5), 1 << 18),
    ("mini", 32, SCREEN, 1, (0.5, 3.5), 1 << 18),
    ("mini", 8, SCREEN, 2, (1.0, 2.0), 1000),          # both lists overflow: writes must stop at the capacity
])
def test_guard_zones_stay_intact(rbmf, name, w, impl, nb, thr, cap):
    import torch
    wl = workload(name)
    plan, big, off, nbytes = _guarded_plan(rbmf, wl, w=w, impl=impl, max_batch=nb, cap=cap)
    strains = torch.from_numpy(strains_of(wl, nb)).cuda()
    for single_cta in (0, 1):
        plan.diag_set(rbmf.RBMF_DIAG_SINGLE_CTA_SCREEN, single_cta)
        for per_cand in (0, 1):
            plan.diag_set(rbmf.RBMF_DIAG_STAGE2_PER_CANDIDATE, per_cand)
            plan.filter_batch_async(strains, *thr)
            nc, nt, st = plan.counts(allow_overflow=True)
            assert nt > 0 and (st == rbmf.RBMF_ERR_OVERFLOW) == (cap == 1000)
            _guards_intact(plan, big, off, nbytes)
    plan.close()


def test_guarded_calls_repeat_bit_exact(rbmf):
    """20 calls: identical beta bytes and identical sorted lists every time (a race between the FFT's producer, its
    consumer groups and the TMA stores, or in the GEMM's multicast pipeline, would show as run-to-run differences)."""
    import torch
    wl = workload("mini")
    plan, big, off, nbytes = _guarded_plan(rbmf, wl, w=8, max_batch=2, cap=1 << 18)
    strains = torch.from_numpy(strains_of(wl, 2)).cuda()
    first = None
    for _ in range(20):
        plan.filter_batch_async(strains, 3.0, 4.0)
        trig = plan.triggers()
        cand = plan.candidates()
        beta = plan.internal("beta", segment=1)
        cur = (trig.tobytes(), cand.tobytes(), beta.tobytes())
        if first is None:
            first = cur
            assert len(trig) > 100
        assert cur == first
    _guards_intact(plan, big, off, nbytes)
    plan.close()


def test_stage_time_history_of_calls_enqueued_back_to_back(rbmf):
    """rbmf_get_stage_ms_history: 70 timed calls enqueued without a host synchronisation in between; afterwards the
    plan still has the stage events of the last 64 -- every stage time positive, the parts adding up to the whole
    (same events), the sum of the per-call totals no longer than the span an outer pair of events measures -- and
    refuses to go further back than it has calls, or than its ring is long."""
    import torch
    wl = workload("mini")
    strain = torch.from_numpy(wl["strain"]).cuda()
    plan = make_plan(rbmf, wl)
    plan.filter_async(strain, 3.0, 4.0)          # untimed call: not part of the history
    plan.set_timing(True)
    with pytest.raises(rbmf.RbmfError) as info:
        plan.stage_ms_history(1)
    assert info.value.status == rbmf.RBMF_ERR_STATE
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    for calls in (5, 70):
        plan.set_timing(True)                    # restarts the history
        e0.record(plan.stream)
        for _ in range(calls):
            plan.filter_async(strain, 3.0, 4.0)
        e1.record(plan.stream)
        plan.stream.synchronize()
        hist = plan.stage_ms_history(min(calls, 64))
        assert len(hist) == min(calls, 64)
        for ms in hist:
            assert ms["fft"] > 0 and ms["gemm"] > 0 and ms["stage2"] > 0
            assert abs(ms["fft"] + ms["gemm"] + ms["stage2"] - ms["total"]) < 2e-3
        assert sum(ms["total"] for ms in hist) <= e0.elapsed_time(e1) * 1.001
        last = plan.stage_ms()
        assert last == hist[-1]
        if calls < 64:
            with pytest.raises(rbmf.RbmfError):
                plan.stage_ms_history(calls + 1)
    plan.close()


def test_scheduling_overrides_change_the_order_not_the_result(rbmf):
    """RBMF_DIAG_FFT_CHUNK_MAJOR / _FFT_LOOKAHEAD / _GEMM_GROUP (rbmf_diag_set; environment variables in earlier
    builds) only reorder the work: beta is bit-identical, candidates and triggers are the same sets."""
    wl = workload("mini")
    import torch
    nb, thr = 3, (3.0, 4.0)
    strains = torch.from_numpy(strains_of(wl, nb)).cuda()
    results = []
    for chunk_major, lookahead, group in ((0, 0, 0), (1, 1, 1), (0, 3, 2)):
        plan = make_plan(rbmf, wl, max_batch=nb)
        plan.diag_set(rbmf.RBMF_DIAG_FFT_CHUNK_MAJOR, chunk_major)
        plan.diag_set(rbmf.RBMF_DIAG_FFT_LOOKAHEAD, lookahead)
        plan.diag_set(rbmf.RBMF_DIAG_GEMM_GROUP, group)
        plan.filter_batch_async(strains, *thr)
        trig = np.sort(plan.triggers(), order=("template", "time"))
        cand = np.sort(plan.candidates(), order=("template", "bin"))
        results.append((trig.tobytes(), cand.tobytes(), plan.internal("beta", segment=nb - 1).tobytes()))
        assert len(trig) > 100
        plan.close()
    assert results[1] == results[0] and results[2] == results[0]


# ------------------------------------------------------------------------------------- the step before the path
@pytest.mark.parametrize("N", [1024, 2048, 16384, 131072, 1 << 20])
def test_prepare_strain_against_oracle(rbmf, N):
    """rbmf_prepare_strain vs the oracle's fp64 forward DFT + whitening, all lengths' splits
    (odd and even log2 N), two segments, with and without a whitening array.  Bar per bin, from the arithmetic (fp32
    radix-2 stages with fp64-computed twiddles): 3e-6 of the bin's own magnitude (~log2(N) 2^-24), plus 4e-6 of the
    noise floor's rms sqrt(N), plus 2^-23 of the tallest spectral line -- the real-input split combines bin j with bin
    N/2 - j of the packed transform, so a line's rounding error shows up at its mirror bin."""
    import torch
    rng = np.random.default_rng(N)
    x = rng.standard_normal((2, N)).astype(np.float32)
    x[1] += (3.0 * np.cos(2 * np.pi * 37 * np.arange(N) / N + 0.4)).astype(np.float32)
    inv_asd = rng.uniform(0.5, 2.0, N // 2 + 1).astype(np.float32)
    plan = rbmf.Plan(N, 1024.0, 30.0, 16, 8, w=1, max_candidates=1024, max_triggers=1024, max_batch=2)
    for wht in (None, inv_asd):
        got = plan.prepare_strain(torch.from_numpy(x).cuda(), None if wht is None else torch.from_numpy(wht).cuda())
        plan.stream.synchronize()
        ref = orc.strain_from_time_series(x, wht)
        err = np.abs(got.cpu().numpy() - ref)
        # per bin: relative to that bin's own magnitude (the cosine's line is 1.5 N high) plus the noise floor's rms
        gain = 2.0 if wht is not None else 1.0
        bar = 3e-6 * np.abs(ref) + 4e-6 * np.sqrt(N) * gain + 2.0 ** -23 * np.abs(ref).max(axis=1, keepdims=True) * gain
        assert (err <= bar).all(), (N, float((err / bar).max()))
    one = plan.prepare_strain(torch.from_numpy(x[1:2]).cuda(), torch.from_numpy(inv_asd).cuda())
    assert np.array_equal(one.cpu().numpy()[0], got.cpu().numpy()[1])
    plan.close()


def test_time_series_to_triggers(rbmf):
    """Front end + path: coloured time series -> rbmf_prepare_strain -> rbmf_filter_batch, against the oracle fed
    with its own fp64 transform of the same float32 series."""
    import torch
    wl = workload("mini")
    cfg = wl["config"]
    nb, thr = 3, (3.0, 4.0)
    xs, inv_asd = zip(*[wlm.make_time_series(wl, s) for s in range(nb)])
    x = np.stack(xs)
    plan = make_plan(rbmf, wl, max_batch=nb)
    strain = plan.prepare_strain(torch.from_numpy(x).cuda(), torch.from_numpy(inv_asd[0]).cuda())
    plan.filter_batch_async(strain, *thr)
    got = plan.triggers()
    ref_strain = orc.strain_from_time_series(x, inv_asd[0])
    # the whitened spectrum is the frequency-domain workload itself, up to the float32 rounding of x
    assert np.abs(ref_strain[0, cfg.j_low:cfg.N // 2] - wl["strain"][cfg.j_low:cfg.N // 2]).max() < 2e-3
    ref = batch_oracle(wl, ref_strain.astype(np.complex64), cfg.w, *thr)
    rep = compare.compare_triggers(got, ref, nb * cfg.N, *thr)
    plan.close()
    assert rep["ok"] and rep["n_mandatory"] > 100, rep


# ------------------------------------------------------------------------------------- many sub-banks (f3)
def test_bank_set_of_three_sub_banks(rbmf):
    """Three sub-banks with different basis sizes, template counts and windows (Table I) against one
    strain: one call, one trigger list with global template ids, equal to the oracle's union."""
    import torch
    base = wlm.CONFIGS["mini"]
    subs = wlm.make_subbanks(base, [(1.0, 1.07, 32, 300, 8), (1.07, 1.14, 48, 130, 4), (1.14, 1.2, 16, 257, 8)],
                             device="cuda")
    strain = subs[0]["strain"]
    thr = (3.0, 4.0)
    plans = []
    for i, wl in enumerate(subs):
        cfg = wl["config"]
        p = make_plan(rbmf, wl, w=cfg.w, impl=(SCREEN, X3, SCREEN)[i], cap=1 << 18)
        plans.append(p)
    bs = rbmf.BankSet(plans, max_triggers=1 << 20)
    got = bs.filter(torch.from_numpy(strain), *thr)
    nc, nt, tot, st = bs.counts()
    ref = orc.oracle_filter_banks(strain, [dict(basis=w_["basis"], coeffs=w_["coeffs"], sigma=w_["sigma"],
                                                w=w_["config"].w) for w_ in subs], base.N, base.fs, base.f_low, *thr)
    rep = compare.compare_triggers(got, ref, base.N, *thr)
    assert rep["ok"] and rep["n_mandatory"] > 500, rep
    assert st == rbmf.RBMF_OK and tot == len(got) == sum(nt)
    bounds = np.cumsum([0] + [w_["config"].T for w_ in subs])
    for m in range(3):
        in_m = (got["template"] >= bounds[m]) & (got["template"] < bounds[m + 1])
        assert in_m.sum() == nt[m] > 0
        crep = compare.compare_candidates(plans[m].candidates(), ref["per_bank"][m], base.N // subs[m]["config"].w, thr[0])
        assert crep["ok"], crep
    # the same plans still work on their own afterwards, with local template ids
    one = plans[1].filter(torch.from_numpy(strain), *thr)
    sel = got[(got["template"] >= bounds[1]) & (got["template"] < bounds[2])]
    assert np.array_equal(one["time"], sel["time"]) and np.array_equal(one["template"] + bounds[1], sel["template"])
    # a second call reuses the set
    got2 = bs.filter(torch.from_numpy(strain), *thr)
    assert np.array_equal(got2, got)
    bs.close()
    for p in plans:
        p.close()


@pytest.mark.parametrize("name,nb,calls", [("small", 1, 400), ("small", 3, 150), ("mini", 2, 600)])
def test_soak_hundreds_of_calls_give_identical_digests(rbmf, name, nb, calls):
    """Hundreds of back-to-back calls: an order-independent digest of the trigger list, of the candidate list and of
    the raw beta bytes must never change (no sanitizer on this pool: a rare race in the FFT's hand-offs, the GEMM's
    multicast pipeline or the by-bin regrouping would show here)."""
    import ctypes
    import torch
    wl = workload(name)
    cfg = wl["config"]
    strains = torch.from_numpy(strains_of(wl, nb)).cuda()
    plan = make_plan(rbmf, wl, max_batch=nb, cap=1 << 21)
    thr = (cfg.thr1, cfg.thr2) if name == "small" else (3.0, 4.0)

    def digest():
        rows = plan.triggers_device().to(torch.int64)
        c = plan.candidates_device().to(torch.int64)
        p, nbytes = ctypes.c_void_p(), ctypes.c_size_t()
        assert rbmf.rbmf_get_internal(plan._h, 0, ctypes.byref(p), ctypes.byref(nbytes)) == rbmf.RBMF_OK
        off = p.value - plan._ws.data_ptr()
        beta = plan._ws[off: off + nbytes.value].view(torch.int32).to(torch.int64).sum()
        mix = lambda r: ((r[:, 0] * 1000003 + r[:, 1]) * 998244353 + r[:, 2] * 7919 + r[:, 3]).sum()
        return int(mix(rows)), int(rows.shape[0]), int(mix(c)), int(c.shape[0]), int(beta)

    first = None
    for _ in range(calls):
        plan.filter_batch_async(strains, *thr)
        d = digest()
        if first is None:
            first = d
            assert d[1] > 100
        assert d == first
    plan.close()
