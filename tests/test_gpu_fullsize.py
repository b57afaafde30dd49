"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times ("tiers").

Exhaustive fp64 reconstruction costs 8 T k N flops (2e16 at Paper scale), so at these sizes
  (i)   soundness: reported triggers, sampled (1 %, capped), are re-evaluated pointwise by the literal O(|B|) sum of
        Eq. 4 (`oracle.evaluate_points`, no FFT) -- value, and membership in the allowed set;
  (ii)  completeness: on a template subset S = injected templates + their +-8 nearest neighbours in chirp mass + seeded
        random templates, the exhaustive oracle's sets must match the GPU's restricted to S under the tie-band rule --
        triggers AND first-stage candidates, at the config's own thresholds.  The GPU lists are restricted to S on the
        device (`torch.isin` on the template column), so list sizes of 1e8-1e9 records never cross PCIe;
  (iii) Paper config only: an exhaustive cross-check of EVERY (template, bin) against a torch complex128 restatement
        of the basis route on the GPU -- labelled as such: it is NOT the oracle (it shares the basis-then-GEMM
        structure with the library, though no code), it is never timed, and it exists to catch tile-local defects
        (a raster-group edge, the ragged last template block, the odd partner CTA) outside the sampled blocks.
"""
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


def workload(name):
    if name not in _WL:
        _WL.clear()                                       # one full-size workload on the host at a time
        _WL[name] = wlm.make_workload(wlm.CONFIGS[name], device="cuda")
    return _WL[name]


def records(t, dtype):
    """(n, 4) int32 CUDA tensor -> structured numpy array."""
    a = t.contiguous().cpu().numpy()
    return a.view(dtype).reshape(-1).copy() if len(a) else np.empty(0, dtype=dtype)


def select_templates(rows, subset, T, step=1 << 26):
    """Rows of an (n, 4) int32 record tensor whose template (column 0) is in `subset`, selected on the device in
    slices (a look-up table over the T templates; nothing proportional to n is allocated besides the slice mask)."""
    import torch
    lut = torch.zeros(T, dtype=torch.bool, device=rows.device)
    lut[torch.from_numpy(np.asarray(subset, dtype=np.int64)).to(rows.device)] = True
    parts = []
    for a in range(0, rows.shape[0], step):
        blk = rows[a:a + step]
        parts.append(blk[lut[blk[:, 0].long()]])
    return torch.cat(parts) if parts else rows[:0]


def template_subset(wl, n_random, neighbours=8, extra=()):
    cfg = wl["config"]
    rng = np.random.default_rng(5)
    order = np.argsort(wl["mc"])
    rank = np.empty(cfg.T, dtype=np.int64)
    rank[order] = np.arange(cfg.T)
    sel = set(int(t) for t in extra)
    for inj in wl["injections"]:
        r = rank[inj["template"]]
        sel.update(order[max(0, r - neighbours): r + neighbours + 1].tolist())
    sel.update(rng.choice(cfg.T, size=min(n_random, cfg.T), replace=False).tolist())
    sel.add(cfg.T - 1)                                   # the ragged last template block
    return np.array(sorted(sel), dtype=np.int64)


def run_and_check(rbmf, name, impl, w=None, thr1=None, thr2=None, n_random=1024, neighbours=8, max_points=768,
                  capacity=1 << 22, subset_from_triggers=0):
    import torch
    wl = workload(name)
    cfg = wl["config"]
    w = cfg.w if w is None else w
    thr1 = cfg.thr1 if thr1 is None else thr1
    thr2 = cfg.thr2 if thr2 is None else thr2
    torch.cuda.empty_cache()
    plan = rbmf.Plan(cfg.N, cfg.fs, cfg.f_low, cfg.k, cfg.T, w=w, max_candidates=capacity, max_triggers=capacity)
    plan.set_gemm_impl(impl)
    plan.set_basis(torch.from_numpy(wl["basis"]))
    plan.set_coeffs(torch.from_numpy(wl["coeffs"]), torch.from_numpy(wl["sigma"]))
    plan.filter_async(torch.from_numpy(wl["strain"]).cuda(), thr1, thr2)
    nc, nt, st = plan.counts(allow_overflow=True)
    assert st == rbmf.RBMF_OK, "lists overflowed: %d screened, %d triggers" % (plan.screened_count(), nt)
    trig_dev, cand_dev = plan.triggers_device(), plan.candidates_device()
    assert trig_dev.shape[0] == nt and cand_dev.shape[0] == nc

    extra = ()
    if subset_from_triggers and nt:
        extra = torch.unique(trig_dev[:, 0])[:subset_from_triggers].cpu().numpy()
    subset = template_subset(wl, n_random, neighbours, extra)
    got = np.sort(records(select_templates(trig_dev, subset, cfg.T), rbmf.TRIGGER_DTYPE), order=("template", "time"))
    cand = np.sort(records(select_templates(cand_dev, subset, cfg.T), rbmf.CANDIDATE_DTYPE), order=("template", "bin"))
    # (i) soundness sample over ALL reported triggers
    rng = np.random.default_rng(7)
    n_pts = int(min(max_points, max(16, nt // 100), nt))
    pick = torch.from_numpy(np.unique(rng.integers(0, max(nt, 1), size=n_pts))).cuda() if nt else None
    pts = records(trig_dev[pick], rbmf.TRIGGER_DTYPE) if nt else np.empty(0, dtype=rbmf.TRIGGER_DTYPE)
    plan.close()
    del trig_dev, cand_dev
    torch.cuda.empty_cache()

    basis128 = wl["basis"].astype(np.complex128)          # converted once; the oracle treats the values as exact
    coeffs128 = wl["coeffs"].astype(np.complex128)
    for rec in pts:
        t, n = int(rec["template"]), int(rec["time"])
        rho, rbar = orc.evaluate_points(wl["strain"], basis128, coeffs128, wl["sigma"], cfg.N, cfg.fs, cfg.f_low, w,
                                        t, [n])
        val = complex(rec["re"], rec["im"])
        assert abs(abs(val) - abs(rho[0])) <= 1e-3 * abs(rho[0]), (t, n, val, rho[0])
        assert abs(np.angle(val * np.conj(rho[0]))) <= 1e-3
        assert abs(rho[0]) >= thr2 * (1 - 1e-3) and abs(rbar[0]) >= thr1 * (1 - 1e-3)
    # (ii) completeness on the subset
    ref = orc.oracle_filter(wl["strain"], basis128, coeffs128, wl["sigma"], cfg.N, cfg.fs, cfg.f_low, w, thr1, thr2,
                            templates=subset)
    rep = compare.compare_triggers(got, ref, cfg.N, thr1, thr2)
    crep = compare.compare_candidates(cand, ref, cfg.N // w, thr1)
    print("%s impl=%d w=%d thr=%g/%g: %d candidates, %d triggers on the device; subset of %d templates: %s | %s; "
          "%d points re-evaluated" % (name, impl, w, thr1, thr2, nc, nt, len(subset), rep, crep, len(pts)))
    assert rep["ok"], rep
    assert crep["ok"], crep
    return rep, crep, nc, nt


@pytest.mark.parametrize("impl", [SCREEN, X3])
def test_paper_scale_sampled(rbmf, impl):
    """BASELINE.json configs[2] (N = 524288, k = 256, T = 20000, w = 8, 5 / 6; what bench.py times): injected +- 8
    chirp-mass neighbours + 1024 random templates exhaustively, 1 % of the triggers pointwise."""
    rep, crep, nc, nt = run_and_check(rbmf, "paper", impl)
    assert rep["n_mandatory"] > 1000 and crep["n_mandatory"] > 100


@pytest.mark.parametrize("impl", [SCREEN, X3])
def test_large_bank_at_its_own_thresholds(rbmf, impl):
    """BASELINE.json configs[3] (N = 262144, k = 256, T = 100000, 100 injections) at 5 / 6: this wide bank answers its
    loud injections with ~2.6e8 candidates and ~8.8e8 triggers; the lists (2^30 records each) stay on the device and
    only the sampled templates' records are shipped.  Both tensor-core modes: the fp16 screen + fp32 confirm, and the
    literal bf16x3 GEMM."""
    rep, crep, nc, nt = run_and_check(rbmf, "large", impl, n_random=64, neighbours=2, max_points=256,
                                      capacity=1 << 30)
    assert nc > 1e8 and nt > 1e8
    assert rep["n_mandatory"] > 1000


@pytest.mark.parametrize("name,w,thr1,thr2,capacity", [
    ("sweep_k512_T100000", 8, 5.0, 6.0, 1 << 22),
    ("sweep_k512_T100000", 8, 3.5, 4.5, 1 << 26),
    ("sweep_k32_T1000", 8, 3.5, 4.5, 1 << 22),
    ("sweep_k256_T10000", 1, 5.0, 6.0, 1 << 22),
    ("sweep_k256_T10000", 8, 3.5, 4.5, 1 << 24),
    ("sweep_k128_T10000", 16, 3.0, 4.5, 1 << 24),
])
def test_sweep_grid_points(rbmf, name, w, thr1, thr2, capacity):
    """BASELINE.json configs[4] (N = 2^20, pure noise): the corners of the (k, T) grid and the flat case w = 1.  Noise
    alone yields few triggers at 5 / 6, so the completeness subset also takes templates that reported something."""
    rep, crep, nc, nt = run_and_check(rbmf, name, SCREEN, w=w, thr1=thr1, thr2=thr2, n_random=24, neighbours=0,
                                      max_points=96, capacity=capacity, subset_from_triggers=24)
    assert nc > 0
    if thr1 < 5.0:
        assert rep["n_mandatory"] > 0 and crep["n_mandatory"] > 0


@pytest.mark.parametrize("name", [n for n in wlm.SWEEP_NAMES])
def test_every_sweep_grid_point_at_w8(rbmf, name):
    """All 15 points of BASELINE.json configs[4] (k in 32..512 x T in 1e3..1e5, N = 2^20, pure noise) at the window the
    bench times (w = 8), not only the corners: thresholds 3.5 / 4.5 so that noise alone gives non-empty mandatory sets;
    16 random templates + 16 that reported something + the ragged last one exhaustively, up to 48 triggers pointwise."""
    rep, crep, nc, nt = run_and_check(rbmf, name, SCREEN, w=8, thr1=3.5, thr2=4.5, n_random=16, neighbours=0,
                                      max_points=48, capacity=1 << 26, subset_from_triggers=16)
    assert nc > 0 and rep["n_mandatory"] > 0 and crep["n_mandatory"] > 0


def test_k1024_exhaustive(rbmf):
    """The largest basis the plan accepts (k = 1024: 256 FFT chunks, 32 K blocks), exhaustively on a mini-sized case."""
    import torch
    cfg = wlm.CONFIGS["mini"].replace(k=1024, T=1100, index=77, mc_lo=1.0, mc_hi=3.0)
    wl = wlm.make_workload(cfg, device="cuda")
    for impl, thr1 in ((SCREEN, 3.0), (X3, 3.0)):
        plan = rbmf.Plan(cfg.N, cfg.fs, cfg.f_low, cfg.k, cfg.T, w=cfg.w, max_candidates=1 << 22, max_triggers=1 << 22)
        plan.set_gemm_impl(impl)
        plan.set_basis(torch.from_numpy(wl["basis"]))
        plan.set_coeffs(torch.from_numpy(wl["coeffs"]), torch.from_numpy(wl["sigma"]))
        got = plan.filter(torch.from_numpy(wl["strain"]), thr1, 4.5)
        cand = plan.candidates()
        plan.close()
        ref = orc.oracle_filter(wl["strain"], wl["basis"], wl["coeffs"], wl["sigma"], cfg.N, cfg.fs, cfg.f_low, cfg.w,
                                thr1, 4.5)
        rep = compare.compare_triggers(got, ref, cfg.N, thr1, 4.5)
        crep = compare.compare_candidates(cand, ref, cfg.N // cfg.w, thr1)
        assert rep["ok"] and rep["n_mandatory"] > 0, rep
        assert crep["ok"] and crep["n_mandatory"] > 100, crep


# ------------------------------------------------------------------------- (iii) exhaustive cross-check, NOT the oracle
def torch_fp64_basis_route(wl, w, thr1, thr2, t_chunk=2048):
    """torch complex128 restatement of Eq. 6-7 + Eq. 9 + the two thresholds on the GPU: beta by torch.fft.ifft,
    averaged series by one ZGEMM per template chunk over ALL (template, bin), stage 2 on the bins that pass.
    Returns a dict shaped like oracle_filter's (triggers, candidates, near, cand_near)."""
    import torch
    cfg = wl["config"]
    N, k, T = cfg.N, cfg.k, cfg.T
    dev = "cuda"
    slack = 1.0 - 2e-3
    d = torch.from_numpy(wl["strain"]).to(dev).to(torch.complex128)
    B = torch.from_numpy(wl["basis"]).to(dev)
    G = torch.zeros((k, N), dtype=torch.complex128, device=dev)
    G[:, cfg.j_low:N // 2] = d[None, cfg.j_low:N // 2] * B[:, cfg.j_low:N // 2].to(torch.complex128).conj()
    del B
    beta = torch.fft.ifft(G, dim=1) * (N * (2.0 / N) ** 0.5)              # (k, N): unnormalised inverse DFT times s
    del G
    bavg = beta.view(k, N // w, w).mean(dim=2)                             # (k, N/w)
    A = torch.from_numpy(wl["coeffs"]).to(dev).to(torch.complex128).conj() / \
        torch.from_numpy(wl["sigma"]).to(dev).to(torch.float64)[:, None]  # (T, k): conj(c)/sigma
    ct, cb, cv = [], [], []
    for a in range(0, T, t_chunk):
        R = A[a:a + t_chunk] @ bavg                                        # (chunk, N/w) complex128
        idx = torch.nonzero(R.abs() >= thr1 * slack)
        ct.append(idx[:, 0] + a); cb.append(idx[:, 1]); cv.append(R[idx[:, 0], idx[:, 1]])
        del R
    ct, cb, cv = torch.cat(ct), torch.cat(cb), torch.cat(cv)
    # stage 2 on every near-candidate bin
    tt, tn, tv, ta = [], [], [], []
    step = 1 << 16
    for a in range(0, len(ct), step):
        t_, b_, v_ = ct[a:a + step], cb[a:a + step], cv[a:a + step]
        cols = (b_[:, None] * w + torch.arange(w, device=dev)[None, :])    # (m, w) sample indices
        seg = beta[:, cols.reshape(-1)].view(k, len(t_), w)                # (k, m, w)
        rho = torch.einsum("mk,kmw->mw", A[t_], seg)
        hit = torch.nonzero(rho.abs() >= thr2 * slack)
        tt.append(t_[hit[:, 0]]); tn.append(cols[hit[:, 0], hit[:, 1]]); tv.append(rho[hit[:, 0], hit[:, 1]])
        ta.append(v_.abs()[hit[:, 0]])
    tt, tn, tv, ta = torch.cat(tt), torch.cat(tn), torch.cat(tv), torch.cat(ta)

    trig_dt = np.dtype([("template", np.int64), ("time", np.int64), ("re", np.float64), ("im", np.float64),
                        ("avg_abs", np.float64)])
    cand_dt = np.dtype([("template", np.int64), ("bin", np.int64), ("re", np.float64), ("im", np.float64)])
    near = np.empty(len(tt), dtype=trig_dt)
    near["template"], near["time"] = tt.cpu().numpy(), tn.cpu().numpy()
    near["re"], near["im"], near["avg_abs"] = tv.real.cpu().numpy(), tv.imag.cpu().numpy(), ta.cpu().numpy()
    cnear = np.empty(len(ct), dtype=cand_dt)
    cnear["template"], cnear["bin"] = ct.cpu().numpy(), cb.cpu().numpy()
    cnear["re"], cnear["im"] = cv.real.cpu().numpy(), cv.imag.cpu().numpy()
    cands = cnear[np.hypot(cnear["re"], cnear["im"]) >= thr1]
    trig = near[(near["avg_abs"] >= thr1) & (np.hypot(near["re"], near["im"]) >= thr2)]
    return {"triggers": trig, "candidates": cands, "near": near, "cand_near": cnear}


def test_torch_route_agrees_with_the_oracle_on_small():
    """The cross-check's own pin: on a config the oracle covers exhaustively it reproduces the oracle's sets exactly
    (both are fp64; they differ by rounding order only) -- so what (iii) compares the library with is sound."""
    wl = wlm.make_workload(wlm.CONFIGS["mini"], device="cuda")
    cfg = wl["config"]
    ref = orc.oracle_filter(wl["strain"], wl["basis"], wl["coeffs"], wl["sigma"], cfg.N, cfg.fs, cfg.f_low, cfg.w,
                            3.5, 5.0)
    alt = torch_fp64_basis_route(wl, cfg.w, 3.5, 5.0, t_chunk=128)
    for key, fields in (("triggers", ("template", "time")), ("candidates", ("template", "bin")),
                        ("near", ("template", "time")), ("cand_near", ("template", "bin"))):
        a = np.sort(alt[key], order=fields)
        b = np.sort(ref[key], order=fields)
        assert len(a) == len(b) > 0 and all(np.array_equal(a[f], b[f]) for f in fields), key
        assert np.abs((a["re"] + 1j * a["im"]) - (b["re"] + 1j * b["im"])).max() < 1e-10


def test_paper_scale_exhaustive_fp64_crosscheck_not_the_oracle(rbmf):
    """Every (template, bin) and every trigger of the Paper config against the torch complex128 basis route above
    (2.7e15 fp64 flops on the GPU).  Labelled cross-check: the oracle proper is (i) + (ii)."""
    import torch
    wl = workload("paper")
    cfg = wl["config"]
    plan = rbmf.Plan(cfg.N, cfg.fs, cfg.f_low, cfg.k, cfg.T, w=cfg.w, max_candidates=1 << 22, max_triggers=1 << 22)
    plan.set_basis(torch.from_numpy(wl["basis"]))
    plan.set_coeffs(torch.from_numpy(wl["coeffs"]), torch.from_numpy(wl["sigma"]))
    got = plan.filter(torch.from_numpy(wl["strain"]), cfg.thr1, cfg.thr2)
    cand = plan.candidates()
    plan.close()
    torch.cuda.empty_cache()
    alt = torch_fp64_basis_route(wl, cfg.w, cfg.thr1, cfg.thr2)
    rep = compare.compare_triggers(got, alt, cfg.N, cfg.thr1, cfg.thr2)
    crep = compare.compare_candidates(cand, alt, cfg.N // cfg.w, cfg.thr1)
    print("paper exhaustive cross-check:", rep, crep)
    assert rep["ok"] and rep["n_mandatory"] > 100000, rep
    assert crep["ok"] and crep["n_mandatory"] > 50000, crep
    _WL.clear()


# --------------------------------------------------------------------------------- 8(f) rows at Paper scale
def test_paper_scale_batch_of_two_equals_two_calls_and_oracle_on_segment_one(rbmf):
    """rbmf_filter_batch at BASELINE configs[2] sizes: the batch's lists, cut per segment, are exactly the lists of
    single-segment calls (same kernels, the segments' bins are 128-aligned blocks of the GEMM's M dimension), and
    segment 1 -- a strain no single-segment test sees -- passes the oracle comparison on a template sample."""
    import torch
    wl = workload("paper")
    cfg = wl["config"]
    strains = np.stack([wlm.make_strain(wl, s)[0] for s in range(2)])
    torch.cuda.empty_cache()
    plan = rbmf.Plan(cfg.N, cfg.fs, cfg.f_low, cfg.k, cfg.T, w=cfg.w, max_candidates=1 << 22, max_triggers=1 << 22,
                     max_batch=2)
    plan.set_basis(torch.from_numpy(wl["basis"]))
    plan.set_coeffs(torch.from_numpy(wl["coeffs"]), torch.from_numpy(wl["sigma"]))
    sd = torch.from_numpy(strains).cuda()
    plan.filter_batch_async(sd, cfg.thr1, cfg.thr2)
    both = plan.triggers()
    cands = plan.candidates()
    singles = []
    for s in range(2):
        plan.filter_async(sd[s], cfg.thr1, cfg.thr2)
        singles.append((plan.triggers(), plan.candidates()))
    plan.close()
    for s in range(2):
        seg = both[(both["time"] >= s * cfg.N) & (both["time"] < (s + 1) * cfg.N)].copy()
        seg["time"] -= s * cfg.N
        assert len(seg) > 1000 and np.array_equal(seg, singles[s][0])
        cseg = cands[(cands["bin"] >= s * (cfg.N // cfg.w)) & (cands["bin"] < (s + 1) * (cfg.N // cfg.w))].copy()
        cseg["bin"] -= s * (cfg.N // cfg.w)
        assert np.array_equal(cseg, singles[s][1])
    subset = np.unique(singles[1][0]["template"])[:: max(1, len(np.unique(singles[1][0]["template"])) // 48)]
    subset = np.union1d(subset, np.random.default_rng(3).choice(cfg.T, 64, replace=False))
    ref = orc.oracle_filter(strains[1], wl["basis"].astype(np.complex128), wl["coeffs"].astype(np.complex128), wl["sigma"],
                            cfg.N, cfg.fs, cfg.f_low, cfg.w, cfg.thr1, cfg.thr2, templates=subset)
    got = singles[1][0]
    rep = compare.compare_triggers(got[np.isin(got["template"], subset)], ref, cfg.N, cfg.thr1, cfg.thr2)
    assert rep["ok"] and rep["n_mandatory"] > 100, rep


def test_paper_scale_template_routes_sampled(rbmf):
    """The paper's template routes at BASELINE configs[2] sizes (T = 20000 reconstructed templates = 42 GB, slab 256):
    the first stage by templates (Eq. 10-12) gives the basis route's candidates and triggers; the flat template method's
    triggers match the oracle's Eq. 4 series on a template sample."""
    import torch
    wl = workload("paper")
    cfg = wl["config"]
    torch.cuda.empty_cache()
    c = torch.from_numpy(wl["coeffs"]).cuda()
    b = torch.from_numpy(wl["basis"]).cuda()
    tpl = torch.empty((cfg.T, cfg.bins), dtype=torch.complex64, device="cuda")
    for a in range(0, cfg.T, 2048):
        tpl[a:a + 2048] = c[a:a + 2048] @ b                   # input synthesis: h'_t = sum_k c_tk b_k
    del c, b
    plan = rbmf.Plan(cfg.N, cfg.fs, cfg.f_low, cfg.k, cfg.T, w=cfg.w, max_candidates=1 << 22, max_triggers=1 << 22,
                     template_slab=256)
    plan.set_basis(torch.from_numpy(wl["basis"]))
    plan.set_coeffs(torch.from_numpy(wl["coeffs"]), torch.from_numpy(wl["sigma"]))
    plan.set_templates(tpl, torch.from_numpy(wl["sigma"]))
    sd = torch.from_numpy(wl["strain"]).cuda()
    plan.filter_async(sd, cfg.thr1, cfg.thr2)
    base_t, base_c = plan.triggers(), plan.candidates()
    plan.set_stage1_route(rbmf.RBMF_STAGE1_TEMPLATES)
    plan.filter_async(sd, cfg.thr1, cfg.thr2)
    tm_t, tm_c = plan.triggers(), plan.candidates()
    key = lambda r, f, n: r["template"].astype(np.int64) * n + r[f]
    # the two routes may differ only at threshold ties (fp32 rounding of different summation orders)
    assert len(np.setxor1d(key(base_c, "bin", cfg.N), key(tm_c, "bin", cfg.N))) <= max(8, len(base_c) // 2000)
    assert len(np.setxor1d(key(base_t, "time", cfg.N), key(tm_t, "time", cfg.N))) <= max(8, len(base_t) // 2000)
    common = np.intersect1d(key(base_c, "bin", cfg.N), key(tm_c, "bin", cfg.N), return_indices=True)
    assert np.abs(base_c["re"][common[1]] - tm_c["re"][common[2]]).max() < 2e-4     # averaged SNR values agree
    flat = plan.filter_flat(sd, cfg.thr2)
    subset = np.unique(flat["template"])[:: max(1, len(np.unique(flat["template"])) // 24)][:32]
    ref = orc.template_method_triggers(wl["strain"], tpl[torch.from_numpy(subset).cuda()].cpu().numpy(), wl["sigma"][subset],
                                       cfg.N, cfg.fs, cfg.f_low, cfg.thr2)
    for k_ in ("triggers", "near"):
        ref[k_]["template"] = subset[ref[k_]["template"]]
    frep = compare.compare_triggers(flat[np.isin(flat["template"], subset)], ref, cfg.N, 1.0, cfg.thr2)
    plan.close()
    del tpl
    torch.cuda.empty_cache()
    assert frep["ok"] and frep["n_mandatory"] > 100, frep
    assert len(flat) >= len(base_t)                              # the hierarchical set is a subset of the flat one
