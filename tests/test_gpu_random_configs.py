"""Seeded random small configurations through the whole path (single calls and batches, both tensor-core modes, every
window the size allows) against the exhaustive fp64 oracle: plan sizes, ragged template counts and band edges that no
named config has."""
import numpy as np
import pytest

from oracle import compare
from oracle import rbmf_oracle as orc
from paper_2110_13115_b200 import workloads as wlm

pytestmark = pytest.mark.gpu


def _cases(n=18):
    rng = np.random.default_rng(20211013)
    out = []
    for i in range(n):
        logn = int(rng.integers(10, 15))
        N = 1 << logn
        fs = float(rng.choice([256.0, 512.0, 1024.0]))
        f_low = float(rng.uniform(0.03, 0.12)) * fs                # a non-integer band edge f_low N / fs
        k = int(rng.choice([16, 32, 48, 64]))
        T = int(rng.integers(max(k, 20), 400))
        ws = [w for w in (1, 2, 4, 8, 16, 32) if N // w >= 128 and w <= 1 << ((logn + 1) // 2)]
        w = int(rng.choice(ws))
        nb = int(rng.integers(1, 4))
        impl = int(rng.choice([0, 2]))
        out.append((i, N, fs, f_low, k, T, w, nb, impl))
    return out


@pytest.mark.parametrize("i,N,fs,f_low,k,T,w,nb,impl", _cases())
def test_random_configuration(built_library, i, N, fs, f_low, k, T, w, nb, impl):
    import torch
    from paper_2110_13115_b200 import rbmf
    cfg = wlm.WorkloadConfig("rand%d" % i, 9000 + i, N, fs, f_low, k, T, w, 1.0, 1.4, 2, 7.0, 14.0)
    wl = wlm.make_workload(cfg, device="cuda")
    strains = np.stack([wlm.make_strain(wl, s)[0] for s in range(nb)])
    # thresholds low enough that noise alone exercises both stages, scaled to the window's attenuation
    rho = orc.snr_series_fft(strains[0], orc.reconstructed_templates(wl["coeffs"], wl["basis"], [0, T // 2, T - 1]),
                             wl["sigma"][[0, T // 2, T - 1]], N, cfg.j_low)
    thr1 = float(np.quantile(np.abs(orc.bin_average(rho, w)), 0.98))
    thr2 = float(np.quantile(np.abs(rho), 0.97))
    plan = rbmf.Plan(N, fs, f_low, k, T, w=w, max_candidates=1 << 20, max_triggers=1 << 20, max_batch=nb)
    plan.set_gemm_impl(impl)
    plan.set_basis(torch.from_numpy(wl["basis"]))
    plan.set_coeffs(torch.from_numpy(wl["coeffs"]), torch.from_numpy(wl["sigma"]))
    got = plan.filter_batch(torch.from_numpy(strains), thr1, thr2)
    cand = plan.candidates()
    plan.close()
    ref = orc.oracle_filter_batch(strains, wl["basis"], wl["coeffs"], wl["sigma"], N, fs, f_low, w, thr1, thr2)
    rep = compare.compare_triggers(got, ref, nb * N, thr1, thr2)
    crep = compare.compare_candidates(cand, ref, nb * N // w, thr1)
    assert rep["ok"] and rep["n_mandatory"] > 20, (rep, thr1, thr2)
    assert crep["ok"] and crep["n_mandatory"] > 20, crep
