"""The seeded input generator: determinism, shapes, and that extra strain segments keep the bank."""
import numpy as np

from paper_2110_13115_b200 import workloads as wlm


def test_tiny_workload_is_deterministic_and_shaped():
    a = wlm.make_workload(wlm.CONFIGS["tiny"])
    b = wlm.make_workload(wlm.CONFIGS["tiny"])
    cfg = a["config"]
    assert a["strain"].shape == (cfg.bins,) and a["strain"].dtype == np.complex64
    assert a["basis"].shape == (cfg.k, cfg.bins) and a["basis"].dtype == np.complex64
    assert a["coeffs"].shape == (cfg.T, cfg.k) and a["sigma"].shape == (cfg.T,) and a["sigma"].dtype == np.float32
    for key in ("strain", "basis", "coeffs", "sigma"):
        assert np.array_equal(a[key], b[key])
    assert cfg.j_low == 120 and cfg.bins == 2049
    assert len(a["injections"]) == 1 and a["injections"][0]["snr"] == 12.0


def test_config_table_matches_baseline_json():
    c = wlm.CONFIGS
    assert (c["small"].N, c["small"].k, c["small"].T, c["small"].f_low) == (131072, 128, 2000, 25.0)
    assert (c["paper"].N, c["paper"].k, c["paper"].T, c["paper"].n_inj) == (524288, 256, 20000, 50)
    assert (c["large"].N, c["large"].k, c["large"].T, c["large"].fs) == (262144, 256, 100000, 4096.0)
    assert c["paper"].j_low == 5120 and c["small"].j_low == 1600


def test_extra_segments_share_the_bank():
    wl = wlm.make_workload(wlm.CONFIGS["tiny"])
    s0, inj0 = wlm.make_strain(wl, 0)
    assert s0 is wl["strain"] and inj0 is wl["injections"]
    s1, inj1 = wlm.make_strain(wl, 1)
    s1b, _ = wlm.make_strain(wl, 1)
    assert s1.shape == s0.shape and s1.dtype == np.complex64
    assert np.array_equal(s1, s1b) and not np.array_equal(s1, s0)
    assert len(inj1) == len(inj0)
    # noise normalisation: |d[j]|^2 averages N for unit-variance white noise
    cfg = wl["config"]
    assert abs((np.abs(s1[10:-10]) ** 2).mean() / cfg.N - 1.0) < 0.15


def test_sweep_grid_and_further_segments_and_time_series():
    """BASELINE.json configs[4] as a grid; segments beyond 0 are fresh draws; the coloured time series whitens back to
    the frequency-domain strain; sub-banks carry their own (k, T, w)."""
    import numpy as np
    from paper_2110_13115_b200 import workloads as wlm
    assert len(wlm.SWEEP_NAMES) == 15
    for name in wlm.SWEEP_NAMES:
        c = wlm.CONFIGS[name]
        assert c.N == 1 << 20 and c.n_inj == 0 and c.k in wlm.SWEEP_K and c.T in wlm.SWEEP_T
    assert len({wlm.CONFIGS[n].seed for n in wlm.CONFIGS}) == len(wlm.CONFIGS)      # one seed per config
    wl = wlm.make_workload(wlm.CONFIGS["tiny"])
    cfg = wl["config"]
    s0, inj0 = wlm.make_strain(wl, 0)
    s1, inj1 = wlm.make_strain(wl, 1)
    s1b, _ = wlm.make_strain(wl, 1)
    assert s0 is wl["strain"] and np.array_equal(s1, s1b) and not np.array_equal(s0, s1) and len(inj1) == cfg.n_inj
    x, inv_asd = wlm.make_time_series(wl, 1)
    assert x.dtype == np.float32 and x.shape == (cfg.N,) and inv_asd.shape == (cfg.bins,) and (inv_asd > 0).all()
    back = np.fft.rfft(x.astype(np.float64)) * inv_asd
    assert np.abs(back - s1)[cfg.j_low:cfg.N // 2].max() < 1e-3          # float32 rounding of x only
    subs = wlm.make_subbanks(cfg, [(1.0, 1.2, 16, 20, 4), (1.2, 1.5, 8, 12, 2)])
    assert [w["coeffs"].shape for w in subs] == [(20, 16), (12, 8)] and subs[1]["config"].w == 2
    assert subs[0]["mc"].max() <= 1.2 < subs[1]["mc"].min()
