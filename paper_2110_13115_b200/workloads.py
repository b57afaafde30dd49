"""Seeded synthetic workloads for the reduced-basis hierarchical matched filter.

This module only *produces inputs* (strain, basis, coefficients, sigma, injection
list).  It holds none of the method's arithmetic (no correlation, FFT of the
product, averaging, reconstruction or thresholding) and is the one module that
both the CPU oracle's tests and the CUDA path's tests/bench draw inputs from.

The inputs stand in for the paper's PyCBC aLIGO-PSD noise, the O2 template bank
and IMRPhenomPv2 templates, none of which exist here.
Shapes, sizes and recipe follow BASELINE.json `configs` and SURVEY.md §8(d):

* templates: Newtonian SPA chirps  h(f) = f^(-7/6) exp(-i (3/128) (pi Mc f)^(-5/3)),
  zero outside the band [j_low, N/2), unit-normalised ("normalized to unity",
  PAPER.md:152);
* basis: top-k right singular vectors of the (T x bins) template matrix
  (Eq. 5b), computed through the T x T Gram matrix, re-orthonormalised
  by QR in fp64; for T > `basis_subset` a seeded random subset of templates is used
  (any orthonormal k-set is a valid input to the hot path);
* coefficients: c_tk = sum_j conj(b_k[j]) u_t[j], from the
  complex64-rounded basis so that sum_k c_tk b_k is the projection onto the
  basis actually handed to the filter;
* sigma_t = ||c_t||_2 (norm of the filter actually applied), float32;
* strain: rfft of N(0,1) white noise plus injections of optimal SNR A,
  d[j] += A sqrt(N/2) u_t[j] exp(-2 pi i j n0/N) exp(i phi).

RNG draws always come from numpy's default_rng on the host in the order
Mc[T] -> noise x[N] -> per injection (A, template, n0, phi) -> basis subset;
the heavy linear algebra runs in torch complex128 on `device` (CPU or CUDA).
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional

import numpy as np
import torch

MSUN_SECONDS = 4.925490947e-6  # G Msun / c^3
BASE_SEED = 20211013


@dataclasses.dataclass(frozen=True)
class WorkloadConfig:
    name: str
    index: int          # seed = BASE_SEED + index
    N: int              # samples per segment
    fs: float           # sampling rate, Hz
    f_low: float        # lower cutoff, Hz
    k: int              # reduced-basis size
    T: int              # templates
    w: int              # stage-1 averaging window (Eq. 9)
    mc_lo: float        # chirp-mass range, Msun
    mc_hi: float
    n_inj: int
    snr_lo: float
    snr_hi: float
    thr1: float = 5.0
    thr2: float = 6.0
    basis_subset: int = 4096

    @property
    def bins(self) -> int:
        return self.N // 2 + 1

    @property
    def j_low(self) -> int:
        return band_start(self.N, self.fs, self.f_low)

    @property
    def seed(self) -> int:
        return BASE_SEED + self.index

    def replace(self, **kw) -> "WorkloadConfig":
        return dataclasses.replace(self, **kw)


def band_start(N: int, fs: float, f_low: float) -> int:
    """First bin of the band [j_low, N/2): j_low = ceil(f_low N / fs)."""
    return int(math.ceil(f_low * N / fs - 1e-12))


# BASELINE.json configs (1-4) + the narrow-Mc variants SURVEY.md §8(d) adds + one
# sweep point; "mini" is a CPU-test-sized case spanning several tiles and a ragged T.
CONFIGS = {
    "tiny": WorkloadConfig("tiny", 1, 4096, 1024.0, 30.0, 16, 64, 4, 1.0, 1.5, 1, 12.0, 12.0),
    "tiny_narrow": WorkloadConfig("tiny_narrow", 11, 4096, 1024.0, 30.0, 16, 64, 4, 1.0, 1.005, 1, 12.0, 12.0),
    "mini": WorkloadConfig("mini", 21, 16384, 1024.0, 30.0, 32, 300, 8, 1.0, 1.2, 3, 8.0, 14.0),
    "small": WorkloadConfig("small", 2, 131072, 2048.0, 25.0, 128, 2000, 8, 1.0, 3.0, 10, 6.0, 15.0),
    "small_narrow": WorkloadConfig("small_narrow", 12, 131072, 2048.0, 25.0, 128, 2000, 8, 1.20, 1.25, 10, 6.0, 15.0),
    "paper": WorkloadConfig("paper", 3, 524288, 2048.0, 20.0, 256, 20000, 8, 1.0, 3.0, 50, 5.0, 20.0),
    "large": WorkloadConfig("large", 4, 262144, 4096.0, 20.0, 256, 100000, 8, 0.5, 5.0, 100, 5.0, 20.0),
}

# BASELINE.json configs[4], the sweep grid: N = 2^20 (256 s at 4096 Hz), f_low not given -> 20 Hz, pure noise,
# k in {32, 64, 128, 256, 512} x T in {1000, 10000, 100000}, Mc ~ U[1, 3]; w = 8 here, w = 1 (and 2, 4, 16) through
# `cfg.replace(w=...)` / `bench.py --w`.  One seed per grid point (index 5 is the k = 256, T = 10000 point of round 1).
SWEEP_K = (32, 64, 128, 256, 512)
SWEEP_T = (1000, 10000, 100000)
for _ik, _k in enumerate(SWEEP_K):
    for _it, _T in enumerate(SWEEP_T):
        _name = "sweep_k%d_T%d" % (_k, _T)
        _index = 5 if (_k, _T) == (256, 10000) else 500 + 10 * _ik + _it
        CONFIGS[_name] = WorkloadConfig(_name, _index, 1 << 20, 4096.0, 20.0, _k, _T, 8, 1.0, 3.0, 0, 0.0, 0.0)
SWEEP_NAMES = tuple("sweep_k%d_T%d" % (_k, _T) for _k in SWEEP_K for _T in SWEEP_T)


def _spa_templates(mc_msun: np.ndarray, cfg: WorkloadConfig, device) -> torch.Tensor:
    """Unit-norm SPA chirps on the band, shape (len(mc), bins) complex128 on `device`."""
    j = torch.arange(cfg.bins, dtype=torch.float64, device=device)
    f = j * (cfg.fs / cfg.N)
    inband = (j >= cfg.j_low) & (j < cfg.N // 2)
    f_safe = torch.where(inband, f, torch.ones_like(f))
    mc = torch.as_tensor(mc_msun, dtype=torch.float64, device=device) * MSUN_SECONDS
    amp = torch.where(inband, f_safe ** (-7.0 / 6.0), torch.zeros_like(f))
    phase = -(3.0 / 128.0) * (math.pi * mc[:, None] * f_safe[None, :]) ** (-5.0 / 3.0)
    h = torch.polar(amp[None, :].expand(len(mc_msun), -1).contiguous(), phase)
    h = h * inband[None, :]
    h = h / torch.linalg.vector_norm(h, dim=1, keepdim=True)
    return h


def _chunks(n: int, size: int):
    for a in range(0, n, size):
        yield a, min(n, a + size)


def make_workload(cfg: WorkloadConfig, device: Optional[str] = None, chunk: Optional[int] = None) -> dict:
    """Generate the seeded inputs of one configuration.

    Returns numpy arrays (what the library and the oracle both receive):
      strain  (bins,)   complex64   raw rfft of the unit-variance whitened series
      basis   (k, bins) complex64   orthonormal over the band
      coeffs  (T, k)    complex64   c_tk, unconjugated
      sigma   (T,)      float32     ||c_t||_2
    plus `mc` (T,), `injections` (list of dicts) and `captured` (fraction of bank
    power the basis captures, mean_t ||c_t||^2).
    """
    dev = torch.device(device or "cpu")
    rng = np.random.default_rng(cfg.seed)
    N, bins, T, k = cfg.N, cfg.bins, cfg.T, cfg.k
    if chunk is None:
        chunk = max(16, int(2.0e9 // (bins * 16)))  # ~2 GB of complex128 templates at a time

    # ---- draws, in the documented order -----------------------------------
    mc = rng.uniform(cfg.mc_lo, cfg.mc_hi, size=T)
    x = rng.standard_normal(N)
    injections = []
    for _ in range(cfg.n_inj):
        A = float(rng.uniform(cfg.snr_lo, cfg.snr_hi)) if cfg.snr_hi > cfg.snr_lo else float(cfg.snr_lo)
        t = int(rng.integers(0, T))
        n0 = int(rng.integers(0, N))
        phi = float(rng.uniform(0.0, 2.0 * math.pi))
        injections.append({"snr": A, "template": t, "n0": n0, "phase": phi})
    if T > cfg.basis_subset:
        subset = np.sort(rng.choice(T, size=cfg.basis_subset, replace=False))
    else:
        subset = np.arange(T)

    # ---- strain -------------------------------------------------------------
    d = np.fft.rfft(x)  # unnormalised forward DFT, bins = N/2+1
    if injections:
        jj = np.arange(bins, dtype=np.float64)
        for inj in injections:
            u = _spa_templates(mc[inj["template"]:inj["template"] + 1], cfg, "cpu")[0].numpy()
            ph = np.exp(-2j * np.pi * ((jj * inj["n0"]) % N) / N) * np.exp(1j * inj["phase"])
            d = d + inj["snr"] * math.sqrt(N / 2.0) * u * ph
    strain = d.astype(np.complex64)

    # ---- basis: top-k right singular vectors via the Gram matrix (Eq. 5a/5b) ----
    S = len(subset)
    G = torch.zeros((S, S), dtype=torch.complex128, device=dev)
    bchunk = max(256, int(1.0e9 // (S * 16)))           # column (bin) chunk
    for a, b in _chunks(bins, bchunk):
        # regenerate template columns a:b for the subset (cheap) to bound memory
        Hs = _spa_templates_cols(mc[subset], cfg, dev, a, b)
        G += Hs @ Hs.conj().T
    evals, V = torch.linalg.eigh(G)                       # ascending
    evals = evals.flip(0)[:k].clamp_min(1e-300)
    V = V.flip(1)[:, :k]                                  # (S, k)
    # B = Lambda^{-1/2} V^H H, built by column chunks, then QR re-orthonormalised
    Bt = torch.empty((bins, k), dtype=torch.complex128, device=dev)
    scale = (1.0 / torch.sqrt(evals)).to(torch.complex128)
    for a, b in _chunks(bins, bchunk):
        Hs = _spa_templates_cols(mc[subset], cfg, dev, a, b)     # (S, cols)
        Bt[a:b] = (Hs.T @ V.conj()) * scale[None, :]
    Q, R = torch.linalg.qr(Bt)                            # Q: (bins, k) orthonormal columns
    # fix the phase convention so that the result does not depend on LAPACK's sign choice
    diag = torch.diagonal(R)
    Q = Q * (diag / diag.abs())[None, :]                  # unique QR: R gets a real positive diagonal
    jrow = torch.arange(bins, device=dev)
    Q = Q * ((jrow >= cfg.j_low) & (jrow < N // 2))[:, None]   # exact zeros outside the band (QR leaves ~1e-17)
    basis = Q.T.contiguous().to(torch.complex64)          # (k, bins)
    del G, V, Bt, Q, R

    # ---- coefficients from the complex64-rounded basis ------------------------
    Bc = basis.to(torch.complex128)
    coeffs = torch.empty((T, k), dtype=torch.complex128, device=dev)
    for a, b in _chunks(T, chunk):
        U = _spa_templates(mc[a:b], cfg, dev)              # (chunk, bins)
        coeffs[a:b] = U @ Bc.conj().T
    sigma = torch.linalg.vector_norm(coeffs, dim=1)
    captured = float((sigma ** 2).mean().item())

    return {
        "config": cfg,
        "strain": strain,
        "basis": basis.cpu().numpy(),
        "coeffs": coeffs.to(torch.complex64).cpu().numpy(),
        "sigma": sigma.to(torch.float32).cpu().numpy(),
        "mc": mc,
        "injections": injections,
        "captured": captured,
    }


def _spa_templates_cols(mc_msun: np.ndarray, cfg: WorkloadConfig, device, a: int, b: int) -> torch.Tensor:
    """Columns a:b of the unit-norm template matrix, (len(mc), b-a) complex128.

    The norm over the full band is evaluated in closed loop over all bins once per
    call chunk (cheap: amplitude only depends on f, not on Mc).
    """
    j_all = torch.arange(cfg.bins, dtype=torch.float64, device=device)
    inband_all = (j_all >= cfg.j_low) & (j_all < cfg.N // 2)
    f_all = torch.where(inband_all, j_all * (cfg.fs / cfg.N), torch.ones_like(j_all))
    amp_all = torch.where(inband_all, f_all ** (-7.0 / 6.0), torch.zeros_like(f_all))
    norm = torch.sqrt((amp_all ** 2).sum())               # same for every Mc
    amp = amp_all[a:b] / norm
    f = f_all[a:b]
    mc = torch.as_tensor(mc_msun, dtype=torch.float64, device=device) * MSUN_SECONDS
    phase = -(3.0 / 128.0) * (math.pi * mc[:, None] * f[None, :]) ** (-5.0 / 3.0)
    return torch.polar(amp[None, :].expand(len(mc_msun), -1).contiguous(), phase)


def make_strain(wl: dict, segment: int) -> tuple:
    """Another strain segment for the same bank: segment 0 is `wl['strain']` itself; segment s > 0 draws fresh
    noise and fresh injections (same count and SNR range) from default_rng(seed * 1000 + s).
    Returns (strain complex64 (bins,), injections)."""
    cfg = wl["config"]
    if segment == 0:
        return wl["strain"], wl["injections"]
    rng = np.random.default_rng(cfg.seed * 1000 + int(segment))
    N, bins = cfg.N, cfg.bins
    d = np.fft.rfft(rng.standard_normal(N))
    injections = []
    jj = np.arange(bins, dtype=np.float64)
    for _ in range(cfg.n_inj):
        A = float(rng.uniform(cfg.snr_lo, cfg.snr_hi)) if cfg.snr_hi > cfg.snr_lo else float(cfg.snr_lo)
        t = int(rng.integers(0, cfg.T))
        n0 = int(rng.integers(0, N))
        phi = float(rng.uniform(0.0, 2.0 * math.pi))
        injections.append({"snr": A, "template": t, "n0": n0, "phase": phi})
        u = _spa_templates(wl["mc"][t:t + 1], cfg, "cpu")[0].numpy()
        d = d + A * math.sqrt(N / 2.0) * u * np.exp(-2j * np.pi * ((jj * n0) % N) / N) * np.exp(1j * phi)
    return d.astype(np.complex64), injections


def bank_templates(wl: dict, idx, device: Optional[str] = None) -> np.ndarray:
    """Unit-norm bank templates u_t for the listed template indices, (len, bins) complex128."""
    cfg = wl["config"]
    idx = np.atleast_1d(np.asarray(idx))
    return _spa_templates(wl["mc"][idx], cfg, device or "cpu").cpu().numpy()


def make_time_series(wl: dict, segment: int = 0) -> tuple:
    """Time-domain input for the step in front of the path: a COLOURED real series whose
    whitened spectrum is the strain of `make_strain(wl, segment)`, and the whitening array that undoes the colouring.
    asd(f) = sqrt(1 + (f0/max(f, f_low))^4 + (f/f1)^2) with f0 = 2 f_low, f1 = fs/4 (a smooth seismic-wall + shot-noise
    shape, flat below the band so that float32 keeps the in-band content; a stand-in for the aLIGO PSD);
    x = irfft(strain * asd).  Returns (x float32 (N,), inv_asd float32 (N/2+1,))."""
    cfg = wl["config"]
    d, _ = make_strain(wl, segment)
    f = np.arange(cfg.bins, dtype=np.float64) * (cfg.fs / cfg.N)
    asd = np.sqrt(1.0 + (2.0 * cfg.f_low / np.maximum(f, cfg.f_low)) ** 4 + (f / (cfg.fs / 4.0)) ** 2)
    x = np.fft.irfft(d.astype(np.complex128) * asd, n=cfg.N)
    return x.astype(np.float32), (1.0 / asd).astype(np.float32)


def make_subbanks(cfg: WorkloadConfig, parts, device: Optional[str] = None) -> list:
    """Sub-banks in the manner of the paper (Table I: the bank is cut into chirp-time slices, each with
    its own basis size): `parts` is a list of (mc_lo, mc_hi, k, T, w); sub-bank m is `make_workload` of `cfg` with
    those fields replaced (seed index 1000 * cfg.index + m).  All are meant to be filtered against the strain of
    sub-bank 0 (its noise and its injections)."""
    out = []
    for m, (mc_lo, mc_hi, k, T, w) in enumerate(parts):
        sub = cfg.replace(name="%s_sub%d" % (cfg.name, m), index=1000 * cfg.index + m, mc_lo=mc_lo, mc_hi=mc_hi, k=k,
                          T=T, w=w)
        out.append(make_workload(sub, device=device))
    return out
