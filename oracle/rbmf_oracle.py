"""CPU fp64 oracle for the hierarchical reduced-basis matched filter (arXiv:2110.13115).

THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only `tests/`,
`__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` / `--impl reference`
legs may import it.  It shares no code with the CUDA path (numpy only, no import
of `paper_2110_13115_b200`), and takes the very arrays the library receives
(complex64 strain / basis / coefficients, float32 sigma), promoted to fp64 and
treated as exact.

It follows the paper step by step, in the paper's order, with no blocking,
fusion or reordering.  The method is not an exact-result accelerator (basis
truncation and the binned first stage change which samples become triggers,
PAPER.md:184-193), so "correct" = this algorithm, not the flat template search.

Notation (the discrete normalisation is reading R2 in
DESIGN.md because PAPER.md Eq. 4 is continuous):
  N samples, bins j = 0..N/2, band B = [j_low, N/2)
  d[j]   = unnormalised forward DFT of the whitened unit-variance series  (s~/sqrt(S_n))
  b_k[j] = orthonormal reduced basis (p~_k), c_tk = decomposition coefficients
  h'_t   = sum_k c_tk b_k
  rho_t[n] = (s/sigma_t) sum_{j in B} d[j] conj(h'_t[j]) exp(+2 pi i j n/N),  s = sqrt(2/N)   (Eq. 4)
  beta_k[n] = s sum_{j in B} d[j] conj(b_k[j]) exp(+2 pi i j n/N)
  rho_t[n] = (1/sigma_t) sum_k conj(c_tk) beta_k[n]                                             (Eq. 7)
  avg:  rho_bar_t[i] = (1/w) sum_{r<w} rho_t[i w + r]                                           (Eq. 9)
  candidates C = {(t,i): |rho_bar_t[i]| >= thr1};  triggers = {(t,n): (t, n//w) in C, |rho_t[n]| >= thr2}

Pins (tests/test_oracle_pins.py, all `-m "not gpu"`):
  normalisation / FFT sign     brute-force time-domain circular correlation at small N; noise-free
                               injection of optimal SNR A peaks at exactly A e^{i phi} at n0
  direct-DFT vs FFT route      `snr_series_direct` (literal sum) vs `snr_series_fft` (numpy ifft)
  reduced-basis identity       Eq. 7 == Eq. 4 with the full basis
  truncation identity          Eq. 8
  averaging                    Eq. 12 alias-fold route (`averaged_series_eq12`) == binned mean; w=1 => flat
  thresholds / sets            independent pure-Python enumeration on tiny inputs
  cost model                   Eq. 13-14 reproduce the paper's quoted ~6x / ~10x (tests/golden/paper_values.txt)
  template routes              flat method: pure-Python enumeration of `snr_series_direct` on the BANK templates, and its
                               count == oracle_filter's n_flat on reconstructed templates; fast first stage: candidates ==
                               oracle_filter's (Eq. 12 route == binned mean, already pinned) incl. the values
  preparation (PCA)            against numpy's SVD (same subspace projector, same singular values), orthonormality, Eq. 8
                               with its own singular values, and optimality: no other orthonormal k-set captures more
  tuning, Eq. 16               hand-built lists with the answer worked out by counting; w = 1 recovers everything
  forward transform, whitening literal O(N^2) sum at small N, a cosine's closed form (N/2 at its bin), Parseval; batches:
                               segment b of `oracle_filter_batch` against the time-domain brute force on strain b alone
Parity status: every function on the path is pinned by at least one of these.
PARITY UNPINNED: `z_total` (Eq. 15).  The paper prints no value of Eq. 15 that its own formula
reproduces (the quoted speed-ups ~6 / ~10 of PAPER.md:316 are matched by Eq. 14 alone, which is what pins `z_first`;
with the p / T term of Eq. 15 they are not reached), so the only check of `z_total` is that it is the sum of its terms,
which restates the formula.  It is a three-line calculator off the hot path; no kernel is compared with it.
"""
from __future__ import annotations

import math

import numpy as np


# --------------------------------------------------------------------------- band
def band(N: int, fs: float, f_low: float):
    """Band B = [j_low, N/2): DC..j_low-1 and the Nyquist bin are ignored."""
    j_low = int(math.ceil(f_low * N / fs - 1e-12))
    return j_low, N // 2


# ------------------------------------------------------------------ reconstruction
def reconstructed_templates(coeffs, basis, idx=None):
    """h'_t[j] = sum_k c_tk b_k[j].  Returns (len(idx), bins) complex128."""
    C = np.asarray(coeffs, dtype=np.complex128)
    if idx is not None:
        C = C[np.atleast_1d(idx)]
    return C @ np.asarray(basis, dtype=np.complex128)


# ------------------------------------------------------------- SNR series, Eq. 4
def snr_series_direct(d, h, sigma, N, j_low, n_chunk=256):
    """rho[n] = (s/sigma) sum_{j in B} d[j] conj(h[j]) e^{+2 pi i j n / N}, evaluated literally
    (direct O(N |B|) DFT; Eq. 4, discretised).  One template.  For small N."""
    d = np.asarray(d, dtype=np.complex128)
    h = np.asarray(h, dtype=np.complex128)
    j = np.arange(j_low, N // 2, dtype=np.int64)
    g = d[j] * np.conj(h[j])
    s = math.sqrt(2.0 / N)
    out = np.empty(N, dtype=np.complex128)
    for a in range(0, N, n_chunk):
        n = np.arange(a, min(N, a + n_chunk), dtype=np.int64)
        ph = ((j[None, :] * n[:, None]) % N).astype(np.float64) * (2.0 * math.pi / N)  # exact index reduction
        out[a:a + len(n)] = (np.exp(1j * ph) * g[None, :]).sum(axis=1)
    return out * (s / float(sigma))


def snr_point(d, h, sigma, N, j_low, n):
    """rho[n] at one sample n by the literal O(|B|) sum of Eq. 4."""
    d = np.asarray(d, dtype=np.complex128)
    h = np.asarray(h, dtype=np.complex128)
    j = np.arange(j_low, N // 2, dtype=np.int64)
    ph = ((j * int(n)) % N).astype(np.float64) * (2.0 * math.pi / N)
    return complex((d[j] * np.conj(h[j]) * np.exp(1j * ph)).sum() * (math.sqrt(2.0 / N) / float(sigma)))


def snr_series_fft(d, h, sigma, N, j_low):
    """Same series as `snr_series_direct`, the inverse DFT taken by numpy's FFT
    ("The SNR as a function of time can be obtained efficiently by performing an inverse FFT").
    `h` may be (bins,) or (M, bins); `sigma` scalar or (M,).  Returns (N,) or (M, N) complex128."""
    d = np.asarray(d, dtype=np.complex128)
    h = np.asarray(h, dtype=np.complex128)
    one = h.ndim == 1
    h2 = np.atleast_2d(h)
    g = np.zeros((h2.shape[0], N), dtype=np.complex128)
    g[:, j_low:N // 2] = d[None, j_low:N // 2] * np.conj(h2[:, j_low:N // 2])
    rho = np.fft.ifft(g, axis=1) * N                      # unnormalised inverse DFT, e^{+2 pi i j n/N}
    rho *= (math.sqrt(2.0 / N) / np.atleast_1d(np.asarray(sigma, dtype=np.float64)))[:, None]
    return rho[0] if one else rho


# ------------------------------------------------- reduced-basis route, Eq. 6 and 7
def basis_series(d, basis, N, j_low):
    """beta_k[n] = s sum_{j in B} d[j] conj(b_k[j]) e^{+2 pi i j n/N}.  (k, N) complex128."""
    k = np.asarray(basis).shape[0]
    return snr_series_fft(d, basis, np.ones(k), N, j_low)


def snr_series_rb(beta, coeffs_t, sigma_t):
    """rho_r[n] = (1/sigma_t) sum_k conj(c_tk) beta_k[n]  (Eq. 7)."""
    c = np.asarray(coeffs_t, dtype=np.complex128)
    return (np.conj(c)[None, :] @ np.asarray(beta, dtype=np.complex128))[0] / float(sigma_t)


def truncation_loss(singular_values, p):
    """<delta rho / rho> = 1 - sum_{k<p} sigma_k^2 / sum_k sigma_k^2  (Eq. 8)."""
    s2 = np.asarray(singular_values, dtype=np.float64) ** 2
    return 1.0 - s2[:p].sum() / s2.sum()


# ------------------------------------------------------------------ averaging, Eq. 9
def bin_average(series, w):
    """x_avg[i] = (1/w) sum_{j<w} x[i w + j]  (Eq. 9): mean of the COMPLEX series over
    non-overlapping bins aligned at sample 0.  Works on the last axis."""
    x = np.asarray(series)
    n = x.shape[-1]
    if n % w:
        raise ValueError("w must divide N")
    return x.reshape(x.shape[:-1] + (n // w, w)).sum(axis=-1) / w


def averaged_series_eq12(d, h, sigma, N, j_low, w):
    """Averaged SNR series by the paper's fast first stage (Eq. 10-12):
    Omega(f') = sum_{l<w} G[l N/w + f'] S(l N/w + f'),  S(f) = (1/w) sum_{r<w} e^{2 pi i f r/N},
    rho_bar[b] = sum_{f'<N/w} e^{2 pi i f' b/(N/w)} Omega(f')  -- an inverse DFT of length N/w.
    (Eq. 12 as printed is garbled; this is Eq. 10 with Eq. 11 substituted, reading R14 in DESIGN.md.)"""
    d = np.asarray(d, dtype=np.complex128)
    h = np.asarray(h, dtype=np.complex128)
    G = np.zeros(N, dtype=np.complex128)
    G[j_low:N // 2] = d[j_low:N // 2] * np.conj(h[j_low:N // 2])
    G *= math.sqrt(2.0 / N) / float(sigma)
    f = np.arange(N, dtype=np.int64)
    S = np.zeros(N, dtype=np.complex128)
    for r in range(w):
        S += np.exp(2j * math.pi * ((f * r) % N) / N)
    S /= w
    M = N // w
    Omega = (G * S).reshape(w, M).sum(axis=0)             # f = l*M + f'
    return np.fft.ifft(Omega) * M


# --------------------------------------------------------------- thresholds and sets
def candidates_from_avg(rho_bar, thr1):
    """First-stage triggers: bins whose averaged SNR modulus is >= thr1."""
    return np.nonzero(np.abs(rho_bar) >= thr1)[0]


def hierarchical_triggers_one(rho, w, thr1, thr2):
    """Both stages for one template's full series `rho` (N,): returns (cand_bins, trig_n, flat_n, rho_bar).
    Stage 2 = every sample inside the triggering bins, thresholded at thr2."""
    rho_bar = bin_average(rho, w)
    cand = candidates_from_avg(rho_bar, thr1)
    mod = np.abs(rho)
    flat = np.nonzero(mod >= thr2)[0]
    in_cand = np.zeros(len(rho_bar), dtype=bool)
    in_cand[cand] = True
    trig = flat[in_cand[flat // w]]
    return cand, trig, flat, rho_bar


def oracle_filter(strain, basis, coeffs, sigma, N, fs, f_low, w, thr1, thr2, templates=None, chunk=64,
                  keep_margins=True):
    """The whole hot path for the listed templates (default all), template route:
    h'_t -> rho_t (Eq. 4 by FFT) -> rho_bar_t (Eq. 9) -> thr1 -> thr2.

    Returns dict with
      triggers   structured array (template, time, re, im, avg_abs) sorted by (template, time)
                 avg_abs = |rho_bar| of the bin the trigger lies in (for the tie-band rule)
      candidates structured array (template, bin, re, im) sorted
      n_flat     number of flat triggers |rho| >= thr2 over the same templates
      near       structured array of every (template, time, re, im, avg_abs) with
                 |rho| >= thr2 (1 - 2e-3) and |rho_bar| >= thr1 (1 - 2e-3): superset used for the allowed set
      cand_near  structured array (template, bin, re, im) of every bin with |rho_bar| >= thr1 (1 - 2e-3):
                 superset of `candidates` used for the allowed set of the first stage (keep_margins only)
    """
    j_low, _ = band(N, fs, f_low)
    T = np.asarray(coeffs).shape[0]
    tids = np.arange(T) if templates is None else np.atleast_1d(np.asarray(templates))
    trig_dt = np.dtype([("template", np.int64), ("time", np.int64), ("re", np.float64), ("im", np.float64),
                        ("avg_abs", np.float64)])
    cand_dt = np.dtype([("template", np.int64), ("bin", np.int64), ("re", np.float64), ("im", np.float64)])
    trig_parts, cand_parts, near_parts, cnear_parts = [], [], [], []
    n_flat = 0
    slack = 1.0 - 2e-3
    for a in range(0, len(tids), chunk):
        ids = tids[a:a + chunk]
        h = reconstructed_templates(coeffs, basis, ids)
        rho = snr_series_fft(strain, h, np.asarray(sigma, dtype=np.float64)[ids], N, j_low)
        for m, t in enumerate(ids):
            cand, trig, flat, rho_bar = hierarchical_triggers_one(rho[m], w, thr1, thr2)
            n_flat += len(flat)
            if len(cand):
                c = np.empty(len(cand), dtype=cand_dt)
                c["template"], c["bin"] = t, cand
                c["re"], c["im"] = rho_bar[cand].real, rho_bar[cand].imag
                cand_parts.append(c)
            if len(trig):
                r = np.empty(len(trig), dtype=trig_dt)
                r["template"], r["time"] = t, trig
                r["re"], r["im"] = rho[m][trig].real, rho[m][trig].imag
                r["avg_abs"] = np.abs(rho_bar[trig // w])
                trig_parts.append(r)
            if keep_margins:
                cn = np.nonzero(np.abs(rho_bar) >= thr1 * slack)[0]
                if len(cn):
                    c = np.empty(len(cn), dtype=cand_dt)
                    c["template"], c["bin"] = t, cn
                    c["re"], c["im"] = rho_bar[cn].real, rho_bar[cn].imag
                    cnear_parts.append(c)
                mod = np.abs(rho[m])
                nn = np.nonzero(mod >= thr2 * slack)[0]
                nn = nn[np.abs(rho_bar[nn // w]) >= thr1 * slack]
                if len(nn):
                    r = np.empty(len(nn), dtype=trig_dt)
                    r["template"], r["time"] = t, nn
                    r["re"], r["im"] = rho[m][nn].real, rho[m][nn].imag
                    r["avg_abs"] = np.abs(rho_bar[nn // w])
                    near_parts.append(r)
    cat = lambda parts, dt: np.concatenate(parts) if parts else np.empty(0, dtype=dt)
    return {"triggers": cat(trig_parts, trig_dt), "candidates": cat(cand_parts, cand_dt),
            "near": cat(near_parts, trig_dt), "cand_near": cat(cnear_parts, cand_dt), "n_flat": n_flat}


# ------------------------------------------------- the step before the path, and batches of segments
def strain_from_time_series(x, inv_asd=None):
    """Step 1 of the paper's scheme (PAPER.md:175 "FFT of the data", :177 "divided by sqrt(S_n)"):
    d[j] = inv_asd[j] * sum_n x[n] e^{-2 pi i j n / N}, j = 0..N/2 -- the unnormalised forward DFT of the real series
    (SURVEY.md App. A), times the caller's whitening array 1/sqrt(S_n(f_j)) (omitted = already white).
    x: (N,) or (B, N) real.  Returns complex128 (N/2+1,) or (B, N/2+1)."""
    x = np.asarray(x, dtype=np.float64)
    d = np.fft.rfft(x, axis=-1)
    if inv_asd is not None:
        d = d * np.asarray(inv_asd, dtype=np.float64)
    return d


def oracle_filter_batch(strains, basis, coeffs, sigma, N, fs, f_low, w, thr1, thr2, templates=None, chunk=64):
    """A batch of segments filtered against the same resident basis and coefficients ("filtering each
    segment in parallel"): segment b is the whole hot path on strains[b], independent of the others; its records are
    reported with time = b N + n and bin = b N/w + i.  Same fields as `oracle_filter`."""
    strains = np.asarray(strains)
    out = None
    for b in range(strains.shape[0]):
        r = oracle_filter(strains[b], basis, coeffs, sigma, N, fs, f_low, w, thr1, thr2, templates=templates,
                          chunk=chunk)
        for key in ("triggers", "near"):
            r[key]["time"] += b * N
        for key in ("candidates", "cand_near"):
            r[key]["bin"] += b * (N // w)
        if out is None:
            out = r
        else:
            for key in ("triggers", "near", "candidates", "cand_near"):
                out[key] = np.concatenate([out[key], r[key]])
            out["n_flat"] += r["n_flat"]
    return out


def oracle_filter_banks(strain, banks, N, fs, f_low, thr1, thr2):
    """Many sub-banks against one strain (Table I): `banks` is a list of dicts with keys basis, coeffs,
    sigma, w -- each sub-bank has its own basis size and window.  Every sub-bank is the whole hot path on its own;
    triggers of sub-bank m are reported with template = (templates of the sub-banks before it) + t.
    Returns {'triggers', 'near', 'n_flat', 'per_bank': [oracle_filter results with local ids]}."""
    out = {"triggers": [], "near": [], "n_flat": 0, "per_bank": []}
    base = 0
    for bk in banks:
        r = oracle_filter(strain, bk["basis"], bk["coeffs"], bk["sigma"], N, fs, f_low, bk["w"], thr1, thr2)
        out["per_bank"].append(r)
        for key in ("triggers", "near"):
            c = r[key].copy()
            c["template"] += base
            out[key].append(c)
        out["n_flat"] += r["n_flat"]
        base += np.asarray(bk["coeffs"]).shape[0]
    out["triggers"] = np.concatenate(out["triggers"])
    out["near"] = np.concatenate(out["near"])
    return out


# ------------------------------------------------- the paper's template routes
def template_method_triggers(strain, templates, sigma, N, fs, f_low, thr, chunk=64):
    """The flat template method (PAPER.md:61-68; cost Eq. 13, :238; the paper's cuFFT baseline, :338): for every
    template h_t the full SNR series of Eq. 4 by one inverse FFT, and a trigger for every sample with |rho| >= thr.
    templates: (T, bins) filters h_t; sigma: (T,) or None (=> 1).  Returns a dict shaped like `oracle_filter`'s:
    'triggers' and 'near' (|rho| >= thr (1 - 2e-3)) with avg_abs = +inf (there is no first stage), 'n_flat'."""
    j_low, _ = band(N, fs, f_low)
    templates = np.asarray(templates)
    T = templates.shape[0]
    sg = np.ones(T) if sigma is None else np.asarray(sigma, dtype=np.float64)
    dt = np.dtype([("template", np.int64), ("time", np.int64), ("re", np.float64), ("im", np.float64),
                   ("avg_abs", np.float64)])
    parts, near = [], []
    for a in range(0, T, chunk):
        rho = snr_series_fft(strain, templates[a:a + chunk], sg[a:a + chunk], N, j_low)
        mod = np.abs(rho)
        for lst, level in ((parts, thr), (near, thr * (1.0 - 2e-3))):
            m, n = np.nonzero(mod >= level)
            r = np.empty(len(m), dtype=dt)
            r["template"], r["time"] = a + m, n
            r["re"], r["im"], r["avg_abs"] = rho[m, n].real, rho[m, n].imag, np.inf
            lst.append(r)
    trig = np.concatenate(parts) if parts else np.empty(0, dtype=dt)
    return {"triggers": trig, "near": np.concatenate(near) if near else np.empty(0, dtype=dt), "n_flat": len(trig)}


def first_stage_by_templates(strain, templates, sigma, N, fs, f_low, w, thr1):
    """The paper's fast first stage by templates: rho_bar_t from the alias-folded spectrum and an
    inverse FFT of length N/w (`averaged_series_eq12`), thresholded at thr1.  Returns 'candidates' and 'cand_near'
    (|rho_bar| >= thr1 (1 - 2e-3)) as in `oracle_filter`."""
    j_low, _ = band(N, fs, f_low)
    templates = np.asarray(templates)
    T = templates.shape[0]
    sg = np.ones(T) if sigma is None else np.asarray(sigma, dtype=np.float64)
    dt = np.dtype([("template", np.int64), ("bin", np.int64), ("re", np.float64), ("im", np.float64)])
    cand, near = [], []
    for t in range(T):
        rb = averaged_series_eq12(strain, templates[t], sg[t], N, j_low, w)
        for lst, level in ((cand, thr1), (near, thr1 * (1.0 - 2e-3))):
            i = np.nonzero(np.abs(rb) >= level)[0]
            c = np.empty(len(i), dtype=dt)
            c["template"], c["bin"], c["re"], c["im"] = t, i, rb[i].real, rb[i].imag
            lst.append(c)
    return {"candidates": np.concatenate(cand), "cand_near": np.concatenate(near)}


def evaluate_points(strain, basis, coeffs, sigma, N, fs, f_low, w, template, times):
    """Pointwise re-evaluation for one template: returns (rho[n] for n in times, rho_bar of each n's bin),
    every value by the literal O(|B|) sum of Eq. 4 (no FFT)."""
    j_low, _ = band(N, fs, f_low)
    h = reconstructed_templates(coeffs, basis, [template])[0]
    sg = float(np.asarray(sigma, dtype=np.float64)[template])
    rho, rbar = [], []
    for n in np.atleast_1d(times):
        n = int(n)
        rho.append(snr_point(strain, h, sg, N, j_low, n))
        b = n // w
        rbar.append(sum(snr_point(strain, h, sg, N, j_low, b * w + r) for r in range(w)) / w)
    return np.array(rho), np.array(rbar)


# ------------------------------------------------------- preparation: PCA of a (sub-)bank
def pca_basis(templates, k):
    """The preparation step as the paper describes it (readings R5-R7): templates
    stored row-wise in T (S x bins, unit norm, no centering), covariance C = T T^H (S x S), EVD, basis vectors
    p_i = lambda_i^{-1/2} v_i^H T for the k largest eigenvalues, decomposition coefficients D = T P^H.
    Returns (basis (k, bins) complex128 orthonormal rows, coeffs (S, k), singular values sqrt(lambda) descending (S,))."""
    Tm = np.asarray(templates, dtype=np.complex128)
    C = Tm @ Tm.conj().T
    lam, V = np.linalg.eigh(C)
    lam, V = lam[::-1], V[:, ::-1]
    lam = np.clip(lam, 0.0, None)
    basis = (V[:, :k].conj().T @ Tm) / np.sqrt(lam[:k])[:, None]
    coeffs = Tm @ basis.conj().T
    return basis, coeffs, np.sqrt(lam)


def captured_power(templates, basis):
    """mean_t ||c_t||^2 with c = T P^H: the fraction of the bank's power an orthonormal basis captures (the complement
    of the mean SNR loss of Eq. 8)."""
    c = np.asarray(templates, dtype=np.complex128) @ np.asarray(basis, dtype=np.complex128).conj().T
    return float((np.abs(c) ** 2).sum(axis=1).mean())


# ------------------------------------------------------- tuning of (w, rho_I), Eq. 16
def rho_target(final_mods, flat_mods, grid, ratio=0.99):
    """Eq. 16: rho_target(w, rho_I) = min{rho_II : n_final(rho_II) >= ratio * n_flat(rho_II)}, with
    n_final / n_flat the numbers of hierarchical / flat triggers whose SNR modulus is >= rho_II, searched over the
    ascending thresholds `grid`.  The hierarchical set is a subset of the flat one and the recovered fraction grows
    with rho_II in noise, so "min" is read as the first grid value from which the condition holds for ALL larger grid
    values with flat triggers (a single lucky threshold below a failing one does not count).  Returns (rho_target or
    None if never reached, n_final[grid], n_flat[grid])."""
    fm = np.sort(np.asarray(final_mods, dtype=np.float64))
    fl = np.sort(np.asarray(flat_mods, dtype=np.float64))
    grid = np.asarray(grid, dtype=np.float64)
    n_final = len(fm) - np.searchsorted(fm, grid, side="left")
    n_flat = len(fl) - np.searchsorted(fl, grid, side="left")
    ok = n_final >= ratio * n_flat
    target = None
    for i in range(len(grid) - 1, -1, -1):
        if not ok[i]:
            break
        if n_flat[i] > 0:
            target = float(grid[i])
    return target, n_final, n_flat


# ------------------------------------------------------- cost model, Eq. 13-15
def z_basic(N, T):
    """Template-method flops, Eq. 13; log base 2 (reading R19)."""
    return N * T * (5.0 * math.log2(N) + 6.0)


def z_first(N, T, w):
    """First-stage flops by the template route, Eq. 14."""
    return N * T * (5.0 / w * math.log2(N / w) + 6.0 + 2.0 / w)


def z_total(N, T, w, p, f_triggers):
    """Eq. 15: z_first + 4 p w f T + N p (5 log N + 6)."""
    return z_first(N, T, w) + 4.0 * p * w * f_triggers * T + N * p * (5.0 * math.log2(N) + 6.0)


def throughput(N_seconds, T, t_seconds):
    """Templates processed in real time = N T / t."""
    return N_seconds * T / t_seconds
