"""The error bound behind RBMF_GEMM_SCREEN (gemm_tcgen05.cu header), checked on the CPU.

The screen computes R_16 = sum_k conj(a16_k) b16_k with every complex component of a = c_t / sigma_t and
b = beta^avg[i] rounded once to float16, and lowers thr_stage1 by

    delta = (2u + u^2) ||a|| ||b|| + eta sqrt(k) (||a|| + ||b||)            u = 2^-11, eta = sqrt(2) 2^-25

(+ an accumulation term that is not exercised here: products of two float16 numbers are exact in fp32 and the test
sums in fp64).  If |R_16 - R| could exceed delta, a true candidate could be missed -- so this is the one piece of host
arithmetic on which "identical trigger sets" rests.  numpy's float16 is IEEE binary16 with round-to-nearest-even,
the conversion the kernels use (__float2half_rn / __floats2half2_rn).
"""
import os
import re

import numpy as np
import pytest

U = 2.0 ** -11
ETA = np.sqrt(2.0) * 2.0 ** -25


def bound(a, b):
    na, nb, k = np.linalg.norm(a), np.linalg.norm(b), a.size
    return (2 * U + U * U) * na * nb + ETA * np.sqrt(k) * (na + nb)


def r16(a, b):
    a16 = a.real.astype(np.float16).astype(np.float64) + 1j * a.imag.astype(np.float16).astype(np.float64)
    b16 = b.real.astype(np.float16).astype(np.float64) + 1j * b.imag.astype(np.float16).astype(np.float64)
    return np.sum(np.conj(a16) * b16)


def check(a, b):
    a = a.astype(np.complex64).astype(np.complex128)      # the kernels start from fp32 values
    b = b.astype(np.complex64).astype(np.complex128)
    err = abs(r16(a, b) - np.sum(np.conj(a) * b))
    assert err <= bound(a, b), (err, bound(a, b))
    return err / bound(a, b)


@pytest.mark.parametrize("k", [16, 256, 1024])
def test_random_vectors(k):
    rng = np.random.default_rng(k)
    worst = 0.0
    for trial in range(200):
        a = rng.normal(size=k) + 1j * rng.normal(size=k)
        a /= np.linalg.norm(a) * rng.uniform(0.5, 2.0)              # ||c_t|| / sigma_t around 1
        b = (rng.normal(size=k) + 1j * rng.normal(size=k)) * rng.uniform(0.1, 30.0)
        worst = max(worst, check(a, b))
    assert worst < 1.0


def test_adversarial_midpoints_all_errors_aligned():
    """Every component sits just past a rounding midpoint and all signs conspire: the bound is approached, not passed."""
    k = 256
    m = 1.0 + 2.0 ** -11 + 2.0 ** -20                            # just above the midpoint between 1 and 1 + 2^-10
    for e in (0, 4, 9):
        a = np.full(k, m * 2.0 ** -5) * (1 + 1j)                   # power-of-two scales keep the midpoint position
        b = np.full(k, m * 2.0 ** e) * (1 + 1j)
        ratio = check(a, b)
        assert 0.9 < ratio <= 1.0                                  # Cauchy-Schwarz is attained: the bound is sharp


def test_subnormal_range_and_mixed_magnitudes():
    rng = np.random.default_rng(7)
    k = 512
    a = (rng.normal(size=k) + 1j * rng.normal(size=k)) * 10.0 ** rng.uniform(-9, -1, size=k)   # down into fp16 subnormals
    b = (rng.normal(size=k) + 1j * rng.normal(size=k)) * 10.0 ** rng.uniform(-8, 1.5, size=k)
    check(a, b)
    check(a * 1e-3, b)
    check(a, np.zeros(k))


def test_constants_match_the_library_source():
    src = open(os.path.join(os.path.dirname(__file__), "..", "paper_2110_13115_b200", "csrc", "rbmf_api.cu")).read()
    assert re.search(r"u = ldexp\(1\.0, -11\)", src) and re.search(r"eta = ldexp\(1\.0, -25\) \* 1\.4142135623730951", src)
    # kappa1 carries 2u + u^2 (plus the accumulation term), kappa2 carries eta sqrt(k); both inflated, never deflated
    assert "2.0 * u + u * u" in src and "eta * sqrt(k) * 1.001" in src
