"""Pins of oracle/fitting.py (forward-fitting pieces): the counter-based generator against its published
known-answer vectors, the Poisson sampler against scipy.stats.poisson, the discrepancies against closed forms, hand-worked
examples, brute force and scipy's log-pmf."""
import math
import os

import numpy as np
import pytest
from scipy import stats

from oracle import fitting as F

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def test_philox_known_answer_vectors():
    rows = [l.split() for l in open(os.path.join(GOLDEN, "philox4x32_10_kat.txt")) if l.strip() and not l.startswith("#")]
    assert len(rows) == 3
    for r in rows:
        v = [int(x, 16) for x in r]
        assert list(F.philox4x32_10(v[0:4], v[4:6])) == v[6:10]


def test_uniforms_are_open_unit_interval_and_counter_based():
    u = np.array([F._uniforms(p, 3, 0, 99) for p in range(4000)])
    assert u.min() > 0.0 and u.max() < 1.0
    assert abs(u.mean() - 0.5) < 0.02 and abs(np.corrcoef(u[:, 0], u[:, 1])[0, 1]) < 0.05
    assert F._uniforms(17, 3, 0, 99) == F._uniforms(17, 3, 0, 99) != F._uniforms(17, 3, 1, 99)
    assert F._uniforms(17, 3, 0, 99) != F._uniforms(17, 4, 0, 99) != F._uniforms(17, 4, 0, 100)
    assert F._uniforms((1 << 32) + 17, 3, 0, 99) != F._uniforms(17, 3, 0, 99)          # high word of the pixel index counts


@pytest.mark.parametrize("lam", [0.3, 4.0, 9.9, 10.0, 37.5, 1000.0, 1.0e5])
def test_poisson_moments(lam):
    n = 20000
    x = np.array([F.poisson_sample(lam, p, 0, 12345) for p in range(n)], dtype=np.float64)
    assert abs(x.mean() - lam) < 5.0 * math.sqrt(lam / n)
    # var of the sample variance ~ (2 lam^2 + lam) / n
    assert abs(x.var() - lam) < 5.0 * math.sqrt((2 * lam * lam + lam) / n)
    assert x.min() >= 0 and np.all(x == np.floor(x))


@pytest.mark.parametrize("lam", [4.0, 9.999, 10.0, 37.5])
def test_poisson_pmf_chi_square(lam):
    """Both branches (inversion below 10, transformed rejection from 10 on) reproduce the Poisson pmf."""
    n = 40000
    x = np.array([F.poisson_sample(lam, p, 1, 777) for p in range(n)])
    lo, hi = int(stats.poisson.ppf(1e-3, lam)), int(stats.poisson.ppf(1 - 1e-3, lam))
    edges = np.arange(lo, hi + 2)
    obs = np.array([np.sum(x < lo)] + [np.sum(x == k) for k in edges[:-1]] + [np.sum(x > hi)], dtype=np.float64)
    exp = n * np.array([stats.poisson.cdf(lo - 1, lam)] + [stats.poisson.pmf(k, lam) for k in edges[:-1]] +
                       [stats.poisson.sf(hi, lam)])
    keep = exp > 5
    chi2 = np.sum((obs[keep] - exp[keep]) ** 2 / exp[keep])
    assert chi2 < stats.chi2.ppf(1 - 1e-4, keep.sum() - 1)


def test_poisson_degenerate_means():
    assert F.poisson_sample(0.0, 5, 0, 1) == 0 and F.poisson_sample(-1.0, 5, 0, 1) == 0
    assert F.poisson_sample(float("nan"), 5, 0, 1) == 0


def test_ideal_detector_means_and_streams():
    rng = np.random.default_rng(5)
    I = rng.uniform(0.0, 2.0, (3, 500))
    I[1] = 0.0                                                  # an empty pattern stays empty
    n_ph = np.array([1.0e3, 5.0e4, 2.0e6])
    lam = F.ideal_detector_means(I, n_ph)
    assert np.allclose(lam.sum(axis=1), [1.0e3, 0.0, 2.0e6], rtol=1e-12)
    c = F.ideal_detector(I, n_ph, seed=42)
    assert np.all(c[1] == 0) and np.array_equal(c, F.ideal_detector(I, n_ph, seed=42))
    assert not np.array_equal(c, F.ideal_detector(I, n_ph, seed=43))
    assert abs(c[0].sum() - 1.0e3) < 5 * math.sqrt(1.0e3) and abs(c[2].sum() - 2.0e6) < 5 * math.sqrt(2.0e6)
    # a pixel's draw depends only on (its mean, pixel index, item index, seed): permuting the other items changes nothing
    c2 = F.ideal_detector(I[[0]], n_ph[[0]], seed=42)
    assert np.array_equal(c2[0], c[0])
    # signal to noise grows with the photon number: relative scatter ~ 1 / sqrt(lambda)
    r0 = np.std((c[0] - lam[0])[lam[0] > 1]) / np.mean(lam[0][lam[0] > 1])
    r2 = np.std((c[2] - lam[2])[lam[2] > 1]) / np.mean(lam[2][lam[2] > 1])
    assert r2 < 0.1 * r0


def test_discrepancy_l2_closed_forms():
    rng = np.random.default_rng(8)
    I = rng.uniform(0.1, 3.0, (4, 300))
    assert np.all(F.discrepancy_l2(I, I[0])[0:1] < 1e-30)
    assert np.all(F.discrepancy_l2(I, 3.7 * I) < 1e-28)                         # scale-free
    assert np.allclose(F.discrepancy_l2(np.array([[1.0, 3.0]]), np.array([1.0, 1.0])), [0.125], rtol=1e-15)   # by hand
    M = rng.uniform(0.1, 3.0, 300)
    mask = (rng.uniform(size=300) < 0.6).astype(np.uint8)
    d = F.discrepancy_l2(I, M, mask)
    keep = mask != 0
    assert np.allclose(d, F.discrepancy_l2(I[:, keep], M[keep]), rtol=1e-13)    # masked pixels do not exist
    brute = []
    for b in range(4):
        si = sum(I[b, p] for p in range(300) if mask[p])
        sm = sum(M[p] for p in range(300) if mask[p])
        brute.append(sum((I[b, p] / si - M[p] / sm) ** 2 for p in range(300) if mask[p]))
    assert np.allclose(d, brute, rtol=1e-12)
    # symmetric in its two arguments, per-item measured patterns
    Mb = rng.uniform(0.1, 3.0, (4, 300))
    assert np.allclose(F.discrepancy_l2(I, Mb), F.discrepancy_l2(Mb, I), rtol=1e-13)


def test_discrepancy_poisson_is_the_scale_fitted_deviance():
    rng = np.random.default_rng(9)
    I = rng.uniform(0.5, 4.0, (3, 200))
    assert np.all(np.abs(F.discrepancy_poisson(I, 5.0 * I)) < 1e-9)              # exact model: zero deviance
    # by hand: I = (1, 1), M = (1, 3): c = 2, mu = (2, 2): 2 [ln(1/2) + 1 + 3 ln(3/2) - 1]
    assert np.allclose(F.discrepancy_poisson(np.array([[1.0, 1.0]]), np.array([1.0, 3.0])),
                       [2.0 * (math.log(0.5) + 1.0 + 3.0 * math.log(1.5) - 1.0)], rtol=1e-14)
    M = rng.poisson(7.0 * I[0]).astype(np.float64)
    M[:5] = 0.0                                                                  # empty pixels: M log M = 0
    mask = (rng.uniform(size=200) < 0.7).astype(np.uint8)
    d = F.discrepancy_poisson(I, M, mask)
    keep = mask != 0
    for b in range(3):
        c = M[keep].sum() / I[b, keep].sum()
        mu = c * I[b, keep]
        ref = 2.0 * np.sum(stats.poisson.logpmf(M[keep], np.where(M[keep] > 0, M[keep], 1e-300)) - stats.poisson.logpmf(M[keep], mu))
        assert np.isclose(d[b], ref, rtol=1e-9)
    assert np.all(d >= 0) and d[0] < d[1] and d[0] < d[2]                        # the true model fits best
