"""GPU parity of the forward-fitting pieces (scatman_discrepancy, scatman_ideal_detector; fit_kernels.cu) against
oracle/fitting.py: discrepancies to FP64 summation-order accuracy, Poisson counts integer for integer."""
import math

import numpy as np
import pytest

from oracle import fitting as F
from oracle import oracle as O
from paper_2202_03411_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def sm():
    import torch
    from paper_2202_03411_b200 import binding as B, build
    build.build()
    assert torch.cuda.is_available()
    s = B.Scatman(0)
    yield s
    s.close()


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.mark.parametrize("metric", [0, 1])
@pytest.mark.parametrize("per_item", [False, True])
def test_discrepancy_matches_oracle_over_several_chunks_and_a_ragged_tail(sm, metric, per_item):
    rng = np.random.default_rng(101 + metric)
    B_, npix = 5, 2 * 32768 + 777
    I = (rng.uniform(0.0, 1.0, (B_, npix)) ** 4 * 1e3).astype(np.float32)          # wide dynamic range, like a pattern
    M = rng.poisson(3.0 * I[0] if not per_item else 3.0 * I).astype(np.float32)
    mask = (rng.uniform(size=npix) < 0.8).astype(np.uint8)
    fn = F.discrepancy_l2 if metric == 0 else F.discrepancy_poisson
    for mk in (None, mask):
        got = sm.discrepancy(dev(I), dev(M), None if mk is None else dev(mk), metric=metric).cpu().numpy()
        ref = fn(I, M, mk)
        assert np.allclose(got, ref, rtol=1e-11, atol=0), (metric, per_item, got, ref)


@pytest.mark.parametrize("metric", [0, 1])
def test_discrepancy_with_16_byte_loads_and_without(sm, metric):
    """Pixel counts that are multiples of four take 16-byte loads of the patterns and 4-byte loads of the mask (a last chunk
    that is not full, a count below one load per thread, mask bytes other than 1, NaN under the mask); the same data
    through views that start one element later (no longer 16-byte aligned) takes the scalar kernels: both against the oracle."""
    import torch
    rng = np.random.default_rng(131 + metric)
    fn = F.discrepancy_l2 if metric == 0 else F.discrepancy_poisson
    # (pixels per block: 2048 or 8192 for the small problems, 32768 for the last one -- 1800 chunks; the first has more than 32
    # chunks per item, so its sums go through the reduction launch, the others add them inside pass 2)
    for B_, npix, per_item in ((4, 2 * 32768 + 4 * 333, True), (3, 32768, False), (2, 8, False), (3, 4 * 1024 + 4, True),
                               (600, 3 * 32768 - 20, False)):
        I = (rng.uniform(0.0, 1.0, (B_, npix)) ** 4 * 1e3 + 1e-3).astype(np.float32)
        M = rng.poisson(3.0 * I if per_item else 3.0 * I[0]).astype(np.float32)
        mask = ((rng.uniform(size=npix) < 0.8) * rng.integers(1, 256, npix)).astype(np.uint8)
        Ibad = I.copy()
        Ibad[:, mask == 0] = np.nan                                   # what the mask hides is never used
        ref = fn(I, M, mask)
        got = sm.discrepancy(dev(Ibad), dev(M), dev(mask), metric=metric).cpu().numpy()
        assert np.allclose(got, ref, rtol=1e-11, atol=0), (npix, got, ref)
        assert np.allclose(sm.discrepancy(dev(I), dev(M), metric=metric).cpu().numpy(), fn(I, M, None), rtol=1e-11, atol=0)
        # one element off the 16-byte grid
        pad = lambda a: torch.cat([torch.zeros(1, dtype=a.dtype, device="cuda"), a.reshape(-1)])[1:].reshape(a.shape)
        Iu, Mu, mu = pad(dev(Ibad)), pad(dev(M)), pad(dev(mask))
        assert Iu.data_ptr() % 16 == 4 and mu.data_ptr() % 4 == 1
        got = sm.discrepancy(Iu, Mu, mu, metric=metric).cpu().numpy()
        assert np.allclose(got, ref, rtol=1e-11, atol=0), (npix, got, ref)


def test_discrepancy_degenerate_cases(sm):
    rng = np.random.default_rng(7)
    I = rng.uniform(0.5, 2.0, (2, 1000)).astype(np.float32)
    assert np.all(sm.discrepancy(dev(I), dev(I), metric=0).cpu().numpy() == 0.0)              # identical patterns
    d = sm.discrepancy(dev(I), dev((4.0 * I).astype(np.float32)), metric=1).cpu().numpy()    # scaled copy: zero deviance
    assert np.all(np.abs(d) < 1e-6)
    one = sm.discrepancy(dev(I[:, :1]), dev(I[0, :1]), metric=0).cpu().numpy()                # a single pixel: 1/1 - 1/1
    assert np.all(one < 1e-30)                                                                # x * (1 / x) may miss 1 by an ulp
    M = I[0].copy()
    M[:10] = 0.0                                                                              # empty measured pixels
    got = sm.discrepancy(dev(I), dev(M), metric=1).cpu().numpy()
    assert np.allclose(got, F.discrepancy_poisson(I, M), rtol=1e-11)


def test_ideal_detector_counts_equal_the_oracles(sm):
    rng = np.random.default_rng(55)
    B_, npix = 3, 3000
    I = (rng.uniform(0.0, 1.0, (B_, npix)) ** 6).astype(np.float32)
    I[1, ::7] = 0.0
    n_ph = np.array([2.0e3, 6.0e4, 3.0e8])                       # means from << 1 (inversion) to ~1e5 (transformed rejection)
    got = sm.ideal_detector(dev(I), n_ph, seed=2022_03411).cpu().numpy().astype(np.float64)
    ref = F.ideal_detector(I, n_ph, seed=2022_03411)
    lam = F.ideal_detector_means(I, n_ph)
    assert (lam < 10).sum() > 500 and (lam >= 10).sum() > 500
    assert np.sum(got != ref) <= 1, np.flatnonzero(got != ref)   # FP64 library roundings could flip a draw once in ~1e13
    assert np.all(got[1, ::7] == 0)
    again = sm.ideal_detector(dev(I), n_ph, seed=2022_03411).cpu().numpy()
    assert np.array_equal(again, got.astype(np.float32))
    other = sm.ideal_detector(dev(I), n_ph, seed=1).cpu().numpy()
    assert not np.array_equal(other, got.astype(np.float32))


def test_ideal_detector_full_detector_sampled_pixels_and_totals(sm):
    """cfg5's 1024 x 1024 detector, two items: totals within Poisson scatter, seeded pixels checked one by one."""
    rng = np.random.default_rng(56)
    npix = 1024 * 1024
    I = (rng.uniform(0.0, 1.0, (2, npix)) ** 8).astype(np.float32)
    n_ph = np.array([1.0e5, 1.0e9])
    got = sm.ideal_detector(dev(I), n_ph, seed=77).cpu().numpy().astype(np.float64)
    for b in range(2):
        assert abs(got[b].sum() - n_ph[b]) < 6.0 * math.sqrt(n_ph[b])
    lam = F.ideal_detector_means(I, n_ph)
    pix = W.sample_pixels(91, npix, 300)
    for b in range(2):
        ref = np.array([F.poisson_sample(float(lam[b, p]), int(p), b, 77) for p in pix])
        assert np.sum(got[b, pix] != ref) <= 1
    zero = sm.ideal_detector(dev(np.zeros((1, 4096), np.float32)), 1.0e6, seed=3).cpu().numpy()
    assert np.all(zero == 0)


def test_simulated_pattern_through_detector_and_discrepancy(sm):
    """Hot path -> Ideal detector -> deviance: the noisy counts of the true shape fit it with deviance ~ 1 per pixel, a wrong
    shape fits worse (the forward-fitting loop of PAPER.md:431 in one pass)."""
    import torch
    w = W.config(0)
    vox = (w.dx, w.dy, w.dz)
    g = w.grid(0)
    g2 = g.copy()
    g2[:, :, :12] = 0.0                                           # a truncated sphere: the wrong candidate
    I = sm.simulate(dev(np.stack([g, g2])), vox, w.lam, w.npx, w.npy, w.theta_max_deg)
    counts = sm.ideal_detector(I[:1].contiguous(), 5.0e6, seed=11)
    d = sm.discrepancy(I, counts[0].contiguous(), metric=1).cpu().numpy()
    npix = w.npx * w.npy
    assert 0.8 < d[0] / npix < 1.25 and d[1] > 3.0 * d[0]
    ref = F.discrepancy_poisson(I.cpu().numpy().reshape(2, -1), counts[0].cpu().numpy().ravel())
    assert np.allclose(d, ref, rtol=1e-10)


def test_fitting_error_codes(sm):
    import torch
    from paper_2202_03411_b200 import binding as B
    I = dev(np.ones((2, 100), np.float32))
    with pytest.raises(B.ScatmanError) as e:
        sm.discrepancy(I, I, metric=7)
    assert e.value.status == B.INVALID_ARGUMENT
    with pytest.raises(B.ScatmanError) as e:
        sm.ideal_detector(I, -5.0, seed=1)
    assert e.value.status == B.INVALID_ARGUMENT
