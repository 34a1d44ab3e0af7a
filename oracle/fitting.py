"""Forward-fitting pieces -- FP64 CPU oracle, TEST INFRASTRUCTURE ONLY (imported by tests/, smoke() and
bench.py's cpu_baseline leg; never by the product path).  Plain numpy / Python, no code shared with the CUDA path.

What the paper fixes and what is a reading (R22-R24):
  * Comparing a simulation with a measured pattern: "both ... profiles were normalized on their integral value computed
    between 10 and 30 degrees" (Fig. 5) -> `discrepancy_l2`: squared distance of the two patterns after each is
    divided by its integral over the masked region.
  * Ideal detector: "even a perfect real-life detector is subjected to Poisson statistics of photons ... an
    estimate on the amount of scattered photons has to be calculated, and then used to add the proper Poisson noise".  The
    estimate itself is in the Supplemental Material, which is not available: here the caller passes the expected number of
    detected photons per pattern, the pixel means are lambda_p = n_photons * I_p / sum(I) and the counts are Poisson(lambda_p)
    drawn from a counter-based generator (Philox-4x32-10, Salmon et al. 2011) so that both sides draw the same numbers.
  * `discrepancy_poisson`: the Poisson deviance of measured counts against the scale-fitted simulation (the maximum-likelihood
    counterpart of the Ideal detector's noise model).
"""
from __future__ import annotations

import math

import numpy as np

M32 = 0xFFFFFFFF
PHILOX_M0, PHILOX_M1 = 0xD2511F53, 0xCD9E8D57      # multipliers of Philox-4x32
PHILOX_W0, PHILOX_W1 = 0x9E3779B9, 0xBB67AE85      # Weyl key increments (golden ratio, sqrt 3 - 1)


def philox4x32_10(counter, key):
    """One block of Philox-4x32 with 10 rounds: counter = 4 x uint32, key = 2 x uint32 -> 4 x uint32 (Python ints)."""
    c0, c1, c2, c3 = (int(c) & M32 for c in counter)
    k0, k1 = (int(k) & M32 for k in key)
    for _ in range(10):
        p0 = PHILOX_M0 * c0
        p1 = PHILOX_M1 * c2
        c0, c1, c2, c3 = ((p1 >> 32) ^ c1 ^ k0) & M32, p1 & M32, ((p0 >> 32) ^ c3 ^ k1) & M32, p0 & M32
        k0 = (k0 + PHILOX_W0) & M32
        k1 = (k1 + PHILOX_W1) & M32
    return c0, c1, c2, c3


def _uniforms(p: int, b: int, draw: int, seed: int):
    """Two uniforms in (0, 1) for pixel p of item b, draw number `draw`: counter (p lo, p hi, b, draw), key = seed."""
    x = philox4x32_10((p & M32, (p >> 32) & M32, b, draw), (seed & M32, (seed >> 32) & M32))
    return (x[0] + 0.5) * 2.0 ** -32, (x[1] + 0.5) * 2.0 ** -32


def poisson_sample(lam: float, p: int, b: int, seed: int) -> int:
    """One Poisson(lam) variate from the (p, b, seed) stream.  lam < 10: inversion by sequential search on one uniform;
    lam >= 10: Hoermann's transformed rejection with squeeze (PTRS, 1993), one (U, V) pair per attempt."""
    if not lam > 0.0:
        return 0
    if lam < 10.0:
        u, _ = _uniforms(p, b, 0, seed)
        k = 0
        pk = math.exp(-lam)
        s = pk
        while u > s and k < 1000:
            k += 1
            pk *= lam / k
            s += pk
        return k
    slam = math.sqrt(lam)
    loglam = math.log(lam)
    bb = 0.931 + 2.53 * slam
    a = -0.059 + 0.02483 * bb
    invalpha = 1.1239 + 1.1328 / (bb - 3.4)
    vr = 0.9277 - 3.6224 / (bb - 2.0)
    draw = 0
    while True:
        u, v = _uniforms(p, b, draw, seed)
        draw += 1
        u -= 0.5
        us = 0.5 - abs(u)
        k = math.floor((2.0 * a / us + bb) * u + lam + 0.43)
        if us >= 0.07 and v <= vr:
            return int(k)
        if k < 0 or (us < 0.013 and v > us):
            continue
        if math.log(v) + math.log(invalpha) - math.log(a / (us * us) + bb) <= -lam + k * loglam - math.lgamma(k + 1.0):
            return int(k)


def ideal_detector(I: np.ndarray, n_photons, seed: int) -> np.ndarray:
    """Counts float64 [B][npix]: Poisson(n_photons[b] * I[b][p] / sum_p I[b][p]).  I: [B][npix] (any float type)."""
    I = np.asarray(I, dtype=np.float64)
    B, npix = I.shape
    n_photons = np.broadcast_to(np.asarray(n_photons, dtype=np.float64), (B,))
    out = np.zeros((B, npix), dtype=np.float64)
    for b in range(B):
        s = float(np.sum(I[b]))
        if not s > 0.0:
            continue
        gain = n_photons[b] / s
        for p in range(npix):
            out[b, p] = poisson_sample(float(I[b, p]) * gain, p, b, seed)
    return out


def ideal_detector_means(I: np.ndarray, n_photons) -> np.ndarray:
    """The Poisson means lambda[b][p] of `ideal_detector`."""
    I = np.asarray(I, dtype=np.float64)
    n_photons = np.broadcast_to(np.asarray(n_photons, dtype=np.float64), (I.shape[0],))
    s = I.sum(axis=1, keepdims=True)
    return np.where(s > 0, I * (n_photons[:, None] / np.where(s > 0, s, 1.0)), 0.0)


def _masked(I, M, mask):
    I = np.asarray(I, dtype=np.float64)
    M = np.broadcast_to(np.asarray(M, dtype=np.float64), I.shape)
    w = np.ones(I.shape[1]) if mask is None else (np.asarray(mask) != 0).astype(np.float64)
    return I, M, w


def discrepancy_l2(I, M, mask=None) -> np.ndarray:
    """D[b] = sum_p w_p (I[b][p] / S_I - M[p] / S_M)^2 with S = sum_p w_p (.), the integral normalisation of Fig. 5
    (PAPER.md:180); w = mask != 0.  I: [B][npix]; M: [npix] or [B][npix]."""
    I, M, w = _masked(I, M, mask)
    SI = (I * w).sum(axis=1, keepdims=True)
    SM = (M * w).sum(axis=1, keepdims=True)
    return (w * (I / SI - M / SM) ** 2).sum(axis=1)


def discrepancy_poisson(I, M, mask=None) -> np.ndarray:
    """Poisson deviance of measured counts M against the scale-fitted simulation mu = c I, c = S_M / S_I (the maximum-
    likelihood scale): D[b] = 2 sum_p w_p [ M log(M / mu) - (M - mu) ], with M log(M / mu) = 0 where M = 0."""
    I, M, w = _masked(I, M, mask)
    SI = (I * w).sum(axis=1, keepdims=True)
    SM = (M * w).sum(axis=1, keepdims=True)
    mu = I * (SM / SI)
    with np.errstate(divide="ignore", invalid="ignore"):
        t = np.where(M > 0, M * np.log(M / mu), 0.0) - (M - mu)
    return 2.0 * (w * t).sum(axis=1)
