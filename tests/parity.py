"""Parity metrics of BASELINE.json's north_star: rel-L2 over the pattern <= 1e-4 and per-pixel relative
error <= 1e-3 on pixels above 1e-6 of the peak intensity (peak taken from the oracle, R14)."""
import numpy as np

REL_L2_TOL = 1e-4
PIXEL_TOL = 1e-3
PEAK_FLOOR = 1e-6


def metrics(I_gpu, I_ref):
    g = np.asarray(I_gpu, dtype=np.float64).ravel()
    r = np.asarray(I_ref, dtype=np.float64).ravel()
    assert g.shape == r.shape
    denom = np.sqrt(np.sum(r * r))
    rel_l2 = float(np.sqrt(np.sum((g - r) ** 2)) / denom) if denom > 0 else float(np.max(np.abs(g)))
    peak = r.max() if r.size else 0.0
    m = r > PEAK_FLOOR * peak
    pix = float(np.max(np.abs(g[m] - r[m]) / r[m])) if m.any() else 0.0
    return rel_l2, pix


def assert_parity(I_gpu, I_ref, l2_tol=REL_L2_TOL, pix_tol=PIXEL_TOL, what=""):
    assert np.all(np.isfinite(np.asarray(I_gpu))), f"{what}: non-finite output"
    rel_l2, pix = metrics(I_gpu, I_ref)
    assert rel_l2 <= l2_tol and pix <= pix_tol, f"{what}: rel_l2={rel_l2:.3e} (tol {l2_tol}), max pixel rel={pix:.3e} (tol {pix_tol})"
    return rel_l2, pix
