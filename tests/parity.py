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


# ---- full-size sampled parity (pixels are independent, so a seeded subset is exact, not approximate) -------------
_REF_CACHE = {}


def oracle_at_pixels(w, item, g, quat, pix):
    """The oracle's I at the pixels `pix` of item `item` of workload `w` (grid g, orientation quat).  Pixels are independent,
    so every (workload, item, pixel) value is computed once per test session and shared by the routes that are checked
    on the same sample (pixel contraction as CTA pairs and as single CTAs, NUFFT)."""
    from oracle import oracle as O
    cache = _REF_CACHE.setdefault((w.name, w.nx, w.npx, int(item)), {})
    missing = np.array(sorted({int(p) for p in pix} - cache.keys()), dtype=np.int64)
    if missing.size:
        ref = O.simulate(g, (w.dx, w.dy, w.dz), w.lam, w.npx, w.npy, w.theta_max_deg, quat=quat, pixels=missing)
        cache.update(zip(missing.tolist(), np.asarray(ref, dtype=np.float64).tolist()))
    return np.array([cache[int(p)] for p in pix], dtype=np.float64)


# sample sizes of SURVEY 8(d) (cfg3: 2048 of the 8192 it names -- the oracle takes ~20 ms per cfg3 pixel on 16 cores)
FULL_SIZE_SAMPLES = {1: 2048, 2: 2048, 3: 256, 4: 1024}


def sampled_pixels(w, item, I_flat, count):
    """Seeded sample + the pixels DESIGN.md R14 always includes (the GPU pattern's arg-max, the four centre pixels) + corners."""
    from paper_2202_03411_b200 import workloads as W
    c = w.npy // 2 * w.npx + w.npx // 2
    always = [int(np.argmax(I_flat)), c, c - 1, c - w.npx, c - w.npx - 1, 0, w.npx - 1, w.npix - w.npx, w.npix - 1]
    return W.sample_pixels(w.seed + item, w.npix, count, always=always)
