"""Seeded synthetic input generators for the five BASELINE.json configs.

This module serves BOTH the CUDA path and the oracle and therefore holds none of
the method's arithmetic: it only voxelises shapes into FP32 (delta, beta) grids
(binary voxelisation at voxel centres, like the paper's VolumeMap),
draws seeded quaternions, and names the experiment parameters (lambda, theta_max,
detector size).  numpy only.

The paper's own workloads (Fig. 8: Ellipsoid / SphericalHarmonics / RadialMap /
VolumeMap) need data arrays that are not available; the five
configs below take their shapes and sizes and stand in for them (DESIGN.md,
"Input recipe").
"""
from __future__ import annotations

import dataclasses
from typing import List, Optional

import numpy as np

BASE_SEED = 220203411


@dataclasses.dataclass
class Workload:
    name: str
    index: int                   # 0-based index into BASELINE.json configs
    nx: int
    ny: int
    nz: int
    dx: float                    # voxel size, same length unit as lam
    dy: float
    dz: float
    lam: float                   # wavelength
    npx: int
    npy: int
    theta_max_deg: float
    batch: int
    quat: Optional[np.ndarray]   # [batch][4] (w,x,y,z) float64 or None = identity
    seed: int
    _gen: object = None          # callable(b) -> float32 [nz][ny][nx][2]
    _shape: object = None        # callable(b) -> shape descriptor dict (scatman_shape fields) or None if not a single shape

    @property
    def nvox(self) -> int:
        return self.nx * self.ny * self.nz

    @property
    def npix(self) -> int:
        return self.npx * self.npy

    @property
    def terms(self) -> int:
        return self.nvox * self.npix * self.batch

    def grid(self, b: int = 0) -> np.ndarray:
        """Body-frame (delta, beta) grid of batch item b, float32 [nz][ny][nx][2]."""
        return self._gen(b)

    def shapes(self, items=None):
        """Shape descriptors (the fields of scatman_shape, orientation included) of the items: the same particles as grid(b),
        for rendering on the device.  None for workloads that are not one shape per item (cfg5)."""
        if self._shape is None:
            return None
        items = range(self.batch) if items is None else items
        out = []
        for b in items:
            d = dict(self._shape(b))
            if self.quat is not None:
                d["quat"] = [float(v) for v in self.quat[b]]
            out.append(d)
        return out

    def grids(self, items=None) -> np.ndarray:
        items = range(self.batch) if items is None else items
        return np.stack([self.grid(b) for b in items], axis=0)


# ----------------------------------------------------------------------------- geometry
def _centres(n: int, d: float) -> np.ndarray:
    return (np.arange(n, dtype=np.float64) - (n - 1) / 2.0) * d


def _coords(nx, ny, nz, dx, dy, dz):
    z = _centres(nz, dz)[:, None, None]
    y = _centres(ny, dy)[None, :, None]
    x = _centres(nx, dx)[None, None, :]
    return x, y, z


def _fill(mask: np.ndarray, delta: float, beta: float, out: Optional[np.ndarray] = None) -> np.ndarray:
    if out is None:
        out = np.zeros(mask.shape + (2,), dtype=np.float32)
    out[mask, 0] = np.float32(delta)
    out[mask, 1] = np.float32(beta)
    return out


def ellipsoid_mask(nx, ny, nz, dx, dy, dz, a, b, c, centre=(0.0, 0.0, 0.0)) -> np.ndarray:
    x, y, z = _coords(nx, ny, nz, dx, dy, dz)
    return ((x - centre[0]) / a) ** 2 + ((y - centre[1]) / b) ** 2 + ((z - centre[2]) / c) ** 2 <= 1.0


def sh_radius_factor(coeffs, cos_theta: np.ndarray, phi: np.ndarray) -> np.ndarray:
    """1 + sum_lm a_lm Y_lm(theta, phi) with real orthonormal Y_lm (theta = polar angle from +z).

    Associated Legendre functions by the standard upward recurrences (Condon-Shortley phase).
    coeffs = [(l, m, a_lm), ...].
    """
    from math import factorial, pi, sqrt
    lmax = max(l for l, _, _ in coeffs)
    x = np.asarray(cos_theta, dtype=np.float64)
    s = np.sqrt(np.maximum(0.0, 1.0 - x * x))
    P = {}
    pmm = np.ones_like(x)
    for m in range(0, lmax + 1):
        if m > 0:
            pmm = -pmm * (2 * m - 1) * s
        P[(m, m)] = pmm
        if m + 1 <= lmax:
            P[(m + 1, m)] = x * (2 * m + 1) * pmm
        for l in range(m + 2, lmax + 1):
            P[(l, m)] = ((2 * l - 1) * x * P[(l - 1, m)] - (l + m - 1) * P[(l - 2, m)]) / (l - m)
    out = np.ones_like(x)
    for (l, m, a) in coeffs:
        am = abs(m)
        norm = sqrt((2 * l + 1) / (4 * pi) * factorial(l - am) / factorial(l + am))
        if m == 0:
            out += a * norm * P[(l, 0)]
        elif m > 0:
            out += a * sqrt(2.0) * norm * P[(l, am)] * np.cos(am * phi)
        else:
            out += a * sqrt(2.0) * norm * P[(l, am)] * np.sin(am * phi)
    return out


def droplet_mask(nx, ny, nz, dx, dy, dz, r0: float, coeffs) -> np.ndarray:
    """Inside of R(theta,phi) = r0 (1 + sum a_lm Y_lm); coeffs = [(l, m, a_lm), ...]."""
    x, y, z = _coords(nx, ny, nz, dx, dy, dz)
    r = np.sqrt(x * x + y * y + z * z)
    # bracket the radius factor on a coarse angular grid, then evaluate it only in the shell between
    ct_g = np.linspace(-1.0, 1.0, 361)[:, None]
    ph_g = np.linspace(-np.pi, np.pi, 721)[None, :]
    f_g = sh_radius_factor(coeffs, np.broadcast_to(ct_g, (361, 721)), np.broadcast_to(ph_g, (361, 721)))
    f_lo, f_hi = float(f_g.min()) - 0.02, float(f_g.max()) + 0.02
    mask = r <= r0 * f_lo
    shell = (r > r0 * f_lo) & (r <= r0 * f_hi)
    idx = np.nonzero(shell)
    if idx[0].size:
        xs = np.broadcast_to(x, r.shape)[idx]
        ys = np.broadcast_to(y, r.shape)[idx]
        zs = np.broadcast_to(z, r.shape)[idx]
        rs = r[idx]
        ct = np.clip(zs / np.maximum(rs, 1e-300), -1.0, 1.0)
        ph = np.arctan2(ys, xs)
        mask[idx] = rs <= r0 * sh_radius_factor(coeffs, ct, ph)
    return mask


def random_quaternions(rng: np.random.Generator, n: int) -> np.ndarray:
    """Uniform random unit quaternions (w,x,y,z), float64 [n][4]."""
    q = rng.standard_normal((n, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    q[q[:, 0] < 0] *= -1.0
    return q


def quat_from_lat_long_rot(latitude_deg: float, longitude_deg: float, rotation_deg: float) -> np.ndarray:
    """PyScatman-style orientation (Fig. 6) -> body->beam quaternion.

    Reading (R11): the shape's main axis is body +z; latitude 90 deg points it
    towards the incoming beam (-z of the beam frame), latitude 0 puts it on the equator
    (perpendicular to the beam) at the given longitude measured from +x towards +y; the
    shape is then spun by `rotation` about its main axis.
    """
    la, lo, ro = np.deg2rad([latitude_deg, longitude_deg, rotation_deg])
    axis = np.array([np.cos(la) * np.cos(lo), np.cos(la) * np.sin(lo), -np.sin(la)])
    zb = np.array([0.0, 0.0, 1.0])
    v = np.cross(zb, axis)
    s = np.linalg.norm(v)
    c = float(np.dot(zb, axis))
    if s < 1e-15:
        q_align = np.array([1.0, 0.0, 0.0, 0.0]) if c > 0 else np.array([0.0, 1.0, 0.0, 0.0])
    else:
        ang = np.arctan2(s, c)
        q_align = np.concatenate([[np.cos(ang / 2)], np.sin(ang / 2) * v / s])
    q_spin = np.array([np.cos(ro / 2), 0.0, 0.0, np.sin(ro / 2)])
    return quat_mul(q_align, q_spin)


def quat_mul(a: np.ndarray, b: np.ndarray) -> np.ndarray:
    aw, ax, ay, az = a
    bw, bx, by, bz = b
    return np.array([aw * bw - ax * bx - ay * by - az * bz,
                     aw * bx + ax * bw + ay * bz - az * by,
                     aw * by - ax * bz + ay * bw + az * bx,
                     aw * bz + ax * by - ay * bx + az * bw])


# ----------------------------------------------------------------------------- configs
def _sh_coeffs(rng: np.random.Generator, lmax: int, sigma0: float = 0.05):
    out = []
    for l in range(1, lmax + 1):
        for m in range(-l, l + 1):
            out.append((l, m, float(rng.normal(0.0, sigma0 / l))))
    return out


def _triplets(r0: float, coeffs):
    """R0 (1 + sum a_lm Y_lm) as the paper's triplet list (l, m, c) with R = sum c Y_lm: c_00 = R0 sqrt(4 pi), c_lm = R0 a_lm."""
    return [(0, 0, r0 * float(np.sqrt(4.0 * np.pi)))] + [(l, m, r0 * a) for (l, m, a) in coeffs]


def config(index: int, scale: float = 1.0) -> Workload:
    """Workload for BASELINE.json configs[index] (0..4).

    `scale` < 1 shrinks grid and detector resolution (same physical box and angles) to
    make reduced parity cases; scale=1 is the config as stated.
    """
    seed = BASE_SEED + index + 1
    rng = np.random.default_rng(seed)

    def sc(n, mult=8):
        return max(mult, int(round(n * scale / mult)) * mult)

    if index == 0:
        n, npx = sc(32), sc(64)
        d = 4.0 * 32 / n
        gen = lambda b: _fill(ellipsoid_mask(n, n, n, d, d, d, 60.0, 60.0, 60.0), 0.01, 0.001)
        shp = lambda b: {"kind": "ellipsoid", "delta": 0.01, "beta": 0.001, "a": 60.0, "b": 60.0, "c": 60.0}
        return Workload("cfg1_sphere_32", 0, n, n, n, d, d, d, 20.0, npx, npx, 30.0, 1, None, seed, gen, shp)
    if index == 1:
        n, npx = sc(128), sc(256)
        d = 4.0 * 128 / n
        quat = random_quaternions(rng, 1)
        gen = lambda b: _fill(ellipsoid_mask(n, n, n, d, d, d, 200.0, 150.0, 120.0), 0.02, 0.005)
        shp = lambda b: {"kind": "ellipsoid", "delta": 0.02, "beta": 0.005, "a": 200.0, "b": 150.0, "c": 120.0}
        return Workload("cfg2_ellipsoid_128", 1, n, n, n, d, d, d, 13.5, npx, npx, 40.0, 1, quat, seed, gen, shp)
    if index == 2:
        n, npx = sc(256), sc(512)
        d = 4.0 * 256 / n
        coeffs = _sh_coeffs(rng, 6)
        gen = lambda b: _fill(droplet_mask(n, n, n, d, d, d, 400.0, coeffs), 0.03, 0.01)
        shp = lambda b: {"kind": "spherical_harmonics", "delta": 0.03, "beta": 0.01, "coeffs": _triplets(400.0, coeffs)}
        return Workload("cfg3_droplet_256", 2, n, n, n, d, d, d, 30.0, npx, npx, 45.0, 1, None, seed, gen, shp)
    if index == 3:
        n, npx = sc(128), sc(256)
        d = 6.0 * 128 / n
        batch = 256
        quat = random_quaternions(rng, batch)
        r0 = rng.uniform(100.0, 300.0, batch)
        delta = rng.uniform(0.005, 0.05, batch)
        beta = rng.uniform(0.0, 0.02, batch)
        ratios = rng.uniform(0.6, 1.0, (batch, 2))
        sh_seeds = rng.integers(0, 2 ** 31 - 1, batch)

        def gen(b):
            if b % 2 == 0:
                m = ellipsoid_mask(n, n, n, d, d, d, r0[b], r0[b] * ratios[b, 0], r0[b] * ratios[b, 1])
            else:
                co = _sh_coeffs(np.random.default_rng(int(sh_seeds[b])), 4)
                m = droplet_mask(n, n, n, d, d, d, r0[b], co)
            return _fill(m, delta[b], beta[b])

        def shp(b):
            if b % 2 == 0:
                return {"kind": "ellipsoid", "delta": float(delta[b]), "beta": float(beta[b]), "a": float(r0[b]),
                        "b": float(r0[b] * ratios[b, 0]), "c": float(r0[b] * ratios[b, 1])}
            co = _sh_coeffs(np.random.default_rng(int(sh_seeds[b])), 4)
            return {"kind": "spherical_harmonics", "delta": float(delta[b]), "beta": float(beta[b]), "coeffs": _triplets(float(r0[b]), co)}
        return Workload("cfg4_fit_batch_256x128", 3, n, n, n, d, d, d, 20.0, npx, npx, 35.0, batch, quat, seed, gen, shp)
    if index == 4:
        n, npx = sc(512), sc(1024)
        d = 2.0 * 512 / n
        r_shell, r_core = 480.0, 380.0
        rad = rng.uniform(40.0, 100.0, 8)
        cen = []
        for i in range(8):
            while True:
                c = rng.uniform(-r_core, r_core, 3)
                if np.linalg.norm(c) + rad[i] <= r_core:
                    cen.append(c)
                    break

        def gen(b):
            out = _fill(ellipsoid_mask(n, n, n, d, d, d, r_shell, r_shell, r_shell), 0.02, 0.002)
            _fill(ellipsoid_mask(n, n, n, d, d, d, r_core, r_core, r_core), 0.05, 0.05, out)
            for i in range(8):
                _fill(ellipsoid_mask(n, n, n, d, d, d, rad[i], rad[i], rad[i], centre=cen[i]), 0.08, 0.03, out)
            return out
        return Workload("cfg5_coreshell_512", 4, n, n, n, d, d, d, 10.0, npx, npx, 60.0, 1, None, seed, gen)
    raise ValueError("config index must be 0..4")


def random_grid(seed: int, nx: int, ny: int, nz: int, fill: float = 0.6,
                delta=(-0.02, 0.05), beta=(0.0, 0.02)) -> np.ndarray:
    """Unstructured random (delta, beta) grid with exact zeros: stresses every index."""
    rng = np.random.default_rng(seed)
    out = np.zeros((nz, ny, nx, 2), dtype=np.float32)
    m = rng.random((nz, ny, nx)) < fill
    out[..., 0] = np.where(m, rng.uniform(delta[0], delta[1], m.shape), 0.0)
    out[..., 1] = np.where(m, rng.uniform(beta[0], beta[1], m.shape), 0.0)
    return out


def sparse_blobs_grid(seed: int, nx: int, ny: int, nz: int, nblobs: int = 6, max_extent: int = 24) -> np.ndarray:
    """A few small random boxes of material per slice range in an otherwise empty grid: most 16 x 16 (x, y) blocks of
    most slices are exactly zero, and the occupied x / y ranges differ from slice to slice and tile to tile."""
    rng = np.random.default_rng(seed)
    out = np.zeros((nz, ny, nx, 2), dtype=np.float32)
    for _ in range(nblobs):
        ex, ey, ez = (int(rng.integers(1, max(2, min(max_extent, n)))) for n in (nx, ny, nz))
        x0, y0, z0 = int(rng.integers(0, nx - ex + 1)), int(rng.integers(0, ny - ey + 1)), int(rng.integers(0, nz - ez + 1))
        out[z0:z0 + ez, y0:y0 + ey, x0:x0 + ex, 0] = rng.uniform(-0.02, 0.05)
        out[z0:z0 + ez, y0:y0 + ey, x0:x0 + ex, 1] = rng.uniform(0.0, 0.02)
    return out


def sample_pixels(seed: int, npix: int, count: int, always: List[int] = ()) -> np.ndarray:
    """Seeded pixel subset (sorted, unique) for sampled parity at full sizes."""
    rng = np.random.default_rng(seed)
    count = min(count, npix)
    idx = rng.choice(npix, size=count, replace=False)
    return np.unique(np.concatenate([idx, np.asarray(list(always), dtype=np.int64)])).astype(np.int64)
