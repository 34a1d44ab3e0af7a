"""Pins of the shape-rendering oracle (oracle/render.py) against what the paper and the mathematics fix: library
spherical harmonics, closed forms, orthonormality, the paper's worked RadialMap / VolumeMap examples, volumes, and the
orientation convention already pinned for a0.  CPU only."""
from math import pi, sqrt

import numpy as np
import pytest

from oracle import oracle as O
from oracle import render as R


def _scipy_ylm(l, m, theta, phi):
    import scipy.special as sp
    if hasattr(sp, "sph_harm_y"):
        return sp.sph_harm_y(l, m, theta, phi)          # (degree, order, polar, azimuth)
    return sp.sph_harm(m, l, phi, theta)                 # older scipy: (order, degree, azimuth, polar)


def test_real_harmonics_match_library_complex_harmonics():
    """Eq. 10: m = 0 -> Y_l^0; m > 0 -> sqrt(2) Re Y_l^m; m < 0 -> sqrt(2) Im Y_l^|m| (scipy, Condon-Shortley)."""
    rng = np.random.default_rng(1)
    theta = rng.uniform(0, pi, 200)
    phi = rng.uniform(-pi, pi, 200)
    for l in range(0, 9):
        for m in range(-l, l + 1):
            got = R.real_sph_harm(l, m, np.cos(theta), phi)
            y = _scipy_ylm(l, abs(m), theta, phi)
            ref = y.real if m == 0 else (sqrt(2) * y.real if m > 0 else sqrt(2) * y.imag)
            assert np.allclose(got, ref, rtol=1e-11, atol=1e-12), (l, m)


def test_harmonics_closed_forms():
    th = np.linspace(0.05, 3.0, 17)
    ph = np.linspace(-3.0, 3.0, 17)
    ct, st = np.cos(th), np.sin(th)
    assert np.allclose(R.real_sph_harm(0, 0, ct, ph), 1 / sqrt(4 * pi))
    assert np.allclose(R.real_sph_harm(1, 0, ct, ph), sqrt(3 / (4 * pi)) * ct)
    assert np.allclose(R.real_sph_harm(1, 1, ct, ph), -sqrt(3 / (4 * pi)) * st * np.cos(ph))
    assert np.allclose(R.real_sph_harm(1, -1, ct, ph), -sqrt(3 / (4 * pi)) * st * np.sin(ph))
    assert np.allclose(R.real_sph_harm(2, 0, ct, ph), sqrt(5 / (16 * pi)) * (3 * ct ** 2 - 1))
    assert np.allclose(R.real_sph_harm(2, 2, ct, ph), sqrt(15 / (16 * pi)) * st ** 2 * np.cos(2 * ph))


def test_harmonics_are_orthonormal():
    x, w = np.polynomial.legendre.leggauss(48)
    nphi = 96
    ph = (np.arange(nphi) + 0.5) * 2 * pi / nphi - pi
    X, P = np.meshgrid(x, ph, indexing="ij")
    W = w[:, None] * (2 * pi / nphi)
    lm = [(l, m) for l in range(0, 6) for m in range(-l, l + 1)]
    Y = np.stack([R.real_sph_harm(l, m, X, P) for l, m in lm])
    G = np.einsum("aij,bij,ij->ab", Y, Y, W * np.ones_like(X))
    assert np.allclose(G, np.eye(len(lm)), atol=1e-10)


def test_sphere_from_l0_triplet_equals_ellipsoid_sphere():
    dims, voxel, rad = (33, 31, 29), (2.0, 2.0, 2.0), 21.3
    a = R.render({"kind": "spherical_harmonics", "delta": 0.02, "beta": 0.003, "coeffs": [(0, 0, rad * sqrt(4 * pi))]}, dims, voxel)
    b = R.render({"kind": "ellipsoid", "delta": 0.02, "beta": 0.003, "a": rad, "b": rad, "c": rad}, dims, voxel)
    assert np.array_equal(a, b)
    assert a[..., 0].max() == np.float32(0.02) and a[..., 1].max() == np.float32(0.003)


def test_ellipsoid_volume_and_axes():
    dims, voxel = (96, 96, 96), (1.0, 1.0, 1.0)
    a, b, c = 40.0, 27.0, 18.0
    g = R.render({"kind": "ellipsoid", "delta": 1.0, "beta": 0.0, "a": a, "b": b, "c": c}, dims, voxel)
    vol = float(g[..., 0].sum())
    assert abs(vol - 4 / 3 * pi * a * b * c) / (4 / 3 * pi * a * b * c) < 5e-3
    ext = [np.nonzero(g[..., 0].any(axis=ax))[0] for ax in ((0, 1), (0, 2), (1, 2))]   # extents along x, y, z
    assert [int(e.max() - e.min() + 1) for e in ext] == [80, 54, 36]


def test_orientation_convention_matches_a0_on_quarter_turns():
    """Rendering with a quaternion == a0's (already pinned) resampling of the unrotated rendering, exact for quarter turns."""
    dims, voxel = (24, 24, 24), (1.5, 1.5, 1.5)
    shape = {"kind": "ellipsoid", "delta": 0.03, "beta": 0.01, "a": 15.0, "b": 9.0, "c": 5.0}
    base = R.render(shape, dims, voxel)
    s = sqrt(0.5)
    for quat in ([s, s, 0, 0], [s, 0, s, 0], [s, 0, 0, s], [0.5, 0.5, 0.5, 0.5]):
        got = R.render({**shape, "quat": quat}, dims, voxel)
        ref = O.orient(base, voxel, np.array(quat, dtype=np.float64))
        assert np.allclose(got, ref, rtol=0, atol=1e-9), quat   # sqrt(1/2) quaternions give matrix entries of 1e-16, not 0
    # 90 degrees about x maps body z to beam -y... in any case an ellipsoid with b and c exchanged
    got = R.render({**shape, "quat": [s, s, 0, 0]}, dims, voxel)
    swapped = R.render({**shape, "b": 5.0, "c": 9.0}, dims, voxel)
    assert np.array_equal(got, swapped)


def _golden(name):
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", name)
    return [ln.split() for ln in open(path) if ln.strip() and not ln.startswith("#")]


def test_radial_map_paper_example_sample_positions():
    """PAPER.md:419 (tests/golden/radial_map_example.txt): a 4 x 4 array gives the radii at theta = -pi/2, -pi/4, 0, pi/4 and
    phi = 0, pi/2, pi, 3pi/2."""
    rng = np.random.default_rng(4)
    radii = rng.uniform(5.0, 9.0, (4, 4))
    rows = {r[0]: r for r in _golden("radial_map_example.txt")}
    assert int(rows["theta"][1]) == 4 and int(rows["phi"][1]) == 4
    lats = np.array([float(v) for v in rows["theta"][2:]]) * pi
    lons = np.array([float(v) for v in rows["phi"][2:]]) * pi
    L, M = np.meshgrid(lats, lons, indexing="ij")
    assert np.allclose(R.radial_map_radius(radii, L, M), radii, rtol=0, atol=1e-14)
    # linear in between, periodic in longitude, held above the last latitude sample
    assert np.isclose(R.radial_map_radius(radii, np.array(-3 * pi / 8), np.array(0.0)), 0.5 * (radii[0, 0] + radii[1, 0]))
    assert np.isclose(R.radial_map_radius(radii, np.array(0.0), np.array(7 * pi / 4)), 0.5 * (radii[2, 3] + radii[2, 0]))
    assert np.isclose(R.radial_map_radius(radii, np.array(0.45 * pi), np.array(pi)), radii[3, 2])
    assert np.isclose(R.radial_map_radius(radii, np.array(-pi / 8), np.array(pi / 4)),
                      0.25 * (radii[1, 0] + radii[1, 1] + radii[2, 0] + radii[2, 1]))


def test_radial_map_constant_is_a_sphere_and_analytic_profile():
    dims, voxel = (40, 40, 40), (1.0, 1.0, 1.0)
    const = R.render({"kind": "radial_map", "delta": 0.01, "beta": 0.0, "radii": np.full((7, 12), 14.2)}, dims, voxel)
    sph = R.render({"kind": "ellipsoid", "delta": 0.01, "beta": 0.0, "a": 14.2, "b": 14.2, "c": 14.2}, dims, voxel)
    assert np.array_equal(const, sph)
    # a radius that is linear in latitude is reproduced exactly by linear interpolation (below the last sample row)
    nlat, nlon = 64, 8
    lat_s = -pi / 2 + np.arange(nlat) * pi / nlat
    radii = np.repeat((10.0 + 2.0 * lat_s)[:, None], nlon, axis=1)
    lat = np.linspace(-1.5, 1.4, 50)
    assert np.allclose(R.radial_map_radius(radii, lat, np.full_like(lat, 1.0)), 10.0 + 2.0 * lat, atol=1e-12)


def test_volume_map_paper_example_cube():
    """PAPER.md:423 (tests/golden/volume_map_example.txt): a 10^3 all-True array with dx = 2 is a 20 x 20 x 20 cube; dx = 4 doubles it."""
    cases = [(int(r[0]), float(r[1]), float(r[2])) for r in _golden("volume_map_example.txt")]
    assert cases == [(10, 2.0, 20.0), (10, 4.0, 40.0)]
    vol = np.ones((10, 10, 10), dtype=bool)
    for (cells, dx, side_nm), n in zip(cases, (32, 48)):
        side = int(side_nm)                     # rendered on 1 nm voxels
        g = R.render({"kind": "volume_map", "delta": 1.0, "beta": 0.5, "volume": vol, "dx": dx}, (n, n, n), (1.0, 1.0, 1.0))
        assert int(g[..., 0].sum()) == side ** 3
        idx = np.nonzero(g[..., 0])
        assert all(int(i.max() - i.min() + 1) == side for i in idx)
        assert np.all(g[..., 1][g[..., 0] > 0] == np.float32(0.5))


def test_volume_map_cells_and_layout():
    vol = np.zeros((2, 3, 4), dtype=bool)      # [z][y][x]
    vol[1, 2, 3] = True                        # the cell at the +x +y +z corner
    g = R.render({"kind": "volume_map", "delta": 1.0, "beta": 0.0, "volume": vol, "dx": 2.0}, (8, 6, 4), (1.0, 1.0, 1.0))
    want = np.zeros((4, 6, 8), dtype=bool)
    want[2:4, 4:6, 6:8] = True
    assert np.array_equal(g[..., 0] > 0, want)
