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


# ------------------------------------------------------------------------------------------------------------------
# Anisotropic pins of the voxel -> (theta, phi) / (latitude, longitude) mappings ("the North-South axis is
# along the z direction"; Eq. 10; RadialMap example).  An l = 0 shape or a constant map
# cannot tell z from x or atan2(y, x) from atan2(x, y); these can.
def _half_extents(g):
    """Number of inside voxels strictly beyond the centre voxel along +x, -x, +y, -y, +z, -z (odd dims, centre inside)."""
    occ = g[..., 0] > 0
    nz, ny, nx = occ.shape
    cz, cy, cx = nz // 2, ny // 2, nx // 2
    assert occ[cz, cy, cx]
    def run(line):
        n = 0
        for v in line:
            if not v:
                break
            n += 1
        return n
    return (run(occ[cz, cy, cx + 1:]), run(occ[cz, cy, cx - 1::-1]), run(occ[cz, cy + 1:, cx]), run(occ[cz, cy - 1::-1, cx]),
            run(occ[cz + 1:, cy, cx]), run(occ[cz - 1::-1, cy, cx]))


_SH_DIMS, _SH_VOX = (81, 81, 81), (1.0, 1.0, 1.0)
_R0, _S = 25.4, 6.2                           # R = R0 +- S along the dipole's axis: half extents 31 / 19, 25 elsewhere


def _dipole(m):
    c = _S / sqrt(3 / (4 * pi))
    return R.render({"kind": "spherical_harmonics", "delta": 1.0, "beta": 0.0,
                     "coeffs": [(0, 0, _R0 * sqrt(4 * pi)), (1, m, c)]}, _SH_DIMS, _SH_VOX)


def test_sh_l1_m0_dipole_points_along_plus_z():
    """Y_1^0 = sqrt(3/4pi) cos(theta), theta from body +z: R = R0 + S cos(theta) -> longer towards +z, shorter towards -z,
    R0 along x and y."""
    assert _half_extents(_dipole(0)) == (25, 25, 25, 25, 31, 19)


def test_sh_l1_m1_dipole_points_along_minus_x():
    """sqrt(2) Re Y_1^1 = -sqrt(3/4pi) sin(theta) cos(phi) (Condon-Shortley), phi from +x towards +y: for c > 0 the shape
    is longer towards -x, shorter towards +x, R0 along y and z."""
    assert _half_extents(_dipole(1)) == (19, 31, 25, 25, 25, 25)


def test_sh_l1_mneg1_dipole_points_along_minus_y():
    """sqrt(2) Im Y_1^1 = -sqrt(3/4pi) sin(theta) sin(phi): for c > 0 longer towards -y, shorter towards +y."""
    assert _half_extents(_dipole(-1)) == (25, 25, 19, 31, 25, 25)


def test_sh_l2_m2_distinguishes_x_from_y():
    """sqrt(2) Re Y_2^2 = sqrt(15/16pi) sin^2(theta) cos(2 phi): +S along +-x, -S along +-y, nothing along z."""
    c = _S / sqrt(15 / (16 * pi))
    g = R.render({"kind": "spherical_harmonics", "delta": 1.0, "beta": 0.0,
                  "coeffs": [(0, 0, _R0 * sqrt(4 * pi)), (2, 2, c)]}, _SH_DIMS, _SH_VOX)
    assert _half_extents(g) == (31, 31, 19, 19, 25, 25)


def _ray_count(g, d):
    """Inside voxels at centre + n d, n = 1, 2, ... (d an integer direction), until the first outside one."""
    occ = g[..., 0] > 0
    nz, ny, nx = occ.shape
    z, y, x = nz // 2, ny // 2, nx // 2
    n = 0
    while True:
        x, y, z = x + d[0], y + d[1], z + d[2]
        if not (0 <= x < nx and 0 <= y < ny and 0 <= z < nz) or not occ[z, y, x]:
            return n
        n += 1


def test_radial_map_raised_sample_sits_at_its_latitude_and_longitude():
    """in a 4 x 4 map the sample (i, j) = (3, 1) is the radius at latitude +pi/4, longitude pi/2, i.e. along
    (0, +1, +1)/sqrt(2): above the equator (z is the North-South axis), on the +y meridian."""
    radii = np.full((4, 4), 10.0)
    radii[3, 1] = 20.0
    g = R.render({"kind": "radial_map", "delta": 1.0, "beta": 0.0, "radii": radii}, (41, 41, 41), (1.0, 1.0, 1.0))
    assert _ray_count(g, (0, 1, 1)) == 14                  # n sqrt(2) <= 20
    for d in ((0, -1, 1), (0, 1, -1), (0, -1, -1), (1, 0, -1), (-1, 0, -1), (1, 1, 0), (-1, 1, 0)):
        assert _ray_count(g, d) == 7, d                    # n sqrt(2) <= 10: untouched directions
    # (1, 0, 1) and (-1, 0, 1) lie at latitude pi/4 a quarter turn of longitude from the bump: bilinear weight 0 there
    assert _ray_count(g, (1, 0, 1)) == 7 and _ray_count(g, (-1, 0, 1)) == 7
    # sample (1, 2): latitude -pi/4, longitude pi -> along (-1, 0, -1)/sqrt(2)
    radii = np.full((4, 4), 10.0)
    radii[1, 2] = 20.0
    g = R.render({"kind": "radial_map", "delta": 1.0, "beta": 0.0, "radii": radii}, (41, 41, 41), (1.0, 1.0, 1.0))
    assert _ray_count(g, (-1, 0, -1)) == 14
    for d in ((1, 0, -1), (-1, 0, 1), (0, -1, -1), (0, 1, -1), (1, 0, 1)):
        assert _ray_count(g, d) == 7, d


# ------------------------------------------------------------------------------------------------------------------
# The (latitude, longitude, rotation) helper of the input generators (workloads.quat_from_lat_long_rot, R11)
# against Fig. 6's caption and PAPER.md:281.
def test_lat_long_rot_helper_follows_fig6():
    from paper_2202_03411_b200 import workloads as W
    zb, xb = np.array([0.0, 0.0, 1.0]), np.array([1.0, 0.0, 0.0])
    M = lambda la, lo, ro: R.rotation_matrix(W.quat_from_lat_long_rot(la, lo, ro))
    # "90 deg latitude indicates a direction towards the incoming beam": the beam travels along +z, so the main axis
    # (body z) points to -z; "-90 deg latitude towards the detector": +z
    assert np.allclose(M(90, 0, 0) @ zb, [0, 0, -1], atol=1e-12)
    assert np.allclose(M(90, 123, 0) @ zb, [0, 0, -1], atol=1e-12)
    assert np.allclose(M(-90, 0, 0) @ zb, [0, 0, 1], atol=1e-12)
    # "the equator, at 0 deg latitude, lies on the plane orthogonal to the beam": longitude 0 -> +x, 90 -> +y
    assert np.allclose(M(0, 0, 0) @ zb, [1, 0, 0], atol=1e-12)
    assert np.allclose(M(0, 90, 0) @ zb, [0, 1, 0], atol=1e-12)
    assert np.allclose(M(0, 180, 0) @ zb, [-1, 0, 0], atol=1e-12)
    la, lo = np.radians(30.0), np.radians(40.0)
    assert np.allclose(M(30, 40, 0) @ zb, [np.cos(la) * np.cos(lo), np.cos(la) * np.sin(lo), -np.sin(la)], atol=1e-12)
    # "once the main axis is oriented, a rotation is applied to the sample along this axis": the main axis stays, a
    # body vector perpendicular to it turns by the rotation angle, right-handed about the main axis
    for (a, b) in ((0, 0), (30, 40), (-55, 200), (90, 0)):
        M0 = M(a, b, 0)
        axis = M0 @ zb
        for rot in (10.0, 90.0, 170.0):
            M1 = M(a, b, rot)
            assert np.allclose(M1 @ zb, axis, atol=1e-12)
            u0, u1 = M0 @ xb, M1 @ xb
            assert np.isclose(np.dot(u0, u1), np.cos(np.radians(rot)), atol=1e-12)
            assert np.isclose(np.dot(np.cross(u0, u1), axis), np.sin(np.radians(rot)), atol=1e-12)
            assert np.isclose(np.linalg.det(M1), 1.0, atol=1e-12)
    # every quaternion is unit (the boundary rejects others)
    assert np.isclose(np.linalg.norm(W.quat_from_lat_long_rot(12, 34, 56)), 1.0, atol=1e-15)


def test_lat_long_rot_helper_orients_a_rendered_shape():
    """An ellipsoid that is long along its main (body z) axis, rendered through the oracle with the helper's quaternion:
    latitude 90 -> long along the beam (grid z); latitude 0, longitude 0 -> long along grid x; longitude 90 -> grid y."""
    from paper_2202_03411_b200 import workloads as W
    shape = {"kind": "ellipsoid", "delta": 1.0, "beta": 0.0, "a": 5.3, "b": 8.3, "c": 14.3}
    dims, vox = (41, 41, 41), (1.0, 1.0, 1.0)
    ext = lambda la, lo, ro: _half_extents(R.render({**shape, "quat": W.quat_from_lat_long_rot(la, lo, ro)}, dims, vox))
    assert ext(90, 0, 0)[4:] == (14, 14)
    assert ext(0, 0, 0)[:2] == (14, 14)
    assert ext(0, 90, 0)[2:4] == (14, 14)
    # rotation about the main axis exchanges the two short axes after a quarter turn
    e0, e1 = ext(90, 0, 0), ext(90, 0, 90)
    assert sorted((e0[0], e0[2])) == [5, 8] and (e1[0], e1[2]) == (e0[2], e0[0])
