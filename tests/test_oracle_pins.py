"""Pins of the FP64 oracle against things other than itself.

Each pin is chosen so that a plausible slip in oracle/msft_oracle.c (dropped term, wrong sign or
index, transposed axis, inclusive instead of exclusive prefix, missing dV) fails at least one.
"""
import numpy as np
import pytest

from oracle import oracle as O
from oracle.eq9_literal import eq9_field
from paper_2202_03411_b200 import workloads as W


def centres(n, d):
    return (np.arange(n) - (n - 1) / 2.0) * d


def rand_q(rng, n, k):
    """Random Ewald-sphere q's (north_star sign: q = k(s - z^)) up to ~50 degrees."""
    th = rng.uniform(0.0, np.deg2rad(50.0), n)
    ph = rng.uniform(-np.pi, np.pi, n)
    return np.stack([k * np.sin(th) * np.cos(ph), k * np.sin(th) * np.sin(ph), k * (np.cos(th) - 1.0)], axis=1)


# --------------------------------------------------------------------------------------- P1
def test_p1_tables_equal_direct_tiny():
    rng = np.random.default_rng(1)
    dn = W.random_grid(11, 5, 6, 7)
    voxel, lam = (3.0, 2.5, 2.0), 17.0
    q = rand_q(rng, 40, 2 * np.pi / lam)
    for mode in (O.RHO_LINEAR, O.RHO_N2M1):
        I1, A1 = O.simulate_q(dn, voxel, lam, q, rho_mode=mode, method="direct", return_amplitude=True)
        I2, A2 = O.simulate_q(dn, voxel, lam, q, rho_mode=mode, method="tables", return_amplitude=True)
        assert np.max(np.abs(A1 - A2)) <= 1e-12 * np.max(np.abs(A1))
        assert np.allclose(I1, I2, rtol=1e-11, atol=0)


def test_p1_brute_force_numpy_3d_sum():
    """Independent numpy brute force: the 3-D sum of Eq. 1 with the attenuation written as a cumsum."""
    rng = np.random.default_rng(2)
    nx, ny, nz = 4, 3, 5
    dn = W.random_grid(12, nx, ny, nz, fill=0.8)
    voxel, lam = (1.5, 2.0, 2.5), 11.0
    k = 2 * np.pi / lam
    q = rand_q(rng, 9, k)
    c = dn[..., 0].astype(np.float64) + 1j * dn[..., 1].astype(np.float64)
    Cex = np.cumsum(c, axis=0) - c                          # exclusive prefix along z
    rho = c * np.exp(1j * k * voxel[2] * Cex) * np.prod(voxel)
    Z, Y, X = np.meshgrid(centres(nz, voxel[2]), centres(ny, voxel[1]), centres(nx, voxel[0]), indexing="ij")
    A = np.array([np.sum(rho * np.exp(1j * (qq[0] * X + qq[1] * Y + qq[2] * Z))) for qq in q])
    I, Ao = O.simulate_q(dn, voxel, lam, q, return_amplitude=True)
    assert np.max(np.abs(Ao - A)) <= 1e-12 * np.max(np.abs(A))
    assert np.allclose(I, np.abs(A) ** 2, rtol=1e-11)


# --------------------------------------------------------------------------------------- P2
def geom(q, x0, d, n):
    r = np.exp(1j * q * d)
    return np.exp(1j * q * x0) * (1 - r ** n) / (1 - r)


@pytest.mark.parametrize("mode", [O.RHO_LINEAR, O.RHO_N2M1])
def test_p2_homogeneous_absorbing_cuboid_closed_form(mode):
    """Homogeneous block: A = f(c) dV S_x S_y S_z with geometric sums; S_z carries k c dz per slice."""
    rng = np.random.default_rng(3)
    nx, ny, nz = 9, 7, 11
    bx, by, bz = (2, 7), (1, 5), (3, 10)          # block index ranges [lo, hi)
    delta, beta = np.float32(0.031), np.float32(0.012)
    dn = np.zeros((nz, ny, nx, 2), np.float32)
    dn[bz[0]:bz[1], by[0]:by[1], bx[0]:bx[1]] = (delta, beta)
    voxel, lam = (2.0, 3.0, 1.5), 9.0
    k = 2 * np.pi / lam
    q = rand_q(rng, 25, k)
    c = float(delta) + 1j * float(beta)
    f = c if mode == O.RHO_LINEAR else c * (2 - c)
    x = centres(nx, voxel[0]); y = centres(ny, voxel[1]); z = centres(nz, voxel[2])
    Sx = geom(q[:, 0], x[bx[0]], voxel[0], bx[1] - bx[0])
    Sy = geom(q[:, 1], y[by[0]], voxel[1], by[1] - by[0])
    # slice m of the block (m = 0..): phase e^{i qz z_m} * e^{i k dz c m}
    rz = np.exp(1j * (q[:, 2] + k * c) * voxel[2])
    Sz = np.exp(1j * q[:, 2] * z[bz[0]]) * (1 - rz ** (bz[1] - bz[0])) / (1 - rz)
    A = f * np.prod(voxel) * Sx * Sy * Sz
    I, Ao = O.simulate_q(dn, voxel, lam, q, rho_mode=mode, return_amplitude=True)
    assert np.max(np.abs(Ao - A)) <= 1e-12 * np.max(np.abs(A))
    assert np.allclose(I, np.abs(A) ** 2, rtol=1e-11)


# --------------------------------------------------------------------------------------- P3
def test_p3_forward_pixel_and_born_limit():
    dn = W.random_grid(13, 6, 5, 8)
    voxel, lam = (2.0, 2.0, 2.0), 15.0
    k = 2 * np.pi / lam
    q0 = np.zeros((1, 3))
    c = dn[..., 0].astype(np.float64) + 1j * dn[..., 1].astype(np.float64)
    Cex = np.cumsum(c, axis=0) - c
    exact = np.sum(c * np.exp(1j * k * voxel[2] * Cex)) * 8.0
    I, A = O.simulate_q(dn, voxel, lam, q0, return_amplitude=True)
    assert abs(A[0] - exact) <= 1e-13 * abs(exact)
    # Born limit: tiny contrast -> I(0) = |sum dn dV|^2   (north_star)
    weak = (dn * np.float32(1e-6)).astype(np.float32)
    Iw = O.simulate_q(weak, voxel, lam, q0)
    born = abs(np.sum(weak[..., 0].astype(np.float64) + 1j * weak[..., 1].astype(np.float64)) * 8.0) ** 2
    assert abs(Iw[0] - born) <= 1e-5 * born


# --------------------------------------------------------------------------------------- P4
def test_p4_born_sphere_form_factor():
    """Non-absorbing weak sphere: I = |delta V 3(sin u - u cos u)/u^3|^2, u = |q| R (north_star)."""
    n, d, R = 64, 1.0, 26.0
    lam = 8.0
    delta = np.float32(1e-6)
    mask = W.ellipsoid_mask(n, n, n, d, d, d, R, R, R)
    dn = np.zeros((n, n, n, 2), np.float32)
    dn[mask, 0] = delta
    Vvox = mask.sum() * d ** 3
    npx = 24
    q = O.qmap(npx, npx, 12.0, lam)
    I = O.simulate_q(dn, (d, d, d), lam, q)
    u = np.linalg.norm(q, axis=1) * R
    ff = 3 * (np.sin(u) - u * np.cos(u)) / u ** 3
    ref = (float(delta) * Vvox * ff) ** 2
    rel_l2 = np.sqrt(np.sum((I - ref) ** 2) / np.sum(ref ** 2))
    assert rel_l2 < 5e-3, rel_l2          # voxelisation-limited
    # |q| = 2 k sin(theta/2) on the Ewald sphere (Eq. 3)
    k = 2 * np.pi / lam
    uu = (np.arange(npx) + 0.5 - npx / 2) * 2 * np.tan(np.deg2rad(12.0)) / npx
    U, V = np.meshgrid(uu, uu)
    theta = np.arctan(np.sqrt(U ** 2 + V ** 2)).ravel()
    assert np.allclose(np.linalg.norm(q, axis=1), 2 * k * np.sin(theta / 2), rtol=1e-12)


def test_qmap_geometry():
    """Outer edge mid-points at theta_max; q = k(s - z^) with |s| = 1; qz <= 0; ix fastest."""
    npx, npy, th, lam = 10, 6, 35.0, 7.0
    k = 2 * np.pi / lam
    q = O.qmap(npx, npy, th, lam).reshape(npy, npx, 3)
    s = q / k + np.array([0, 0, 1.0])
    assert np.allclose(np.linalg.norm(s, axis=-1), 1.0, atol=1e-14)
    assert np.all(q[..., 2] <= 0)
    pitch = 2 * np.tan(np.deg2rad(th)) / npx
    # tan of the angle in x of the last pixel's outer edge = theta_max: centre + pitch/2
    u_last = s[0, -1, 0] / s[0, -1, 2]
    assert np.isclose(u_last + pitch / 2, np.tan(np.deg2rad(th)), rtol=1e-13)
    assert np.allclose(q[:, ::-1, 0], -q[:, :, 0], atol=1e-15) and np.allclose(q[::-1, :, 1], -q[:, :, 1], atol=1e-15)
    assert q[0, 1, 0] > q[0, 0, 0] and np.isclose(q[0, 1, 1], q[0, 0, 1], rtol=0.2)   # ix is the fast index
    # detector-centre offset shifts by whole pixels
    q2 = O.qmap(npx, npy, th, lam, cx=1.0, cy=-2.0).reshape(npy, npx, 3)
    assert np.allclose(q2[2:, :-1], q[:-2, 1:], atol=1e-14)


# --------------------------------------------------------------------------------------- P5
def test_p5_d4_symmetry_of_sphere_pattern():
    w = W.config(0)
    I = O.simulate(w.grid(0), (w.dx, w.dy, w.dz), w.lam, 16, 16, w.theta_max_deg)
    assert np.allclose(I, I[:, ::-1], rtol=1e-11)
    assert np.allclose(I, I[::-1, :], rtol=1e-11)
    assert np.allclose(I, I.T, rtol=1e-11)


# --------------------------------------------------------------------------------------- P6
def test_p6_translation_invariance():
    rng = np.random.default_rng(6)
    core = W.random_grid(16, 4, 4, 4, fill=0.9)
    voxel, lam = (2.0, 2.0, 2.0), 12.0
    q = rand_q(rng, 20, 2 * np.pi / lam)

    def place(ox, oy, oz):
        g = np.zeros((9, 9, 9, 2), np.float32)
        g[oz:oz + 4, oy:oy + 4, ox:ox + 4] = core
        return g
    I0 = O.simulate_q(place(1, 1, 1), voxel, lam, q)
    for off in [(4, 1, 1), (1, 5, 1), (1, 1, 3), (3, 2, 5)]:
        assert np.allclose(O.simulate_q(place(*off), voxel, lam, q), I0, rtol=1e-10)


# --------------------------------------------------------------------------------------- P7
@pytest.mark.parametrize("mode,strength", [(O.RHO_N2M1, "n2-1"), (O.RHO_LINEAR, "n-1")])
def test_p7_literal_eq9_is_conjugate(mode, strength):
    """Paper's loop with the paper's signs: A_northstar = -conj(Psi_paper) e^{i qz z_0}; same I."""
    rng = np.random.default_rng(7)
    nx, ny, nz = 5, 6, 7
    dn = W.random_grid(17, nx, ny, nz)
    voxel, lam = (2.0, 1.5, 1.0), 9.0
    q = rand_q(rng, 30, 2 * np.pi / lam)
    psi = eq9_field(dn, voxel, lam, -q, strength=strength)
    I, A = O.simulate_q(dn, voxel, lam, q, rho_mode=mode, return_amplitude=True)
    z0 = -(nz - 1) / 2.0 * voxel[2]
    assert np.max(np.abs(A - (-np.conj(psi)) * np.exp(1j * q[:, 2] * z0))) <= 1e-12 * np.max(np.abs(A))
    assert np.allclose(I, np.abs(psi) ** 2, rtol=1e-11)


# --------------------------------------------------------------------------------------- P8
def test_p8_single_slice_matches_numpy_fft2():
    nx, ny = 8, 6
    dn = W.random_grid(18, nx, ny, 1, fill=1.0)
    dx, dy, dz = 1.7, 2.3, 1.0
    lam = 10.0
    rho = (dn[0, :, :, 0].astype(np.float64) + 1j * dn[0, :, :, 1].astype(np.float64)) * dx * dy * dz
    Fk = np.fft.fft2(rho)                                    # sum rho e^{-2 pi i (my iy/ny + mx ix/nx)}
    my, mx = np.meshgrid(np.arange(ny), np.arange(nx), indexing="ij")
    qx = -2 * np.pi * mx / (nx * dx)
    qy = -2 * np.pi * my / (ny * dy)
    q = np.stack([qx.ravel(), qy.ravel(), np.zeros(nx * ny)], axis=1)
    _, A = O.simulate_q(dn, (dx, dy, dz), lam, q, return_amplitude=True)
    # oracle uses centred coordinates: x_i = (i - (nx-1)/2) dx -> extra phase e^{i q x_0}
    shift = np.exp(1j * (qx * (-(nx - 1) / 2 * dx) + qy * (-(ny - 1) / 2 * dy))).ravel()
    assert np.max(np.abs(A - Fk.ravel() * shift)) <= 1e-12 * np.max(np.abs(Fk))


# --------------------------------------------------------------------------------------- P9
def test_p9_one_and_two_voxels():
    rng = np.random.default_rng(9)
    voxel, lam = (2.0, 2.0, 3.0), 14.0
    k = 2 * np.pi / lam
    q = rand_q(rng, 15, k)
    dV = 12.0
    g = np.zeros((5, 5, 5, 2), np.float32)
    g[1, 3, 2] = (0.02, 0.004)
    c1 = float(np.float32(0.02)) + 1j * float(np.float32(0.004))
    assert np.allclose(O.simulate_q(g, voxel, lam, q), abs(c1 * dV) ** 2, rtol=1e-12)
    # second voxel two slices further down the same column: attenuated by the first only (exclusive prefix)
    g[3, 3, 2] = (0.05, 0.01)
    c2 = float(np.float32(0.05)) + 1j * float(np.float32(0.01))
    A = dV * (c1 + c2 * np.exp(1j * k * voxel[2] * c1) * np.exp(1j * q[:, 2] * 2 * voxel[2]))
    assert np.allclose(O.simulate_q(g, voxel, lam, q), np.abs(A) ** 2, rtol=1e-11)
    # a voxel in a different column is NOT attenuated
    h = np.zeros((5, 5, 5, 2), np.float32)
    h[1, 3, 2] = (0.02, 0.004)
    h[3, 3, 4] = (0.05, 0.01)
    A = dV * (c1 + c2 * np.exp(1j * (q[:, 2] * 2 * voxel[2] + q[:, 0] * 2 * voxel[0])))
    assert np.allclose(O.simulate_q(h, voxel, lam, q), np.abs(A) ** 2, rtol=1e-11)


# --------------------------------------------------------------------------------------- P10
def test_p10_n2m1_vs_linear_homogeneous():
    w = W.config(0)
    g = w.grid(0)
    c = float(np.float32(0.01)) + 1j * float(np.float32(0.001))
    args = ((w.dx, w.dy, w.dz), w.lam, 8, 8, w.theta_max_deg)
    Il = O.simulate(g, *args, rho_mode=O.RHO_LINEAR)
    In = O.simulate(g, *args, rho_mode=O.RHO_N2M1)
    assert np.allclose(In, abs(2 - c) ** 2 * Il, rtol=1e-11)


# --------------------------------------------------------------------------------------- P11
def test_p11_orientation_quarter_turns_and_point_reflection():
    n = 7
    g = W.random_grid(21, n, n, n)
    voxel = (2.0, 2.0, 2.0)
    s = np.sqrt(0.5)
    # +90 deg about z (beam): r_beam = Rz r_body -> out[z, y, x] = in[z, -x, y] in centred index terms
    out = O.orient(g, voxel, [s, 0, 0, s])
    exp = np.zeros_like(g)
    for iy in range(n):
        for ix in range(n):
            # r_body = Rz^T r_beam: (xo, yo) = (y, -x)
            exp[:, iy, ix] = g[:, (n - 1) - ix, iy]
    assert np.allclose(out, exp, rtol=1e-6, atol=1e-12)      # sqrt(1/2) is inexact: weights are 1 - O(1e-16)
    # +90 deg about x: r_body = Rx^T r_beam: (yo, zo) = (z, -y)
    out = O.orient(g, voxel, [s, s, 0, 0])
    exp = np.zeros_like(g)
    for iz in range(n):
        for iy in range(n):
            exp[iz, iy, :] = g[(n - 1) - iy, iz, :]
    assert np.allclose(out, exp, rtol=1e-6, atol=1e-12)
    # identity quaternion reproduces the grid
    assert np.array_equal(O.orient(g, voxel, [1, 0, 0, 0]), g)
    # 180 deg about the beam axis point-reflects the pattern
    lam = 11.0
    I0 = O.simulate(g, voxel, lam, 6, 6, 30.0)
    I180 = O.simulate(g, voxel, lam, 6, 6, 30.0, quat=[0, 0, 0, 1])
    assert np.allclose(I180, I0[::-1, ::-1], rtol=1e-10)


def test_p11_half_voxel_trilinear_weights():
    """A non-lattice case: rotating by 0 but checking weights via a 2-voxel average is not
    reachable through a pure rotation, so check a 45-degree turn about z at the centre voxel
    column and the zero-outside rule with hand-computed trilinear weights."""
    n = 5
    g = np.zeros((n, n, n, 2), np.float32)
    g[:, 2, 3] = (1.0, 0.5)          # column at body (x=+1, y=0)
    a = np.deg2rad(45.0)
    out = O.orient(g, (1.0, 1.0, 1.0), [np.cos(a / 2), 0, 0, np.sin(a / 2)])
    # beam voxel (x=+1, y=+1) maps to body R^T r = (sqrt2, 0): between x=+1 (w=2-sqrt2) and x=+2 (empty)
    wgt = 2 - np.sqrt(2.0)
    assert np.allclose(out[:, 3, 3, 0], np.float32(wgt)) and np.allclose(out[:, 3, 3, 1], np.float32(0.5 * wgt))
    # beam voxel (x=+2, y=+2) maps to body (2 sqrt2, 0): outside the grid (x index 4.83 -> neighbour 5 is out, 4 is empty)
    assert np.all(out[:, 4, 4] == 0)


# ------------------------------------------------------------------------------------------ tensor-grid detector
def test_qgrid_points_lie_on_the_ewald_sphere_and_match_the_flat_detector():
    """qgrid_q: |q + k z^| = k for every propagating point (Eq. 3-4); fed the (qx, qy) of a flat-detector pixel it returns that
    pixel's qz (the q-map is pinned by geometry above); forward point qz = 0; |q_xy| = k is 90 degrees: qz = -k."""
    lam = 13.0
    k = 2 * np.pi / lam
    qx = np.linspace(-0.9 * k, 1.1 * k, 23)
    qy = np.linspace(-0.5 * k, 0.7 * k, 17)
    q, ok = O.qgrid_q(qx, qy, lam)
    assert q.shape == (17 * 23, 3) and np.array_equal(q[:23, 0], qx) and np.all(q[:23, 1] == qy[0])
    r = np.sqrt(q[:, 0] ** 2 + q[:, 1] ** 2 + (q[:, 2] + k) ** 2)
    assert np.allclose(r[ok], k, rtol=1e-13)
    assert np.array_equal(ok, (q[:, 0] ** 2 + q[:, 1] ** 2) <= k * k) and not ok.all() and np.all(q[~ok, 2] == 0)
    qm = O.qmap(9, 7, 50.0, lam, 0.3, -0.2)
    for p in range(0, 63, 5):
        qq, okp = O.qgrid_q([qm[p, 0]], [qm[p, 1]], lam)
        assert okp[0] and np.isclose(qq[0, 2], qm[p, 2], rtol=1e-12, atol=1e-15)
    q0, _ = O.qgrid_q([0.0, k], [0.0], lam)
    assert q0[0, 2] == 0.0 and np.isclose(q0[1, 2], -k)


def test_qgrid_single_slice_on_the_dft_grid_is_numpy_fft2():
    """One slice, q on the DFT grid: the whole tensor-grid pattern equals |dV fft2(rho)|^2 (library routine), and qz drops out."""
    rng = np.random.default_rng(21)
    nx, ny, d = 12, 10, 1.5
    g = np.zeros((1, ny, nx, 2), np.float32)
    g[0, ..., 0] = rng.uniform(-0.02, 0.05, (ny, nx))
    g[0, ..., 1] = rng.uniform(0.0, 0.02, (ny, nx))
    lam = 2.0                                   # k = 3.14 > max |q_xy| = 2.96 so that every point propagates
    mx, my = np.arange(nx), np.arange(ny)
    qx = -2 * np.pi * np.where(mx < nx / 2, mx, mx - nx) / (nx * d)     # e^{i q x} = e^{-2 pi i m n / N}
    qy = -2 * np.pi * np.where(my < ny / 2, my, my - ny) / (ny * d)
    I = O.simulate_qgrid(g, (d, d, 2.0), lam, qx, qy)
    rho = g[0, ..., 0].astype(np.float64) + 1j * g[0, ..., 1].astype(np.float64)
    ref = np.abs(np.fft.fft2(rho) * d * d * 2.0) ** 2
    assert np.allclose(I, ref, rtol=1e-11)


def test_oracle_matches_its_stored_values():
    """tests/golden/cfg1_oracle_pixels.txt (written by tests/golden/make_golden.py, which calls only oracle/): the oracle as it
    stands reproduces its stored intensities on config 1; an unintended change of its arithmetic fails here."""
    import os
    from paper_2202_03411_b200 import workloads as W
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "cfg1_oracle_pixels.txt")
    rows = [ln.split() for ln in open(path) if ln.strip() and not ln.startswith("#")]
    pix = np.array([int(r[0]) for r in rows], dtype=np.int64)
    want = np.array([float(r[1]) for r in rows])
    w = W.config(0)
    got = O.simulate(w.grid(0), (w.dx, w.dy, w.dz), w.lam, w.npx, w.npy, w.theta_max_deg, pixels=pix)
    assert np.allclose(got, want, rtol=1e-12, atol=0)
