"""GPU parity of shape rendering (scatman_render, render_kernels.cu) against oracle/render.py, voxel by voxel, and of
the rendered-then-simulated path against the oracle's."""
from math import pi, sqrt

import numpy as np
import pytest

from oracle import oracle as O
from oracle import render as R
from paper_2202_03411_b200 import workloads as W
from parity import assert_parity

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


def _to_device(shape):
    import torch
    d = dict(shape)
    if "radii" in d:
        d["radii"] = torch.from_numpy(np.ascontiguousarray(d["radii"], dtype=np.float64)).cuda()
    if "volume" in d:
        d["volume"] = torch.from_numpy(np.ascontiguousarray(d["volume"]).astype(np.uint8)).cuda()
    return d


def _check(sm, shapes, dims, voxel, tie=1e-9):
    """Byte-exact (delta, beta) everywhere, except voxels whose centre lies on the surface to within rounding: there the
    inside test is an FP64 comparison of two nearly equal numbers and either answer is valid."""
    got = sm.render([_to_device(s) for s in shapes], dims, voxel).cpu().numpy()
    for b, s in enumerate(shapes):
        ref, margin = R.render(s, dims, voxel, return_margin=True)
        diff = np.any(got[b] != ref, axis=-1)
        if diff.any():
            scale = 100.0 if s["kind"] in ("spherical_harmonics", "radial_map") else 1.0   # margin is a length there
            assert np.all(np.abs(margin[diff]) <= tie * scale), (b, s["kind"], int(diff.sum()), float(np.abs(margin[diff]).max()))
            assert diff.sum() <= 1e-5 * diff.size + 2
        vals = got[b][np.any(got[b] != 0, axis=-1)]
        if vals.size:
            assert np.all(vals[:, 0] == np.float32(s["delta"])) and np.all(vals[:, 1] == np.float32(s["beta"]))
    return got


def _droplet_coeffs(rng, r0, lmax, sigma0=0.05):
    co = [(0, 0, r0 * sqrt(4 * pi))]
    for l in range(1, lmax + 1):
        for m in range(-l, l + 1):
            co.append((l, m, r0 * rng.normal(0.0, sigma0 / l)))
    return co


def test_ellipsoids_ragged_dims_random_orientations(sm):
    rng = np.random.default_rng(11)
    quats = W.random_quaternions(rng, 4)
    shapes = [{"kind": "ellipsoid", "delta": 0.02 + 0.01 * i, "beta": 0.005 * i, "quat": quats[i],
               "a": 30.0 - 3 * i, "b": 17.5 + i, "c": 9.25 + 2 * i} for i in range(4)]
    shapes.append({"kind": "ellipsoid", "delta": -0.01, "beta": 0.0, "a": 500.0, "b": 500.0, "c": 500.0})   # fills the grid
    shapes.append({"kind": "ellipsoid", "delta": 0.01, "beta": 0.0, "a": 0.1, "b": 0.1, "c": 0.1})          # holds only the centre voxel (odd dims)
    got = _check(sm, shapes, (45, 37, 29), (1.7, 2.1, 1.3))
    assert np.all(got[4][..., 0] == np.float32(-0.01))
    assert int(np.count_nonzero(got[5][..., 0])) == 1 and got[5][14, 18, 22, 0] == np.float32(0.01)


def test_spherical_harmonics_droplets(sm):
    rng = np.random.default_rng(12)
    quats = W.random_quaternions(rng, 3)
    shapes = [{"kind": "spherical_harmonics", "delta": 0.03, "beta": 0.01, "coeffs": _droplet_coeffs(rng, 40.0, 6)},
              {"kind": "spherical_harmonics", "delta": 0.03, "beta": 0.01, "quat": quats[0], "coeffs": _droplet_coeffs(rng, 25.0, 4, 0.15)},
              {"kind": "spherical_harmonics", "delta": 0.01, "beta": 0.0, "quat": quats[1],
               "coeffs": [(0, 0, 100.0), (8, 5, 30.0), (8, -8, 25.0), (3, -2, 20.0), (5, 0, -15.0)]},
              {"kind": "spherical_harmonics", "delta": 0.01, "beta": 0.0, "quat": quats[2], "coeffs": [(0, 0, 33.0 * sqrt(4 * pi))]},
              # degrees above 8 take the triplet walker, 5 and 7 the dense tables of the next even degree; a repeated (l, m) adds up
              {"kind": "spherical_harmonics", "delta": 0.02, "beta": 0.001, "quat": quats[1],
               "coeffs": [(0, 0, 110.0), (12, 7, 22.0), (10, -3, 18.0), (9, 0, 12.0), (2, 1, -9.0)]},
              {"kind": "spherical_harmonics", "delta": 0.02, "beta": 0.001, "quat": quats[0],
               "coeffs": [(0, 0, 105.0), (5, -4, 16.0), (5, 5, -14.0), (1, 0, 6.0), (3, 3, 9.0), (5, -4, 5.0)]},
              {"kind": "spherical_harmonics", "delta": 0.02, "beta": 0.001, "quat": quats[2],
               "coeffs": [(0, 0, 105.0), (7, -7, 13.0), (7, 2, -15.0), (6, -1, 11.0), (4, 4, 9.0)]}]
    _check(sm, shapes, (64, 60, 56), (1.6, 1.6, 1.6))


def test_radial_maps(sm):
    rng = np.random.default_rng(13)
    nlat, nlon = 48, 96
    lat = (-pi / 2 + np.arange(nlat) * pi / nlat)[:, None]
    lon = (np.arange(nlon) * 2 * pi / nlon)[None, :]
    smooth = 30.0 + 6.0 * np.cos(3 * lon) * np.cos(lat) ** 2 + 4.0 * np.sin(2 * lat) + rng.uniform(-0.5, 0.5, (nlat, nlon))
    quats = W.random_quaternions(rng, 2)
    shapes = [{"kind": "radial_map", "delta": 0.02, "beta": 0.05, "radii": smooth},
              {"kind": "radial_map", "delta": 0.02, "beta": 0.05, "quat": quats[0], "radii": smooth},
              {"kind": "radial_map", "delta": 0.02, "beta": 0.0, "quat": quats[1], "radii": rng.uniform(20.0, 38.0, (4, 4))},
              {"kind": "radial_map", "delta": 0.02, "beta": 0.0, "radii": np.full((1, 1), 21.0)}]
    _check(sm, shapes, (50, 50, 50), (1.9, 1.9, 1.9))


def test_volume_maps(sm):
    rng = np.random.default_rng(14)
    quats = W.random_quaternions(rng, 2)
    vol = rng.random((11, 17, 23)) < 0.5
    shapes = [{"kind": "volume_map", "delta": 0.04, "beta": 0.02, "volume": vol, "dx": 3.7},
              {"kind": "volume_map", "delta": 0.04, "beta": 0.02, "quat": quats[0], "volume": vol, "dx": 3.7},
              {"kind": "volume_map", "delta": 0.04, "beta": 0.02, "quat": quats[1], "volume": np.ones((10, 10, 10), bool), "dx": 2.0}]
    got = _check(sm, shapes, (64, 48, 40), (1.0, 1.0, 1.0), tie=1e-9)
    cube = sm.render([_to_device({"kind": "volume_map", "delta": 1.0, "beta": 0.0, "volume": np.ones((10, 10, 10), bool), "dx": 2.0})],
                     (32, 32, 32), (1.0, 1.0, 1.0)).cpu().numpy()
    assert int(cube[0, ..., 0].sum()) == 20 ** 3          # the paper's example


def test_rendered_shapes_through_the_whole_path(sm):
    """render -> simulate on the GPU against oracle render -> oracle simulate (the rendered grid is already oriented)."""
    rng = np.random.default_rng(15)
    quats = W.random_quaternions(rng, 3)
    dims, voxel, lam = (48, 40, 36), (3.0, 3.0, 3.0), 18.0
    shapes = [{"kind": "ellipsoid", "delta": 0.02, "beta": 0.004, "quat": quats[0], "a": 55.0, "b": 35.0, "c": 25.0},
              {"kind": "spherical_harmonics", "delta": 0.03, "beta": 0.01, "quat": quats[1], "coeffs": _droplet_coeffs(rng, 40.0, 4, 0.1)},
              {"kind": "volume_map", "delta": 0.05, "beta": 0.0, "quat": quats[2], "volume": rng.random((6, 7, 8)) < 0.6, "dx": 9.0}]
    g = sm.render([_to_device(s) for s in shapes], dims, voxel)
    I = sm.simulate(g, voxel, lam, 24, 20, 30.0).cpu().numpy()
    gh = g.cpu().numpy()
    for b, s in enumerate(shapes):
        ref_grid = R.render(s, dims, voxel)
        assert np.mean(np.any(gh[b] != ref_grid, axis=-1)) < 1e-4
        ref = O.simulate(gh[b], voxel, lam, 24, 20, 30.0)
        assert_parity(I[b], ref, what=f"rendered {s['kind']}")


def test_render_error_codes(sm):
    import torch
    from paper_2202_03411_b200 import binding as B
    dims, voxel = (8, 8, 8), (1.0, 1.0, 1.0)
    bad = [{"kind": "ellipsoid", "delta": 0.01, "beta": 0.0, "a": -1.0, "b": 1.0, "c": 1.0},
           {"kind": "ellipsoid", "delta": 0.01, "beta": 0.0, "quat": [2.0, 0, 0, 0], "a": 1.0, "b": 1.0, "c": 1.0},
           {"kind": "spherical_harmonics", "delta": 0.01, "beta": 0.0, "coeffs": [(2, 3, 1.0)]},
           {"kind": "spherical_harmonics", "delta": 0.01, "beta": 0.0, "coeffs": [(1.5, 0, 1.0)]},
           {"kind": "volume_map", "delta": 0.01, "beta": 0.0, "volume": torch.ones((2, 2, 2), dtype=torch.uint8, device="cuda"), "dx": 0.0}]
    for s in bad:
        with pytest.raises(B.ScatmanError) as e:
            sm.render([s], dims, voxel)
        assert e.value.status == B.INVALID_ARGUMENT


def test_simulate_shapes_equals_render_then_simulate_and_matches_oracle(sm):
    """scatman_simulate_shapes = scatman_render + scatman_simulate on the rendered grids, and the result matches
    the oracle run on the oracle's own rendering (cfg4 shapes at quarter scale: ellipsoids and l <= 4 droplets, oriented)."""
    import torch
    w = W.config(3, scale=0.25)
    items = [0, 1, 2, 3, 4, 5]
    shapes = w.shapes(items)
    dims, vox = (w.nx, w.ny, w.nz), (w.dx, w.dy, w.dz)
    I = sm.simulate_shapes(shapes, dims, vox, w.lam, w.npx, w.npy, w.theta_max_deg)
    g = sm.render(shapes, dims, vox)
    I2 = sm.simulate(g, vox, w.lam, w.npx, w.npy, w.theta_max_deg)
    assert torch.allclose(I, I2, rtol=1e-4, atol=1e-6 * float(I2.max()))     # two MMA issuers: equal to FP32 summation order
    I = I.cpu().numpy()
    for i, s in enumerate(shapes):
        ref_grid = R.render(s, dims, vox)
        assert np.mean(np.any(g[i].cpu().numpy() != ref_grid, axis=-1)) < 1e-4
        ref = O.simulate(g[i].cpu().numpy(), vox, w.lam, w.npx, w.npy, w.theta_max_deg)
        assert_parity(I[i], ref, what=f"shapes item {items[i]}")


def test_simulate_shapes_qgrid_equals_render_then_qgrid_and_matches_oracle(sm):
    """scatman_simulate_shapes_qgrid = scatman_render + scatman_simulate_qgrid on the rendered grids, and matches the oracle's
    direct sum at the grid points (cfg4 shapes at quarter scale on a uniform (qx, qy) grid)."""
    import torch
    w = W.config(3, scale=0.25)
    items = [0, 1, 2, 3, 4]
    shapes = w.shapes(items)
    dims, vox = (w.nx, w.ny, w.nz), (w.dx, w.dy, w.dz)
    k = 2 * np.pi / w.lam
    q1 = (np.arange(w.npx) + 0.5 - 0.5 * w.npx) * (2 * k * np.sin(np.radians(w.theta_max_deg)) / w.npx)
    qx = qy = torch.from_numpy(q1).cuda()
    I = sm.simulate_shapes_qgrid(shapes, dims, vox, w.lam, qx, qy)
    g = sm.render(shapes, dims, vox)
    I2 = sm.simulate_qgrid(g, vox, w.lam, qx, qy)
    assert torch.allclose(I, I2, rtol=1e-4, atol=1e-6 * float(I2.max()))
    I = I.cpu().numpy()
    for i in (0, 3):
        ref = O.simulate_qgrid(g[i].cpu().numpy(), vox, w.lam, q1, q1)
        assert_parity(I[i], ref, what=f"shapes qgrid item {items[i]}")


def test_simulate_shapes_nufft_equals_render_then_nufft_and_matches_oracle(sm):
    """scatman_simulate_shapes_nufft = scatman_render + scatman_simulate_nufft on the rendered grids, and matches the
    oracle on the flat detector (cfg4 shapes at quarter scale)."""
    import torch
    w = W.config(3, scale=0.25)
    items = [0, 1, 2, 3, 4, 5]
    shapes = w.shapes(items)
    dims, vox = (w.nx, w.ny, w.nz), (w.dx, w.dy, w.dz)
    I = sm.simulate_shapes_nufft(shapes, dims, vox, w.lam, w.npx, w.npy, w.theta_max_deg)
    g = sm.render(shapes, dims, vox)
    I2 = sm.simulate_nufft(g, vox, w.lam, w.npx, w.npy, w.theta_max_deg)
    assert torch.allclose(I, I2, rtol=1e-4, atol=1e-6 * float(I2.max()))     # tcgen05 stages: equal to FP32 summation order
    I = I.cpu().numpy()
    for i in (0, 1, 4):
        ref = O.simulate(g[i].cpu().numpy(), vox, w.lam, w.npx, w.npy, w.theta_max_deg)
        assert_parity(I[i], ref, what=f"shapes nufft item {items[i]}")


def test_shape_batches_large_enough_for_the_sparse_render_and_fused_prefix_pass(sm):
    """24 shapes on 128 x 120 x 24 voxels: the chunk has more than 4 * 2^16 columns, so scatman_simulate_shapes_nufft / _qgrid render
    SPARSELY (tiles outside the circumscribed sphere are neither written nor read: tile map) into a workspace that is poisoned
    first, and the fused prefix pass packs the planes.  Equal (to FP32 summation order) to render -> simulate on dense grids, and
    items of each kind against the oracle."""
    import torch
    rng = np.random.default_rng(401)
    quats = W.random_quaternions(rng, 24)
    shapes = []
    for i in range(24):
        if i % 3 == 0:
            shapes.append({"kind": "ellipsoid", "delta": 0.01 + 0.001 * i, "beta": 0.002, "quat": quats[i],
                           "a": 20.0 + 3 * i, "b": 16.0 + 2 * i, "c": 12.0 + i})
        elif i % 3 == 1:
            shapes.append({"kind": "spherical_harmonics", "delta": 0.02, "beta": 0.004, "quat": quats[i],
                           "coeffs": _droplet_coeffs(rng, 25.0 + 2.5 * i, 4, 0.08)})
        else:
            shapes.append({"kind": "spherical_harmonics", "delta": 0.03, "beta": 0.0, "quat": quats[i],
                           "coeffs": [(0, 0, (15.0 + 2 * i) * sqrt(4 * pi)), (10, 4, 6.0), (3, -1, 4.0)]})     # degree > 8: the triplet walker
    shapes[5] = {"kind": "ellipsoid", "delta": 0.02, "beta": 0.001, "a": 0.4, "b": 0.4, "c": 0.4}      # smaller than a voxel, off every centre: vacuum
    dims, vox, lam = (128, 120, 24), (2.0, 2.0, 2.5), 12.0
    npx, npy, th = 21, 18, 30.0
    g = sm.render(shapes, dims, vox)
    # poison the caches of freed blocks: the sparse renderer must not depend on what its workspace held
    junk = torch.full((64 << 20,), float("nan"), dtype=torch.float32, device="cuda")
    del junk
    I = sm.simulate_shapes_nufft(shapes, dims, vox, lam, npx, npy, th)
    I2 = sm.simulate_nufft(g, vox, lam, npx, npy, th)
    assert bool(torch.isfinite(I).all())
    assert torch.allclose(I, I2, rtol=2e-4, atol=1e-6 * float(I2.max()))
    assert float(I[5].abs().max()) == 0.0
    In = I.cpu().numpy()
    for i in (0, 1, 2, 23):
        assert_parity(In[i], O.simulate(g[i].cpu().numpy(), vox, lam, npx, npy, th), what=f"sparse-rendered nufft item {i}")
    k = 2 * np.pi / lam
    qx = (np.arange(23) + 0.5 - 11.5) * (2 * k * np.sin(np.radians(30.0)) / 23)
    qy = (np.arange(19) + 0.5 - 9.5) * (2 * k * np.sin(np.radians(25.0)) / 19)
    dqx, dqy = torch.from_numpy(qx).cuda(), torch.from_numpy(qy).cuda()
    J = sm.simulate_shapes_qgrid(shapes, dims, vox, lam, dqx, dqy)
    J2 = sm.simulate_qgrid(g, vox, lam, dqx, dqy)
    assert torch.allclose(J, J2, rtol=2e-4, atol=1e-6 * float(J2.max()))
    assert_parity(J[1].cpu().numpy(), O.simulate_qgrid(g[1].cpu().numpy(), vox, lam, qx, qy), what="sparse-rendered qgrid item 1")


def test_workload_shape_descriptors_describe_the_same_particles_as_the_grids(sm):
    """The descriptors of cfg1 / cfg3 (identity orientation) render to exactly the voxel grids the generators produce."""
    for idx, scale in ((0, 1.0), (2, 0.25)):
        w = W.config(idx, scale=scale)
        got = sm.render(w.shapes([0]), (w.nx, w.ny, w.nz), (w.dx, w.dy, w.dz)).cpu().numpy()[0]
        ref = w.grid(0)
        assert np.mean(np.any(got != ref, axis=-1)) < 1e-5, idx
