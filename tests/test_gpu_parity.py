"""GPU parity: the CUDA path (through the C ABI) against the FP64 oracle on the same seeded inputs."""
import numpy as np
import pytest

from oracle import oracle as O
from paper_2202_03411_b200 import workloads as W
from parity import assert_parity, metrics

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


# name -> (method, flags): CTA-pair tensor kernel (default), single-CTA tensor kernel, CUDA-core sincos and table variants
METHODS = {"tensor": (1, 0), "tensor_1cta": (1, 1), "simt_sincos": (2, 0), "simt_table": (3, 0)}


# ------------------------------------------------------------------------------------------ stage kernels
def test_qmap_matches_oracle(sm):
    for (npx, npy, th, lam, cx, cy) in [(64, 64, 30.0, 20.0, 0, 0), (37, 21, 60.0, 10.0, 1.5, -2.0), (1, 1, 10.0, 1.0, 0, 0)]:
        q = sm.qmap(npx, npy, th, lam, cx, cy).cpu().numpy()
        ref = O.qmap(npx, npy, th, lam, cx, cy)
        assert np.allclose(q, ref, rtol=1e-13, atol=1e-300)


def test_orient_matches_oracle(sm):
    rng = np.random.default_rng(5)
    g = np.stack([W.random_grid(31 + i, 13, 9, 11) for i in range(3)])
    quat = W.random_quaternions(rng, 3)
    voxel = (2.0, 1.5, 1.0)
    out = sm.orient(dev(g), voxel, quat).cpu().numpy()
    for b in range(3):
        ref = O.orient(g[b], voxel, quat[b])
        assert np.allclose(out[b], ref, rtol=2e-7, atol=1e-12)


def test_effective_strength_matches_oracle(sm):
    g = W.random_grid(41, 19, 7, 23, delta=(-0.02, 0.08), beta=(0.0, 0.05))
    voxel, lam = (2.0, 2.0, 3.0), 9.0
    for mode in (0, 1):
        rho = sm.effective_strength(dev(g), voxel, lam, rho_mode=mode).cpu().numpy()
        ref = O.effective_strength(g, voxel, lam, mode) / np.prod(voxel)
        got = rho[..., 0] + 1j * rho[..., 1]
        assert np.max(np.abs(got - ref)) <= 2e-7 * np.max(np.abs(ref))
        assert np.all(got[ref == 0] == 0)


# ------------------------------------------------------------------------------------------ whole path
@pytest.mark.parametrize("method", list(METHODS))
def test_cfg1_sphere_full_pattern(sm, method):
    w = W.config(0)
    g = w.grid(0)
    I = sm.simulate(dev(g), (w.dx, w.dy, w.dz), w.lam, w.npx, w.npy, w.theta_max_deg, method=METHODS[method][0], flags=METHODS[method][1]).cpu().numpy()
    ref = O.simulate(g, (w.dx, w.dy, w.dz), w.lam, w.npx, w.npy, w.theta_max_deg)
    assert_parity(I, ref, what=f"cfg1 {method}")


@pytest.mark.parametrize("method", list(METHODS))
@pytest.mark.parametrize("mode", [0, 1])
def test_ragged_random_batch_with_orientations(sm, method, mode):
    """Odd sizes everywhere: several tiles plus ragged tails in x, y, pixels; batch with quaternions."""
    rng = np.random.default_rng(8)
    nx, ny, nz, B = 150, 70, 13, 3
    g = np.stack([W.random_grid(51 + i, nx, ny, nz, fill=0.5) for i in range(B)])
    quat = W.random_quaternions(rng, B)
    quat[1] = [1, 0, 0, 0]
    voxel, lam = (2.0, 2.5, 3.0), 14.0
    npx, npy, th = 23, 19, 35.0
    I = sm.simulate(dev(g), voxel, lam, npx, npy, th, quat=quat, rho_mode=mode, method=METHODS[method][0], flags=METHODS[method][1]).cpu().numpy()
    for b in range(B):
        ref = O.simulate(g[b], voxel, lam, npx, npy, th, quat=quat[b], rho_mode=mode)
        assert_parity(I[b], ref, what=f"ragged b={b} {method} mode={mode}")


@pytest.mark.parametrize("method", ["tensor", "tensor_1cta"])
@pytest.mark.parametrize("seed", [71, 72, 73])
def test_sparse_blobs_exercise_block_skipping(sm, method, seed):
    """Mostly empty grids whose occupied 16 x 16 blocks differ per slice, x tile and y group: the contraction skips
    empty y steps and narrows each unit to its occupied x range; the result must not change."""
    nx, ny, nz, B = 300, 200, 10, 2
    g = np.stack([W.sparse_blobs_grid(seed + 10 * i, nx, ny, nz, nblobs=5 + 3 * i, max_extent=20 + 60 * i) for i in range(B)])
    voxel, lam = (2.0, 2.0, 2.5), 11.0
    npx, npy, th = 20, 17, 25.0
    I = sm.simulate(dev(g), voxel, lam, npx, npy, th, method=METHODS[method][0], flags=METHODS[method][1]).cpu().numpy()
    for b in range(B):
        ref = O.simulate(g[b], voxel, lam, npx, npy, th)
        assert_parity(I[b], ref, what=f"sparse blobs seed={seed} b={b} {method}")


@pytest.mark.parametrize("method", list(METHODS))
def test_cfg2_ellipsoid_half_scale_oriented(sm, method):
    w = W.config(1, scale=0.5)
    g = w.grid(0)
    I = sm.simulate(dev(g), (w.dx, w.dy, w.dz), w.lam, w.npx, w.npy, w.theta_max_deg, quat=w.quat, method=METHODS[method][0], flags=METHODS[method][1]).cpu().numpy()
    ref = O.simulate(g, (w.dx, w.dy, w.dz), w.lam, w.npx, w.npy, w.theta_max_deg, quat=w.quat[0])
    assert_parity(I, ref, what=f"cfg2 half {method}")


def test_cfg3_droplet_quarter_scale(sm):
    w = W.config(2, scale=0.25)
    g = w.grid(0)
    I = sm.simulate(dev(g), (w.dx, w.dy, w.dz), w.lam, w.npx, w.npy, w.theta_max_deg).cpu().numpy()
    ref = O.simulate(g, (w.dx, w.dy, w.dz), w.lam, w.npx, w.npy, w.theta_max_deg)
    assert_parity(I, ref, what="cfg3 quarter")


def test_cfg4_batch_subset_quarter_scale(sm):
    w = W.config(3, scale=0.25)
    items = [0, 1, 2, 3, 4, 5, 6]
    g = w.grids(items)
    quat = w.quat[items]
    I = sm.simulate(dev(g), (w.dx, w.dy, w.dz), w.lam, w.npx, w.npy, w.theta_max_deg, quat=quat).cpu().numpy()
    for i, b in enumerate(items):
        ref = O.simulate(g[i], (w.dx, w.dy, w.dz), w.lam, w.npx, w.npy, w.theta_max_deg, quat=quat[i])
        assert_parity(I[i], ref, what=f"cfg4 item {b}")


def test_cfg5_coreshell_eighth_scale(sm):
    w = W.config(4, scale=0.125)
    g = w.grid(0)
    I = sm.simulate(dev(g), (w.dx, w.dy, w.dz), w.lam, w.npx, w.npy, w.theta_max_deg).cpu().numpy()
    ref = O.simulate(g, (w.dx, w.dy, w.dz), w.lam, w.npx, w.npy, w.theta_max_deg)
    assert_parity(I, ref, what="cfg5 eighth")


# ------------------------------------------------------------------------------------------ special cases
def test_forward_pixel_and_explicit_q(sm):
    import torch
    g = W.random_grid(61, 40, 33, 9)
    voxel, lam = (2.0, 2.0, 2.0), 15.0
    k = 2 * np.pi / lam
    rng = np.random.default_rng(3)
    th = rng.uniform(0, 0.8, 200); ph = rng.uniform(-np.pi, np.pi, 200)
    q = np.stack([k * np.sin(th) * np.cos(ph), k * np.sin(th) * np.sin(ph), k * (np.cos(th) - 1)], axis=1)
    q[0] = 0.0
    for m, fl in METHODS.values():
        I = sm.simulate_q(dev(g), voxel, lam, torch.from_numpy(q).cuda(), method=m, flags=fl).cpu().numpy()
        ref = O.simulate_q(g, voxel, lam, q)
        assert_parity(I, ref, what="explicit q")
        assert abs(I[0] - ref[0]) <= 2e-6 * ref[0]


def test_empty_and_single_voxel(sm):
    voxel, lam = (3.0, 3.0, 3.0), 12.0
    z = np.zeros((8, 8, 8, 2), np.float32)
    for m, fl in METHODS.values():
        I = sm.simulate(dev(z), voxel, lam, 16, 16, 30.0, method=m, flags=fl).cpu().numpy()
        assert np.all(I == 0)
        one = z.copy()
        one[2, 5, 1] = (0.03, 0.004)
        I = sm.simulate(dev(one), voxel, lam, 16, 16, 30.0, method=m, flags=fl).cpu().numpy()
        exact = abs((float(np.float32(0.03)) + 1j * float(np.float32(0.004))) * 27.0) ** 2
        assert np.allclose(I, exact, rtol=2e-5)


def test_large_batch_with_vacuum_items_and_many_orientations(sm):
    """40 small grids in one call (more than one 32-matrix upload chunk), random orientations, some items all vacuum, some
    identity: every item's pattern is its own (no cross-talk through the batch loop, the per-item scales or the partial sums)."""
    rng = np.random.default_rng(17)
    B, n = 40, 24
    g = np.stack([W.sparse_blobs_grid(300 + i, n + 8, n, n - 4, nblobs=3, max_extent=10) for i in range(B)])
    g[[3, 17, 39]] = 0.0
    g[5] *= 1e-3                                  # a much weaker item: its FP16 scale differs by 2^10 from its neighbours'
    quat = W.random_quaternions(rng, B)
    quat[[0, 9]] = [1, 0, 0, 0]
    voxel, lam = (3.0, 3.0, 3.0), 16.0
    npx, npy, th = 12, 10, 30.0
    for name in ("tensor", "tensor_1cta"):
        I = sm.simulate(dev(g), voxel, lam, npx, npy, th, quat=quat, method=METHODS[name][0], flags=METHODS[name][1]).cpu().numpy()
        assert np.all(I[[3, 17, 39]] == 0)
        for b in range(B):
            if b in (3, 17, 39):
                continue
            ref = O.simulate(g[b], voxel, lam, npx, npy, th, quat=quat[b])
            assert_parity(I[b], ref, what=f"batch40 {name} b={b}")


def test_n2m1_mode_on_an_absorbing_inhomogeneous_grid(sm):
    """rho = n^2 - 1 (paper, Eq. 5/9) against the oracle on a grid where it is not proportional to n - 1."""
    g = W.random_grid(77, 64, 48, 20, fill=0.7, delta=(-0.05, 0.3), beta=(0.0, 0.2))
    voxel, lam = (2.0, 2.0, 2.0), 9.0
    I1 = sm.simulate(dev(g), voxel, lam, 24, 24, 40.0, rho_mode=1).cpu().numpy()
    I0 = sm.simulate(dev(g), voxel, lam, 24, 24, 40.0, rho_mode=0).cpu().numpy()
    assert_parity(I1, O.simulate(g, voxel, lam, 24, 24, 40.0, rho_mode=1), what="n2m1")
    assert np.max(np.abs(I1 / I0 - 4.0)) > 0.3          # far from the homogeneous-particle constant |2 - dn|^2 ~ 4


def test_issued_block_count(sm):
    """scatman_last_issued_blocks: what the contraction multiplies after skipping empty 16-y steps and narrowing units
    to their occupied 16-x blocks, on grids where the count is known by hand."""
    from paper_2202_03411_b200 import binding as B
    voxel, lam = (2.0, 2.0, 2.0), 12.0
    g = np.full((13, 70, 150, 2), 0.01, np.float32)          # every voxel non-zero: nz=13, ny=70, nx=150
    sm.simulate(dev(g), voxel, lam, 16, 16, 20.0, flags=B.FLAG_COUNT_ISSUED)
    assert sm.last_issued_blocks() == 13 * (5 * 8 + 5 * 2)    # 5 y steps; x tile 0 full (8 blocks), tile 1 holds 22 x (2 blocks)
    sm.simulate(dev(g), voxel, lam, 16, 16, 20.0, flags=B.FLAG_COUNT_ISSUED | B.FLAG_SINGLE_CTA)
    assert sm.last_issued_blocks() == 13 * (5 * 8 + 5 * 8)    # a single CTA runs full tiles
    z = np.zeros_like(g)
    z[3, 40, 100] = (0.02, 0.001)                             # one voxel -> one block
    sm.simulate(dev(z), voxel, lam, 16, 16, 20.0, flags=B.FLAG_COUNT_ISSUED)
    assert sm.last_issued_blocks() == 1
    z[3, 40, 30] = (0.02, 0.001)                              # same y step, x blocks 1..6 of tile 0 -> range of 6
    sm.simulate(dev(z), voxel, lam, 16, 16, 20.0, flags=B.FLAG_COUNT_ISSUED)
    assert sm.last_issued_blocks() == 6
    sm.simulate(dev(z), voxel, lam, 16, 16, 20.0)
    assert sm.last_issued_blocks() == -1


def test_deterministic_and_workspace_reuse(sm):
    import torch
    w = W.config(0)
    d = dev(w.grid(0))
    a = sm.simulate(d, (w.dx, w.dy, w.dz), w.lam, w.npx, w.npy, w.theta_max_deg).clone()
    b = sm.simulate(d, (w.dx, w.dy, w.dz), w.lam, w.npx, w.npy, w.theta_max_deg).clone()
    assert torch.equal(a, b)
    assert sm.last_launch_count() == 7   # q-map, prefix, pack, 2 table launches, contraction, finalize


def test_simulate_host_matches_device_path(sm):
    import torch
    w = W.config(0)
    g = w.grid(0)
    h = torch.from_numpy(g).pin_memory()
    I_h = sm.simulate_host(h, (w.dx, w.dy, w.dz), w.lam, w.npx, w.npy, w.theta_max_deg)
    I_d = sm.simulate(dev(g), (w.dx, w.dy, w.dz), w.lam, w.npx, w.npy, w.theta_max_deg).cpu()
    assert torch.equal(I_h[0], I_d)


def test_error_codes(sm):
    import torch
    from paper_2202_03411_b200 import binding as B
    w = W.config(0)
    d = dev(w.grid(0))
    vox = (w.dx, w.dy, w.dz)
    with pytest.raises(B.ScatmanError) as e:
        sm.simulate(d, vox, w.lam, 64, 64, 30.0, workspace=torch.empty(1024, dtype=torch.uint8, device="cuda"))
    assert e.value.status == B.WORKSPACE_TOO_SMALL
    for bad in [dict(lam=-1.0), dict(theta=95.0), dict(quat=[[2.0, 0, 0, 0]]), dict(method=9)]:
        with pytest.raises(B.ScatmanError) as e:
            sm.simulate(d, vox, bad.get("lam", w.lam), 64, 64, bad.get("theta", 30.0), quat=bad.get("quat"),
                        method=bad.get("method", 0))
        assert e.value.status == B.INVALID_ARGUMENT


# ------------------------------------------------------------------------------------------ full sizes, sampled pixels
def _sampled_full(sm, idx, count, items=None):
    import torch
    w = W.config(idx)
    vox = (w.dx, w.dy, w.dz)
    items = [0] if items is None else items
    g = w.grids(items)
    quat = None if w.quat is None else w.quat[items]
    I = sm.simulate(dev(g), vox, w.lam, w.npx, w.npy, w.theta_max_deg, quat=quat).cpu().numpy()
    for i in range(len(items)):
        flat = I[i].ravel()
        c = w.npy // 2 * w.npx + w.npx // 2
        pix = W.sample_pixels(w.seed + i, w.npix, count, always=[int(np.argmax(flat)), c, c - 1, c - w.npx, c - w.npx - 1])
        ref = O.simulate(g[i], vox, w.lam, w.npx, w.npy, w.theta_max_deg, quat=None if quat is None else quat[i], pixels=pix)
        assert_parity(flat[pix], ref, what=f"{w.name} item {items[i]} sampled")


def test_cfg2_full_size_sampled(sm):
    _sampled_full(sm, 1, 512)


def test_cfg3_full_size_sampled(sm):
    _sampled_full(sm, 2, 192)


def test_cfg4_full_size_items_sampled(sm):
    _sampled_full(sm, 3, 128, items=[0, 1, 2, 3, 4, 5, 6, 7, 8])


def test_cfg5_full_size_sampled(sm):
    _sampled_full(sm, 4, 48)
