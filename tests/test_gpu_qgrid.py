"""GPU parity of the separable tensor-grid route (scatman_simulate_qgrid; tcgen05 stages of sep_tensor_kernels.cu and the
FP32 CUDA-core stages of sep_kernels.cu) against the oracle's direct triple sum at the same grid points, and against
numpy.fft2 where the grid is the DFT grid."""
import numpy as np
import pytest

from oracle import oracle as O
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


METHODS = {"tensor": 1, "simt": 3}
both_methods = pytest.mark.parametrize("method", list(METHODS))


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _uniform_q(lam, theta_max_deg, n):
    """n points of a uniform transverse grid reaching sin(theta_max) k (the paper's 'same angular cross section' pixels)."""
    k = 2 * np.pi / lam
    return (np.arange(n) + 0.5 - 0.5 * n) * (2 * k * np.sin(np.radians(theta_max_deg)) / n)


@both_methods
@pytest.mark.parametrize("mode", [0, 1])
def test_ragged_batch_with_orientations(sm, mode, method):
    rng = np.random.default_rng(31)
    nx, ny, nz, B = 70, 45, 11, 3
    g = np.stack([W.random_grid(81 + i, nx, ny, nz, fill=0.4) for i in range(B)])
    quat = W.random_quaternions(rng, B)
    quat[2] = [1, 0, 0, 0]
    voxel, lam = (2.0, 2.5, 3.0), 14.0
    qx, qy = _uniform_q(lam, 35.0, 37), _uniform_q(lam, 25.0, 29)
    I = sm.simulate_qgrid(dev(g), voxel, lam, dev(qx), dev(qy), quat=quat, rho_mode=mode, method=METHODS[method]).cpu().numpy()
    for b in range(B):
        ref = O.simulate_qgrid(g[b], voxel, lam, qx, qy, quat=quat[b], rho_mode=mode)
        assert_parity(I[b], ref, what=f"qgrid {method} ragged b={b} mode={mode}")


@both_methods
@pytest.mark.parametrize("nx", [126, 125])
def test_fused_prefix_pass_on_an_oriented_batch(sm, method, nx):
    """A batch whose chunk has more than 4 * 2^16 columns: the tensor stages take the fused prefix -> planes pass on the orientation's
    sparse output (tile map, scale from the bound of max |rho~|, layers without material not packed); see test_gpu_nufft.py."""
    ny, nz, B_ = 120, 22, 20
    g = np.stack([W.sparse_blobs_grid(700 + i, nx, ny, nz, nblobs=5, max_extent=30) for i in range(B_)])
    g[3] = W.random_grid(703, nx, ny, nz, fill=0.4, delta=(-0.01, 0.03), beta=(-0.02, 0.0))      # gain
    g[5] = W.random_grid(705, nx, ny, nz, fill=0.2, delta=(-1e-6, 1e-6), beta=(0.0, 1e-7))        # weak
    g[7] = 0.0                                                                                    # vacuum
    quat = W.random_quaternions(np.random.default_rng(77), B_)
    quat[2] = [1, 0, 0, 0]
    voxel, lam = (2.0, 2.0, 2.5), 12.0
    qx, qy = _uniform_q(lam, 30.0, 23), _uniform_q(lam, 25.0, 19)
    I = sm.simulate_qgrid(dev(g), voxel, lam, dev(qx), dev(qy), quat=quat, method=METHODS[method]).cpu().numpy()
    assert np.all(I[7] == 0)
    for b in (0, 2, 3, 5, 11, 19):
        ref = O.simulate_qgrid(g[b], voxel, lam, qx, qy, quat=quat[b])
        assert_parity(I[b], ref, what=f"qgrid {method} fused oriented batch item {b} nx={nx}")


@both_methods
def test_sparse_blobs_and_evanescent_points(sm, method):
    """Mostly empty grid (the kernels skip vacuum rows); a q grid that runs past |q_xy| = k: those points must be exactly 0."""
    g = W.sparse_blobs_grid(91, 150, 130, 9, nblobs=6, max_extent=40)
    voxel, lam = (2.0, 2.0, 2.5), 11.0
    k = 2 * np.pi / lam
    qx, qy = np.linspace(-1.2 * k, 1.2 * k, 41), np.linspace(-0.8 * k, 0.8 * k, 33)
    I = sm.simulate_qgrid(dev(g), voxel, lam, dev(qx), dev(qy), method=METHODS[method]).cpu().numpy()
    ref = O.simulate_qgrid(g, voxel, lam, qx, qy)
    _, ok = O.qgrid_q(qx, qy, lam)
    assert not ok.all() and np.all(I.ravel()[~ok] == 0)
    assert_parity(I, ref, what=f"qgrid sparse {method}")


@both_methods
def test_batch_with_a_vacuum_item_and_a_single_voxel(sm, method):
    """Items are stacked along z inside one set of launches: an all-vacuum item must come out exactly 0, a single voxel as
    |rho dV|^2 at every propagating grid point, and neither may disturb its neighbours."""
    nx, ny, nz = 40, 70, 9
    voxel, lam = (2.0, 2.0, 3.0), 12.0
    g = np.stack([W.random_grid(60 + i, nx, ny, nz, fill=0.3) for i in range(5)])
    g[1] = 0.0
    g[3] = 0.0
    g[3, 4, 33, 17] = (0.02, 0.003)
    k = 2 * np.pi / lam
    qx, qy = np.linspace(-0.7 * k, 0.9 * k, 45), np.linspace(-0.5 * k, 0.5 * k, 31)
    I = sm.simulate_qgrid(dev(g), voxel, lam, dev(qx), dev(qy), method=METHODS[method]).cpu().numpy()
    _, ok = O.qgrid_q(qx, qy, lam)
    ok = ok.reshape(31, 45)
    assert np.all(I[1] == 0)
    one = (0.02 ** 2 + 0.003 ** 2) * (2.0 * 2.0 * 3.0) ** 2
    assert np.allclose(I[3][ok], one, rtol=2e-5) and np.all(I[3][~ok] == 0)
    for b in (0, 2, 4):
        assert_parity(I[b], O.simulate_qgrid(g[b], voxel, lam, qx, qy), what=f"qgrid {method} batch item {b}")


def test_batch_larger_than_one_chunk(sm):
    """The H planes of a chunk are capped at 4 GB: nine items of 512 MB each run as a chunk of eight and a chunk of one.
    Checked at seeded grid points of three items."""
    nx, ny, nz, B_ = 16, 900, 64, 9
    voxel, lam = (3.0, 1.0, 2.0), 9.0
    g = np.stack([W.sparse_blobs_grid(300 + i, nx, ny, nz, nblobs=5, max_extent=12) for i in range(B_)])
    k = 2 * np.pi / lam
    qx, qy = np.linspace(-0.6 * k, 0.6 * k, 1000), np.linspace(-0.3 * k, 0.3 * k, 8)
    I = sm.simulate_qgrid(dev(g), voxel, lam, dev(qx), dev(qy), method=METHODS["tensor"]).cpu().numpy()
    q, ok = O.qgrid_q(qx, qy, lam)
    pix = W.sample_pixels(17, 8000, 60)
    for b in (0, 7, 8):
        ref = O.simulate_q(g[b], voxel, lam, q[pix]) * ok[pix]
        assert_parity(I[b].ravel()[pix], ref, what=f"qgrid chunked batch item {b}")


@pytest.mark.parametrize("nx", [300, 530, 1100])
def test_wide_grids_use_narrower_stage_x_tiles(sm, nx):
    """nx > 256 / > 512: stage X keeps 32- / 16-column Ex tiles resident; nx > 1024 falls back to the CUDA-core stages."""
    g = W.random_grid(97, nx, 20, 3, fill=0.5)
    voxel, lam = (1.5, 2.0, 2.5), 9.0
    qx, qy = _uniform_q(lam, 20.0, 70), _uniform_q(lam, 30.0, 19)
    I = sm.simulate_qgrid(dev(g), voxel, lam, dev(qx), dev(qy), method=METHODS["tensor"]).cpu().numpy()
    ref = O.simulate_qgrid(g, voxel, lam, qx, qy)
    assert_parity(I, ref, what=f"qgrid tensor nx={nx}")


@both_methods
def test_gain_medium_and_weak_items_keep_their_accuracy(sm, method):
    """As in test_gpu_nufft.py: the tensor stages' FP16 scale comes from a bound of max |rho~| taken before the prefix runs."""
    nx, ny, nz = 70, 50, 24
    voxel, lam = (2.0, 2.0, 2.0), 10.0
    g = np.stack([W.random_grid(61, nx, ny, nz, fill=0.5, delta=(-0.01, 0.03), beta=(-0.02, 0.0)),
                  W.random_grid(62, nx, ny, nz, fill=0.9, delta=(0.01, 0.05), beta=(0.2, 0.4)),
                  W.random_grid(63, nx, ny, nz, fill=0.3, delta=(-1e-6, 1e-6), beta=(0.0, 1e-7))])
    qx, qy = _uniform_q(lam, 30.0, 40), _uniform_q(lam, 25.0, 33)
    I = sm.simulate_qgrid(dev(g), voxel, lam, dev(qx), dev(qy), method=METHODS[method]).cpu().numpy()
    for b in range(3):
        assert_parity(I[b], O.simulate_qgrid(g[b], voxel, lam, qx, qy), what=f"qgrid {method} scale bound item {b}")


@pytest.mark.parametrize("ny", [300, 530, 2100])
def test_tall_grids_use_the_streamed_stage_yz_and_beyond_it_the_cuda_core_stages(sm, ny):
    """N_y > 256: stage YZ streams both operands (odd numbers of 128-row b tiles are padded to pairs); N_y > 2048 falls back to the
    CUDA-core stages."""
    g = W.random_grid(98, 20, ny, 3, fill=0.5)
    voxel, lam = (2.0, 0.4, 2.5), 9.0
    qx, qy = _uniform_q(lam, 30.0, 19), _uniform_q(lam, 20.0, 150)      # 150 rows: two b tiles; 19 columns: one (odd) a tile
    I = sm.simulate_qgrid(dev(g), voxel, lam, dev(qx), dev(qy), method=METHODS["tensor"]).cpu().numpy()
    ref = O.simulate_qgrid(g, voxel, lam, qx, qy)
    assert_parity(I, ref, what=f"qgrid tensor ny={ny}")
    qy3 = _uniform_q(lam, 20.0, 300)                                     # three b tiles: an odd count
    I = sm.simulate_qgrid(dev(g), voxel, lam, dev(qx), dev(qy3), method=METHODS["tensor"]).cpu().numpy()
    assert_parity(I, O.simulate_qgrid(g, voxel, lam, qx, qy3), what=f"qgrid tensor ny={ny}, 300 rows")


@both_methods
def test_cfg1_sphere_on_a_uniform_q_grid(sm, method):
    w = W.config(0)
    g = w.grid(0)
    vox = (w.dx, w.dy, w.dz)
    qx = qy = _uniform_q(w.lam, w.theta_max_deg, 64)
    I = sm.simulate_qgrid(dev(g), vox, w.lam, dev(qx), dev(qy), method=METHODS[method]).cpu().numpy()
    ref = O.simulate_qgrid(g, vox, w.lam, qx, qy)
    assert_parity(I, ref, what=f"qgrid cfg1 {method}")
    assert np.allclose(I, I[::-1, :], rtol=1e-4) and np.allclose(I, I.T, rtol=1e-4)   # D4 symmetry of the sphere pattern


@both_methods
def test_cfg3_quarter_scale_droplet(sm, method):
    w = W.config(2, scale=0.25)
    g = w.grid(0)
    vox = (w.dx, w.dy, w.dz)
    qx, qy = _uniform_q(w.lam, w.theta_max_deg, w.npx), _uniform_q(w.lam, w.theta_max_deg, w.npy)
    I = sm.simulate_qgrid(dev(g), vox, w.lam, dev(qx), dev(qy), method=METHODS[method]).cpu().numpy()
    ref = O.simulate_qgrid(g, vox, w.lam, qx, qy)
    assert_parity(I, ref, what=f"qgrid cfg3 quarter {method}")


@both_methods
def test_single_slice_on_the_dft_grid_is_fft2(sm, method):
    rng = np.random.default_rng(33)
    nx, ny, d = 96, 80, 1.5
    g = np.zeros((1, ny, nx, 2), np.float32)
    g[0, ..., 0] = rng.uniform(-0.02, 0.05, (ny, nx))
    g[0, ..., 1] = rng.uniform(0.0, 0.02, (ny, nx))
    lam = 2.0
    mx, my = np.arange(nx), np.arange(ny)
    qx = -2 * np.pi * np.where(mx < nx / 2, mx, mx - nx) / (nx * d)
    qy = -2 * np.pi * np.where(my < ny / 2, my, my - ny) / (ny * d)
    I = sm.simulate_qgrid(dev(g), (d, d, 2.0), lam, dev(qx), dev(qy), method=METHODS[method]).cpu().numpy()
    rho = g[0, ..., 0].astype(np.float64) + 1j * g[0, ..., 1].astype(np.float64)
    ref = np.abs(np.fft.fft2(rho) * d * d * 2.0) ** 2
    assert_parity(I, ref, what=f"qgrid fft2 {method}")


@both_methods
def test_full_size_cfg3_sampled_points(sm, method):
    """256^3 droplet on a 512 x 512 uniform q grid, checked at seeded grid points (the oracle takes them one by one)."""
    w = W.config(2)
    g = w.grid(0)
    vox = (w.dx, w.dy, w.dz)
    qx, qy = _uniform_q(w.lam, w.theta_max_deg, w.npx), _uniform_q(w.lam, w.theta_max_deg, w.npy)
    I = sm.simulate_qgrid(dev(g), vox, w.lam, dev(qx), dev(qy), method=METHODS[method]).cpu().numpy().ravel()
    q, ok = O.qgrid_q(qx, qy, w.lam)
    c = w.npy // 2 * w.npx + w.npx // 2
    pix = W.sample_pixels(w.seed + 7, w.npix, 160, always=[int(np.argmax(I)), c, c - 1, c - w.npx])
    ref = O.simulate_q(g, vox, w.lam, q[pix]) * ok[pix]
    assert_parity(I[pix], ref, what=f"qgrid cfg3 full sampled {method}")


@pytest.mark.parametrize("npx,npy", [(200, 384), (300, 200), (300, 384)])
def test_tile_parities_select_the_stage_yz_variants(sm, npx, npy):
    """Stage YZ pairs CTAs over two column tiles (2 x 3 tiles of 128: transposed form, Ey resident), else over two row tiles
    (3 x 2: both operands streamed), else runs one CTA per item (3 x 3)."""
    w = W.config(2, scale=0.25)
    g = w.grid(0)
    vox = (w.dx, w.dy, w.dz)
    qx, qy = _uniform_q(w.lam, w.theta_max_deg, npx), _uniform_q(w.lam, w.theta_max_deg, npy)
    I = sm.simulate_qgrid(dev(g), vox, w.lam, dev(qx), dev(qy), method=METHODS["tensor"]).cpu().numpy()
    q, ok = O.qgrid_q(qx, qy, w.lam)
    pix = W.sample_pixels(5, npx * npy, 400)
    ref = O.simulate_q(g, vox, w.lam, q[pix]) * ok[pix]
    assert_parity(I.ravel()[pix], ref, what=f"qgrid {npx} x {npy} points")


def test_error_codes(sm):
    import torch
    from paper_2202_03411_b200 import binding as B
    g = dev(W.random_grid(5, 8, 8, 4))
    q = dev(np.linspace(-0.1, 0.1, 8))
    with pytest.raises(B.ScatmanError) as e:
        sm.simulate_qgrid(g, (1.0, 1.0, 1.0), 10.0, q, q, workspace=torch.empty(64, dtype=torch.uint8, device="cuda"))
    assert e.value.status == B.WORKSPACE_TOO_SMALL
    with pytest.raises(B.ScatmanError) as e:
        sm.simulate_qgrid(g, (1.0, 1.0, 1.0), -1.0, q, q)
    assert e.value.status == B.INVALID_ARGUMENT
