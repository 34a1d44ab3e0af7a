"""GPU parity of the flat-detector NUFFT route (scatman_simulate_nufft) against the FP64 oracle's direct sum:
the same tolerances as the pixel x voxel contraction, on the same seeded inputs."""
import numpy as np
import pytest

from oracle import oracle as O
from paper_2202_03411_b200 import workloads as W
from parity import FULL_SIZE_SAMPLES, assert_parity, metrics, oracle_at_pixels, sampled_pixels

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


# the GEMM stages run on tcgen05 tensor cores in FP16x3 split precision (default) or in FP64 on the CUDA cores (method SIMT_TABLE)
@pytest.fixture(params=["tensor", "fp64"])
def sim(request, sm):
    method = 0 if request.param == "tensor" else 3
    def run(*args, **kw):
        return sm.simulate_nufft(*args, method=method, **kw)
    run.exact = request.param == "fp64"      # bitwise reproducible, FP64 sums
    run.name = request.param
    return run


def test_cfg1_sphere_full_pattern(sm, sim):
    w = W.config(0)
    g = w.grid(0)
    I = sim(dev(g), (w.dx, w.dy, w.dz), w.lam, w.npx, w.npy, w.theta_max_deg).cpu().numpy()
    ref = O.simulate(g, (w.dx, w.dy, w.dz), w.lam, w.npx, w.npy, w.theta_max_deg)
    l2, pix = assert_parity(I, ref, what="nufft cfg1")
    if sim.exact:
        assert l2 <= 1e-6 and pix <= 1e-5  # FP64 throughout: only the FP32 store of rho~ and of I is left
    else:
        assert l2 <= 1e-5 and pix <= 1e-4  # FP16x3: 22 bits per factor


@pytest.mark.parametrize("mode", [0, 1])
def test_ragged_random_batch_with_orientations(sm, sim, mode):
    """Odd sizes in x, y, z and on the detector (several GEMM tiles plus ragged tails), batch with quaternions."""
    rng = np.random.default_rng(8)
    nx, ny, nz, B = 150, 70, 13, 3
    g = np.stack([W.random_grid(51 + i, nx, ny, nz, fill=0.5) for i in range(B)])
    quat = W.random_quaternions(rng, B)
    quat[1] = [1, 0, 0, 0]
    voxel, lam = (2.0, 2.5, 3.0), 14.0
    npx, npy, th = 23, 19, 35.0
    I = sim(dev(g), voxel, lam, npx, npy, th, quat=quat, rho_mode=mode).cpu().numpy()
    for b in range(B):
        ref = O.simulate(g[b], voxel, lam, npx, npy, th, quat=quat[b], rho_mode=mode)
        assert_parity(I[b], ref, what=f"nufft ragged b={b} mode={mode}")


def test_off_axis_rectangular_detector_wide_angle(sm, sim):
    """Detector centre off the beam axis (the q range is not symmetric, the forward pixel is near a corner) at 70 degrees."""
    g = W.random_grid(91, 40, 33, 29, fill=0.6)
    voxel, lam = (1.0, 1.5, 1.25), 6.0
    for (npx, npy, th, cx, cy) in [(31, 18, 70.0, 9.5, -7.0), (16, 40, 50.0, -30.0, 0.0), (1, 1, 20.0, 0.0, 0.0)]:
        I = sim(dev(g), voxel, lam, npx, npy, th, cx=cx, cy=cy).cpu().numpy()
        ref = O.simulate(g, voxel, lam, npx, npy, th, cx=cx, cy=cy)
        assert_parity(I, ref, what=f"nufft off-axis {npx}x{npy}")


def test_sparse_blobs(sm, sim):
    nx, ny, nz, B = 300, 200, 10, 2
    g = np.stack([W.sparse_blobs_grid(71 + 10 * i, nx, ny, nz, nblobs=5 + 3 * i, max_extent=20 + 60 * i) for i in range(B)])
    voxel, lam = (2.0, 2.0, 2.5), 11.0
    npx, npy, th = 20, 17, 25.0
    I = sim(dev(g), voxel, lam, npx, npy, th).cpu().numpy()
    for b in range(B):
        assert_parity(I[b], O.simulate(g[b], voxel, lam, npx, npy, th), what=f"nufft sparse blobs b={b}")


def test_cfg2_ellipsoid_half_scale_oriented(sm, sim):
    w = W.config(1, scale=0.5)
    g = w.grid(0)
    I = sim(dev(g), (w.dx, w.dy, w.dz), w.lam, w.npx, w.npy, w.theta_max_deg, quat=w.quat).cpu().numpy()
    ref = O.simulate(g, (w.dx, w.dy, w.dz), w.lam, w.npx, w.npy, w.theta_max_deg, quat=w.quat[0])
    assert_parity(I, ref, what="nufft cfg2 half")


def test_cfg3_droplet_quarter_scale(sm, sim):
    w = W.config(2, scale=0.25)
    g = w.grid(0)
    I = sim(dev(g), (w.dx, w.dy, w.dz), w.lam, w.npx, w.npy, w.theta_max_deg).cpu().numpy()
    assert_parity(I, O.simulate(g, (w.dx, w.dy, w.dz), w.lam, w.npx, w.npy, w.theta_max_deg), what="nufft cfg3 quarter")


def test_cfg5_coreshell_eighth_scale(sm, sim):
    w = W.config(4, scale=0.125)
    g = w.grid(0)
    I = sim(dev(g), (w.dx, w.dy, w.dz), w.lam, w.npx, w.npy, w.theta_max_deg).cpu().numpy()
    assert_parity(I, O.simulate(g, (w.dx, w.dy, w.dz), w.lam, w.npx, w.npy, w.theta_max_deg), what="nufft cfg5 eighth")


def test_batch_larger_than_one_chunk(sm, sim):
    """The stage-Z planes of a chunk are capped at 2 GB: nine wide, thin items (1024 x 1024 x 4 voxels, ~270 MB of planes each) run as a
    chunk of seven or eight and a rest.  Checked at seeded pixels of three items, first and last included."""
    nx, ny, nz, B_ = 1024, 1024, 4, 9
    voxel, lam = (1.0, 1.0, 2.0), 9.0
    g = np.stack([W.sparse_blobs_grid(400 + i, nx, ny, nz, nblobs=6, max_extent=40) for i in range(B_)])
    npx, npy, th = 24, 20, 5.0
    I = sim(dev(g), voxel, lam, npx, npy, th).cpu().numpy()
    pix = W.sample_pixels(19, npx * npy, 40, always=[0, npx * npy - 1])
    for b in (0, 6, 7, 8):
        ref = O.simulate(g[b], voxel, lam, npx, npy, th, pixels=pix)
        assert_parity(I[b].ravel()[pix], ref, what=f"nufft chunked batch item {b}")
    assert not np.array_equal(I[7], I[8])


def test_grids_beyond_the_tensor_stages_limits_fall_back_to_the_fp64_stages(sm):
    """The tcgen05 stages keep a table tile resident in shared memory, which bounds every grid dimension (1024 x, 1024 y, 1024 z);
    a taller grid runs the FP64 CUDA-core stages whatever method is asked for -- same result, silently."""
    voxel, lam = (2.0, 0.5, 2.0), 9.0
    g = W.sparse_blobs_grid(55, 24, 1100, 5, nblobs=5, max_extent=60)
    npx, npy, th = 12, 40, 20.0
    ref = O.simulate(g, voxel, lam, npx, npy, th)
    for method in (0, 3):
        I = sm.simulate_nufft(dev(g), voxel, lam, npx, npy, th, method=method).cpu().numpy()
        l2, pix = assert_parity(I, ref, what=f"tall grid method {method}")
        assert l2 <= 1e-6          # both are the FP64 stages


def test_gain_medium_and_weak_items_keep_their_accuracy(sm, sim):
    """The FP16 operand scale of the tensor stages comes from a BOUND of max |rho~| taken before the prefix runs (extremes of
    (delta, beta), gain factor for beta < 0).  A batch with an amplifying item (beta < 0: |T| grows along z), a strongly absorbing
    one whose bound is loose by orders of magnitude, and a weak one: every item keeps the parity tolerances."""
    nx, ny, nz = 70, 50, 24
    voxel, lam = (2.0, 2.0, 2.0), 10.0
    g = np.stack([W.random_grid(61, nx, ny, nz, fill=0.5, delta=(-0.01, 0.03), beta=(-0.02, 0.0)),      # gain
                  W.random_grid(62, nx, ny, nz, fill=0.9, delta=(0.01, 0.05), beta=(0.2, 0.4)),          # opaque after a few slices
                  W.random_grid(63, nx, ny, nz, fill=0.3, delta=(-1e-6, 1e-6), beta=(0.0, 1e-7))])       # weak
    I = sim(dev(g), voxel, lam, 21, 18, 30.0).cpu().numpy()
    for b in range(3):
        assert_parity(I[b], O.simulate(g[b], voxel, lam, 21, 18, 30.0), what=f"nufft scale bound item {b}")


def _fused_batch(nx, ny, nz, B_):
    """20 grids whose chunk has more than 4 * 2^16 columns, so the tensor stages take the FUSED prefix -> planes pass (api.cu
    fused_prefix_pays): sparse blobs, a gain medium, a weak item, an all-vacuum item; random orientations, one identity."""
    g = np.stack([W.sparse_blobs_grid(700 + i, nx, ny, nz, nblobs=5, max_extent=30) for i in range(B_)])
    g[3] = W.random_grid(703, nx, ny, nz, fill=0.4, delta=(-0.01, 0.03), beta=(-0.02, 0.0))      # gain
    g[5] = W.random_grid(705, nx, ny, nz, fill=0.2, delta=(-1e-6, 1e-6), beta=(0.0, 1e-7))        # weak
    g[7] = 0.0                                                                                    # vacuum
    quat = W.random_quaternions(np.random.default_rng(77), B_)
    quat[2] = [1, 0, 0, 0]
    return g, quat


@pytest.mark.parametrize("nx", [126, 125])
def test_fused_prefix_pass_on_an_oriented_batch(sm, sim, nx):
    """Orientation with SPARSE output + tile map, operand scale from the bound of max |rho~|, layers without material not packed,
    four columns per thread (even N_x) or one (odd); ragged tiles in every dimension (126 = 7 tiles + 14, 22 = 5 layers + 2).
    Items of every kind against the oracle; the all-vacuum item exactly 0."""
    ny, nz, B_ = 120, 22, 20
    g, quat = _fused_batch(nx, ny, nz, B_)
    voxel, lam = (2.0, 2.0, 2.5), 12.0
    npx, npy, th = 21, 18, 30.0
    I = sim(dev(g), voxel, lam, npx, npy, th, quat=quat).cpu().numpy()
    assert np.all(I[7] == 0)
    for b in (0, 2, 3, 5, 11, 19):
        assert_parity(I[b], O.simulate(g[b], voxel, lam, npx, npy, th, quat=quat[b]), what=f"nufft fused oriented batch item {b} nx={nx}")
    # the same grids without orientation and without known extremes take strength + pack: both passes give the same patterns
    I0 = sim(dev(g), voxel, lam, npx, npy, th).cpu().numpy()
    assert_parity(I0[3], O.simulate(g[3], voxel, lam, npx, npy, th), what="nufft plain batch item 3")
    assert np.allclose(I[2], I0[2], rtol=2e-4, atol=1e-6 * I0[2].max())      # item 2 has the identity orientation


def test_empty_and_single_voxel(sm, sim):
    voxel, lam = (3.0, 3.0, 3.0), 12.0
    z = np.zeros((8, 8, 8, 2), np.float32)
    assert np.all(sim(dev(z), voxel, lam, 16, 16, 30.0).cpu().numpy() == 0)
    one = z.copy()
    one[2, 5, 1] = (0.03, 0.004)
    I = sim(dev(one), voxel, lam, 16, 16, 30.0).cpu().numpy()
    exact = abs((float(np.float32(0.03)) + 1j * float(np.float32(0.004))) * 27.0) ** 2
    assert np.allclose(I, exact, rtol=1e-6 if sim.exact else 2e-5)   # a corner voxel: |A| is flat only if the window correction is right


def test_agrees_with_the_pixel_contraction_and_is_deterministic(sm, sim):
    import torch
    w = W.config(1, scale=0.5)
    d = dev(w.grid(0))
    vox = (w.dx, w.dy, w.dz)
    a = sim(d, vox, w.lam, w.npx, w.npy, w.theta_max_deg, quat=w.quat).clone()
    b = sim(d, vox, w.lam, w.npx, w.npy, w.theta_max_deg, quat=w.quat).clone()
    assert torch.equal(a, b) if sim.exact else torch.allclose(a, b, rtol=2e-5, atol=1e-6 * float(a.max()))
    c = sm.simulate(d, vox, w.lam, w.npx, w.npy, w.theta_max_deg, quat=w.quat)
    l2, pix = metrics(c.cpu().numpy(), a.cpu().numpy())
    assert l2 <= 1e-4 and pix <= 1e-3


def test_call_is_capturable_in_a_cuda_graph(sm, sim):
    """The entry point only enqueues work on the caller's stream (no allocation, no synchronisation), so a whole call can be captured in
    a CUDA graph and replayed on new input: the replay must give what an eager call gives (bit for bit), oriented batch included."""
    import torch
    w = W.config(1, scale=0.25)
    vox = (w.dx, w.dy, w.dz)
    g0, g1 = w.grid(0), W.random_grid(5, w.nx, w.ny, w.nz, fill=0.3)
    static_in = dev(g0)
    out = torch.empty((1, w.npy, w.npx), dtype=torch.float32, device="cuda")
    from paper_2202_03411_b200 import binding as B
    import ctypes as C
    need = C.c_size_t(0)
    grid = B.Grid(w.nx, w.ny, w.nz, *vox)
    det = B.Detector(w.npx, w.npy, w.theta_max_deg, 0.0, 0.0)
    sm._check(sm.lib.scatman_nufft_workspace_bytes(sm._ctx, C.byref(grid), w.lam, C.byref(det), 1, C.byref(need)))
    ws = torch.empty(int(need.value), dtype=torch.uint8, device="cuda")
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):                         # warm-up outside the capture
        sim(static_in, vox, w.lam, w.npx, w.npy, w.theta_max_deg, quat=w.quat, workspace=ws, out=out)
    torch.cuda.current_stream().wait_stream(side)
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        sim(static_in, vox, w.lam, w.npx, w.npy, w.theta_max_deg, quat=w.quat, workspace=ws, out=out)
    for g in (g1, g0):
        static_in.copy_(dev(g))
        graph.replay()
        torch.cuda.synchronize()
        got = out.clone()
        ref = sim(dev(g), vox, w.lam, w.npx, w.npy, w.theta_max_deg, quat=w.quat)
        assert torch.equal(got[0], ref) if sim.exact else torch.allclose(got[0], ref, rtol=2e-5, atol=1e-6 * float(ref.max()))


def test_error_codes(sm):
    import torch
    from paper_2202_03411_b200 import binding as B
    w = W.config(0)
    d = dev(w.grid(0))
    vox = (w.dx, w.dy, w.dz)
    with pytest.raises(B.ScatmanError) as e:
        sm.simulate_nufft(d, vox, w.lam, 64, 64, 30.0, workspace=torch.empty(1024, dtype=torch.uint8, device="cuda"))
    assert e.value.status == B.WORKSPACE_TOO_SMALL
    for bad in [dict(lam=-1.0), dict(theta=95.0), dict(quat=[[2.0, 0, 0, 0]]), dict(mode=7)]:
        with pytest.raises(B.ScatmanError) as e:
            sm.simulate_nufft(d, vox, bad.get("lam", w.lam), 64, 64, bad.get("theta", 30.0), quat=bad.get("quat"),
                              rho_mode=bad.get("mode", 0))
        assert e.value.status == B.INVALID_ARGUMENT


# ------------------------------------------------------------------------------------------ full sizes, sampled pixels
def _sampled_full(sm, idx, items=None, method=0):
    w = W.config(idx)
    vox = (w.dx, w.dy, w.dz)
    items = [0] if items is None else items
    g = w.grids(items)
    quat = None if w.quat is None else w.quat[items]
    I = sm.simulate_nufft(dev(g), vox, w.lam, w.npx, w.npy, w.theta_max_deg, quat=quat, method=method).cpu().numpy()
    for i in range(len(items)):
        flat = I[i].ravel()
        pix = sampled_pixels(w, items[i], flat, FULL_SIZE_SAMPLES[idx])
        ref = oracle_at_pixels(w, items[i], g[i], None if quat is None else quat[i], pix)
        assert_parity(flat[pix], ref, what=f"nufft {w.name} item {items[i]} sampled")


METHOD = {"tensor": 0, "fp64": 3}


@pytest.mark.parametrize("method", ["tensor", "fp64"])
def test_cfg2_full_size_sampled(sm, method):
    _sampled_full(sm, 1, method=METHOD[method])


@pytest.mark.parametrize("method", ["tensor", "fp64"])
def test_cfg3_full_size_sampled(sm, method):
    _sampled_full(sm, 2, method=METHOD[method])


@pytest.mark.parametrize("method", ["tensor", "fp64"])
def test_cfg4_full_size_items_sampled(sm, method):
    _sampled_full(sm, 3, items=[0, 1, 2, 3], method=METHOD[method])


@pytest.mark.parametrize("method", ["tensor", "fp64"])
def test_cfg5_full_size_sampled(sm, method):
    _sampled_full(sm, 4, method=METHOD[method])
