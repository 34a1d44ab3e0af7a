"""GPU parity: the CUDA path (through the C ABI) against the FP64 oracle on the same seeded inputs."""
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


@pytest.mark.parametrize("dims", [(91, 93, 5), (92, 90, 6)])
def test_orient_single_grid_whose_slices_are_shared_by_several_blocks(sm, dims):
    """A single grid with few slices of more than 8192 voxels: the bounding-box pass gives every slice to two blocks (odd voxel
    count: scalar loads; even: 16-byte loads).  Material only near two opposite corners of the slice and at the seam between the
    parts, so a part that went unseen would shrink the box and the resampling would drop it."""
    nx, ny, nz = dims
    g = np.zeros((nz, ny, nx, 2), dtype=np.float32)
    rng = np.random.default_rng(17)
    for (ys, xs) in ((slice(10, 13), slice(10, 14)), (slice(ny - 13, ny - 10), slice(nx - 14, nx - 10)), (slice(ny // 2, ny // 2 + 2), slice(10, 12))):
        blk = g[:, ys, xs]
        blk[..., 0] = rng.uniform(0.01, 0.05, blk.shape[:-1])
        blk[..., 1] = rng.uniform(0.001, 0.02, blk.shape[:-1])
    voxel = (1.0, 1.0, 1.0)
    quat = W.random_quaternions(rng, 1)
    quat[0] = (np.cos(0.05), 0.0, 0.0, np.sin(0.05))        # a small turn about z: the material stays inside the grid
    out = sm.orient(dev(g[None]), voxel, quat).cpu().numpy()
    ref = O.orient(g, voxel, quat[0])
    assert np.count_nonzero(ref) > 100
    assert np.allclose(out[0], ref, rtol=2e-7, atol=1e-12)


def test_effective_strength_matches_oracle(sm):
    g = W.random_grid(41, 19, 7, 23, delta=(-0.02, 0.08), beta=(0.0, 0.05))
    voxel, lam = (2.0, 2.0, 3.0), 9.0
    for mode in (0, 1):
        rho = sm.effective_strength(dev(g), voxel, lam, rho_mode=mode).cpu().numpy()
        ref = O.effective_strength(g, voxel, lam, mode) / np.prod(voxel)
        got = rho[..., 0] + 1j * rho[..., 1]
        assert np.max(np.abs(got - ref)) <= 2e-7 * np.max(np.abs(ref))
        assert np.all(got[ref == 0] == 0)


@pytest.mark.parametrize("dims", [(40, 5, 130), (33, 3, 256), (33, 3, 257), (21, 4, 8), (64, 2, 9), (200, 170, 12)])
def test_effective_strength_on_both_column_walks(sm, dims):
    """Grids with few columns cut every column into segments of 8 or 16 slices (one warp of 32 columns per segment, up to 16
    segments, the segment products exchanged through shared memory); more than 32768 columns, nz <= 8 or nz > 256 take one
    thread per column.  Ragged in x, in the last segment and in the segment count; one grid is random (every voxel its own
    factor), one is two homogeneous bodies with vacuum between and inside them (the cached factor carried across the two
    walks of a segment, segments that are all vacuum)."""
    nx, ny, nz = dims
    voxel, lam = (2.0, 2.0, 3.0), 9.0
    g1 = W.random_grid(43 + nz, nx, ny, nz, delta=(-0.02, 0.08), beta=(0.0, 0.05))
    g2 = np.zeros((nz, ny, nx, 2), dtype=np.float32)
    g2[nz // 7: nz // 2, :, 1: nx - 2] = (0.013, 0.004)
    g2[nz // 2 + 1: nz - 1, ny // 2:, nx // 3:] = (-0.007, 0.011)
    g2[nz // 3, :, nx // 2] = 0.0                                     # a hole inside the first body
    for g in (g1, g2):
        for mode in (0, 1):
            rho = sm.effective_strength(dev(g), voxel, lam, rho_mode=mode).cpu().numpy()
            ref = O.effective_strength(g, voxel, lam, mode) / np.prod(voxel)
            got = rho[..., 0] + 1j * rho[..., 1]
            assert np.max(np.abs(got - ref)) <= 2e-7 * np.max(np.abs(ref)), (dims, mode)
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


def test_reuse_tables_is_bit_identical_and_rebuilds_when_anything_changes(sm):
    """SCATMAN_FLAG_REUSE_TABLES skips the q-map and phase-table kernels when grid geometry, lambda, detector, method and
    workspace equal the previous call's -- never otherwise: results with the flag equal results of calls that rebuild everything
    in another workspace (exactly where the route is bitwise reproducible, to FP32 summation order on the tcgen05 routes)."""
    import torch
    from paper_2202_03411_b200 import binding as B
    w = W.config(0)
    vox = (w.dx, w.dy, w.dz)
    g1, g2 = dev(w.grid(0)), dev(W.random_grid(5, w.nx, w.ny, w.nz))
    g3 = dev(np.stack([W.random_grid(6 + i, w.nx, w.ny, w.nz) for i in range(3)]))
    R = B.FLAG_REUSE_TABLES
    k = 2 * np.pi / w.lam
    q1 = torch.from_numpy((np.arange(48) + 0.5 - 24) * (2 * k * np.sin(np.radians(30.0)) / 48)).cuda()
    q2 = (q1 * 0.5).contiguous()
    routes = {
        "pixels": lambda g, lam, th, ws, fl: sm.simulate(g, vox, lam, w.npx, w.npy, th, workspace=ws, flags=fl),
        "pixels_1cta": lambda g, lam, th, ws, fl: sm.simulate(g, vox, lam, w.npx, w.npy, th, workspace=ws, flags=fl | B.FLAG_SINGLE_CTA),
        "nufft": lambda g, lam, th, ws, fl: sm.simulate_nufft(g, vox, lam, w.npx, w.npy, th, workspace=ws, flags=fl),
        "nufft_fp64": lambda g, lam, th, ws, fl: sm.simulate_nufft(g, vox, lam, w.npx, w.npy, th, workspace=ws, flags=fl, method=3),
        "qgrid": lambda g, lam, th, ws, fl: sm.simulate_qgrid(g, vox, lam, q1 if th == 30.0 else q2, q1, workspace=ws, flags=fl),
    }
    for name, run in routes.items():
        ws = torch.empty(1 << 28, dtype=torch.uint8, device="cuda")
        ws2 = torch.empty(1 << 28, dtype=torch.uint8, device="cuda")
        # references first: every one rebuilds its tables (no flag) in another workspace
        ref = {(gi, lam, th): run(g, lam, th, ws2, 0).clone()
               for gi, g in (("g1", g1), ("g2", g2), ("g3", g3)) for lam, th in ((w.lam, 30.0), (0.8 * w.lam, 30.0), (0.8 * w.lam, 25.0))}
        run(g1, w.lam, 30.0, ws2, 0)
        n_full = sm.last_launch_count()
        seq = [(g1, "g1", w.lam, 30.0, ws, True),            # first call on ws after calls on ws2: rebuilt
               (g1, "g1", w.lam, 30.0, ws, False),           # same everything: tables reused
               (g2, "g2", w.lam, 30.0, ws, False),           # new particle, same tables
               (g3, "g3", w.lam, 30.0, ws, False),           # another batch size: same tables (they sit first in the workspace)
               (g2, "g2", 0.8 * w.lam, 30.0, ws, True),      # lambda changed: rebuilt
               (g2, "g2", 0.8 * w.lam, 25.0, ws, True),      # detector / qx changed: rebuilt
               (g2, "g2", 0.8 * w.lam, 25.0, ws2, True),     # other workspace: rebuilt there
               (g2, "g2", 0.8 * w.lam, 25.0, ws, True),      # back: the key is the last call's (ws2) -> rebuilt
               (g1, "g1", 0.8 * w.lam, 25.0, ws, False)]     # and reused again
        for i, (g, gi, lam, th, wsp, rebuilt) in enumerate(seq):
            got = run(g, lam, th, wsp, R)
            n = sm.last_launch_count()
            extra = n - n_full if gi != "g3" else None         # a batch of 3 may launch more kernels per chunk; compare only equals
            want = ref[(gi, lam, th)]
            if name == "nufft_fp64": # CUDA-core FP64 stages: bitwise reproducible, so the comparison is exact
                assert torch.equal(got, want), (name, i)
            else:                    # two MMA issuer threads: FP32 summation order varies from run to run
                assert torch.allclose(got, want, rtol=2e-5, atol=1e-6 * float(want.max())), (name, i)
            if extra is not None:
                assert (n == n_full) == rebuilt and n <= n_full, (name, i, n, n_full)


@pytest.mark.parametrize("route", ["pixels", "qgrid"])
def test_calls_are_capturable_in_a_cuda_graph(sm, route):
    """A whole scatman_simulate / scatman_simulate_qgrid call (oriented batch) only enqueues on the caller's stream, so it can
    be captured in a CUDA graph; a replay on new input in the same buffers equals the eager call within summation order."""
    import torch
    rng = np.random.default_rng(12)
    nx, ny, nz, Bn = 70, 40, 24, 3
    g = [np.stack([W.random_grid(900 + 10 * r + i, nx, ny, nz, fill=0.4) for i in range(Bn)]) for r in range(2)]
    quat = W.random_quaternions(rng, Bn)
    vox, lam = (2.0, 2.0, 2.5), 13.0
    k = 2 * np.pi / lam
    q1 = torch.from_numpy((np.arange(40) + 0.5 - 20) * (2 * k * np.sin(np.radians(25.0)) / 40)).cuda()
    d = dev(g[0])
    ws = torch.empty(1 << 28, dtype=torch.uint8, device="cuda")
    out = torch.empty((Bn, 40, 40), dtype=torch.float32, device="cuda")

    def call(stream=None):
        if route == "pixels":
            sm.simulate(d, vox, lam, 40, 40, 25.0, quat=quat, workspace=ws, out=out, stream=stream)
        else:
            sm.simulate_qgrid(d, vox, lam, q1, q1, quat=quat, workspace=ws, out=out, stream=stream)

    call()
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        call()
    assert sm.last_contraction_ms() == -1.0          # events are not recorded inside a capture
    d.copy_(dev(g[1]))
    graph.replay()
    torch.cuda.synchronize()
    replayed = out.clone()
    call()
    torch.cuda.synchronize()
    assert torch.allclose(replayed, out, rtol=1e-5, atol=1e-6 * float(out.max()))
    assert sm.last_contraction_ms() > 0.0
    ref = O.simulate(g[1][1], vox, lam, 40, 40, 25.0, quat=quat[1]) if route == "pixels" else None
    if ref is not None:
        assert_parity(replayed[1].cpu().numpy(), ref, what="graph replay")


def test_host_entry_points_pipeline_matches_device_paths(sm):
    """scatman_simulate_host / _nufft_host / _qgrid_host on a batch that is cut into several chunks (17 items of 2.1 MB: the
    pipeline cuts batches above 16 MB in two; plus a 1-item call): equal to the device entry points item by item."""
    import torch
    rng = np.random.default_rng(21)
    nx, ny, nz, Bn = 64, 64, 64, 17
    g = np.stack([W.sparse_blobs_grid(700 + i, nx, ny, nz, nblobs=4, max_extent=30) for i in range(Bn)])
    quat = W.random_quaternions(rng, Bn)
    vox, lam = (3.0, 3.0, 3.0), 15.0
    k = 2 * np.pi / lam
    q1 = (np.arange(40) + 0.5 - 20) * (2 * k * np.sin(np.radians(25.0)) / 40)
    h = torch.from_numpy(g).pin_memory()
    for nb in (Bn, 1):
        hh, qq = h[:nb], quat[:nb]
        d = dev(g[:nb])
        I_h = sm.simulate_host(hh, vox, lam, 24, 20, 25.0, quat=qq)
        I_d = sm.simulate(d, vox, lam, 24, 20, 25.0, quat=qq).cpu()
        assert torch.allclose(I_h, I_d, rtol=1e-5, atol=1e-6 * float(I_d.max()))
        N_h = sm.simulate_nufft_host(hh, vox, lam, 24, 20, 25.0, quat=qq)
        N_d = sm.simulate_nufft(d, vox, lam, 24, 20, 25.0, quat=qq).cpu()
        assert torch.allclose(N_h, N_d, rtol=1e-5, atol=1e-6 * float(N_d.max()))
        Q_h = sm.simulate_qgrid_host(hh, vox, lam, q1, q1, quat=qq)
        Q_d = sm.simulate_qgrid(d, vox, lam, torch.from_numpy(q1).cuda(), torch.from_numpy(q1).cuda(), quat=qq).cpu()
        assert torch.allclose(Q_h, Q_d, rtol=1e-5, atol=1e-6 * float(Q_d.max()))
        # a second call reuses the tables kept in the context's arena; new q values rebuild them
        assert torch.allclose(sm.simulate_nufft_host(hh, vox, lam, 24, 20, 25.0, quat=qq), N_h, rtol=1e-5, atol=1e-6 * float(N_d.max()))
        F_h = sm.simulate_nufft_host(hh, vox, lam, 24, 20, 25.0, quat=qq, method=3)      # FP64 stages: exact comparison
        assert torch.equal(F_h, sm.simulate_nufft(d, vox, lam, 24, 20, 25.0, quat=qq, method=3).cpu())
        Q2 = sm.simulate_qgrid_host(hh, vox, lam, 0.5 * q1, q1, quat=qq)
        Q2_d = sm.simulate_qgrid(d, vox, lam, torch.from_numpy(0.5 * q1).cuda(), torch.from_numpy(q1).cuda(), quat=qq).cpu()
        assert torch.allclose(Q2, Q2_d, rtol=1e-5, atol=1e-6 * float(Q2_d.max()))
        for b in {0, nb - 1}:
            ref = O.simulate(g[b], vox, lam, 24, 20, 25.0, quat=quat[b])
            assert_parity(N_h[b].numpy(), ref, what=f"host nufft item {b}")
            assert_parity(I_h[b].numpy(), ref, what=f"host pixels item {b}")


@pytest.mark.parametrize("route", ["pixels", "nufft"])
def test_detector_row_bands_equal_the_full_detector(sm, route):
    """Pixel sharding on one device: the row bands of shard_detector_rows (each a detector of the C ABI with its own npy and
    cy), run back to back and stacked, give the full-detector pattern (ragged band sizes, off-axis detector)."""
    from paper_2202_03411_b200.sharding import shard_detector_rows
    g = W.random_grid(91, 60, 44, 20, fill=0.4)
    vox, lam, npx, npy, th, cx, cy = (2.0, 2.0, 2.5), 12.0, 37, 29, 35.0, 1.5, -2.0
    run = sm.simulate if route == "pixels" else sm.simulate_nufft
    full = run(dev(g), vox, lam, npx, npy, th, cx=cx, cy=cy).cpu().numpy()
    for world in (2, 3):
        bands = []
        for r in range(world):
            y0, y1, cyb = shard_detector_rows(npy, cy, r, world)
            bands.append(run(dev(g), vox, lam, npx, y1 - y0, th, cx=cx, cy=cyb).cpu().numpy())
        stacked = np.concatenate(bands, axis=0)
        assert stacked.shape == full.shape
        assert_parity(stacked, full, l2_tol=2e-6, pix_tol=5e-5, what=f"{route} bands x{world} vs full")
    assert_parity(full, O.simulate(g, vox, lam, npx, npy, th, cx=cx, cy=cy), what=f"{route} off-axis full")


def test_simulate_host_matches_device_path(sm):
    import torch
    w = W.config(0)
    g = w.grid(0)
    h = torch.from_numpy(g).pin_memory()
    I_h = sm.simulate_host(h, (w.dx, w.dy, w.dz), w.lam, w.npx, w.npy, w.theta_max_deg)
    I_d = sm.simulate(dev(g), (w.dx, w.dy, w.dz), w.lam, w.npx, w.npy, w.theta_max_deg).cpu()
    assert torch.equal(I_h[0], I_d)


def test_issuers_stay_in_step_on_mixed_odd_even_kstep_units(sm):
    """The two MMA issuer warps of the contraction share the k-steps of a unit by parity, so units with an odd number of
    live 16-y steps shift which issuer owns a ring slot.  Grid: 40 slices x 3 x-tiles whose live y steps number 1..8 in a
    scrambled order (several hundred k-steps per CTA pair: the 12-slot ring wraps dozens of times, through every
    ownership pattern), checked against the oracle, run to run and between the two tensor kernels."""
    rng = np.random.default_rng(1234)
    nx, ny, nz = 300, 128, 40
    g = np.zeros((nz, ny, nx, 2), np.float32)
    for j in range(nz):
        for xt in range(3):
            nsteps = int(rng.integers(1, 9))
            for ys in rng.choice(8, size=nsteps, replace=False):
                x0 = 128 * xt + int(rng.integers(0, min(128, nx - 128 * xt) - 8))
                y0 = 16 * int(ys) + int(rng.integers(0, 12))
                g[j, y0:y0 + 3, x0:x0 + 6, 0] = rng.uniform(0.01, 0.05)
                g[j, y0:y0 + 3, x0:x0 + 6, 1] = rng.uniform(0.0, 0.01)
    voxel, lam = (2.0, 2.0, 2.0), 12.0
    npx, npy, th = 32, 16, 30.0                     # 512 pixels = 2 CTA pairs
    ref = O.simulate(g, voxel, lam, npx, npy, th)
    outs = {}
    for name in ("tensor", "tensor_1cta"):
        runs = [sm.simulate(dev(g), voxel, lam, npx, npy, th, method=METHODS[name][0], flags=METHODS[name][1]).cpu().numpy()
                for _ in range(6)]
        for r in runs:
            assert_parity(r, ref, what=f"mixed k-steps {name}")
            # Two issuing threads accumulate into one FP32 accumulator in whatever order their MMAs reach the tensor pipe, so
            # runs may differ by FP32 summation order (~1e-7 of the amplitude); a stale operand tile would be orders above.
            assert np.max(np.abs(r - runs[0])) <= 3e-6 * ref.max(), f"{name}: run-to-run difference beyond summation order"
        outs[name] = runs[0]
    assert np.allclose(outs["tensor"], outs["tensor_1cta"], rtol=1e-4, atol=1e-6 * ref.max())


def test_create_destroy_create_runs_every_route():
    """Kernel attributes (dynamic shared memory limits) are set per context creation, not once per process: a second
    context, and one created after the first was destroyed, run every route."""
    import torch
    from paper_2202_03411_b200 import binding as B, build
    build.build()
    w = W.config(0)
    g = w.grid(0)
    vox = (w.dx, w.dy, w.dz)
    k = 2 * np.pi / w.lam
    q1 = torch.from_numpy((np.arange(48) + 0.5 - 24) * (2 * k * np.sin(np.radians(30.0)) / 48)).cuda()
    results = []
    first = B.Scatman(0)
    second = B.Scatman(0)          # two live contexts on one device
    for round_, s in enumerate((first, second, None)):
        if s is None:
            first.close()
            second.close()
            s = B.Scatman(0)       # created after both were destroyed
        r = [s.simulate(dev(g), vox, w.lam, w.npx, w.npy, w.theta_max_deg, method=m, flags=fl).cpu() for m, fl in METHODS.values()]
        r.append(s.simulate_nufft(dev(g), vox, w.lam, w.npx, w.npy, w.theta_max_deg).cpu())
        r.append(s.simulate_qgrid(dev(g), vox, w.lam, q1, q1).cpu())
        r.append(s.simulate_qgrid(dev(g), vox, w.lam, q1, q1, method=B.METHOD_SIMT_TABLE).cpu())
        results.append(r)
        if round_ == 2:
            s.close()
    for r in results[1:]:   # the tcgen05 routes are reproducible to FP32 summation order (two MMA issuer threads), the others bit for bit
        assert all(torch.allclose(a, b, rtol=2e-5, atol=1e-6 * float(a.max())) for a, b in zip(results[0], r))
        assert torch.equal(results[0][2], r[2]) and torch.equal(results[0][3], r[3]) and torch.equal(results[0][-1], r[-1])   # CUDA-core variants


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
def _sampled_full(sm, idx, items=None, method="tensor"):
    w = W.config(idx)
    vox = (w.dx, w.dy, w.dz)
    items = [0] if items is None else items
    g = w.grids(items)
    quat = None if w.quat is None else w.quat[items]
    I = sm.simulate(dev(g), vox, w.lam, w.npx, w.npy, w.theta_max_deg, quat=quat, method=METHODS[method][0],
                    flags=METHODS[method][1]).cpu().numpy()
    for i in range(len(items)):
        flat = I[i].ravel()
        pix = sampled_pixels(w, items[i], flat, FULL_SIZE_SAMPLES[idx])
        ref = oracle_at_pixels(w, items[i], g[i], None if quat is None else quat[i], pix)
        assert_parity(flat[pix], ref, what=f"{w.name} item {items[i]} sampled {method}")


def test_cfg2_full_size_sampled(sm):
    _sampled_full(sm, 1)


def test_cfg3_full_size_sampled(sm):
    _sampled_full(sm, 2)


def test_cfg4_full_size_items_sampled(sm):
    _sampled_full(sm, 3, items=[0, 1, 2, 3, 4, 5, 6, 7, 8])


@pytest.mark.parametrize("method", ["tensor", "tensor_1cta"])
def test_cfg5_full_size_sampled(sm, method):
    """The 298-rad-phase, opaque-core stress case at full size (512^3 on 1024^2), both tensor kernels, 1024 + 9 pixels."""
    _sampled_full(sm, 4, method=method)
