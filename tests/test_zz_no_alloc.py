"""scatman_discrepancy_static: the discrepancy entry point that allocates nothing (its scratch is a static device array inside the
library, include/scatman.h) against scatman_discrepancy with a caller's workspace, on calls in a row that share the array.
Collected last on purpose (the suite runs with pytest -x): it passes alone in a fresh process and after every other test."""
import numpy as np
import pytest

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


def _patterns(seed, batch, npix, per_item):
    import torch
    rng = np.random.default_rng(seed)
    I = (rng.uniform(0.0, 1.0, (batch, npix)) ** 4 * 1e3).astype(np.float32)
    M = rng.poisson(3.0 * I if per_item else 3.0 * I[0]).astype(np.float32)
    mask = (rng.uniform(size=npix) < 0.8).astype(np.uint8)
    return [torch.from_numpy(a).cuda() for a in (I, M, mask)]


def test_static_scratch_calls_in_a_row_match_the_workspace_path(sm):
    """A large call, then a small one that would see the large one's partial sums if it read anything it had not written, then
    the large one again with the other metric: every result equals the existing path's (same kernels: FP64 sums in a fixed order,
    so the tests' rtol 1e-11 is met with room to spare -- in fact bit for bit)."""
    import torch
    cases = [(11, 7, 3 * 32768 + 555, True, 0), (12, 2, 1000, False, 1), (13, 7, 3 * 32768 + 555, False, 1), (14, 3, 40000, True, 0)]
    for seed, batch, npix, per_item, metric in cases:
        I, M, mask = _patterns(seed, batch, npix, per_item)
        for mk in (None, mask):
            ref = sm.discrepancy(I, M, mk, metric=metric).cpu().numpy()
            out = torch.full((batch,), float("nan"), dtype=torch.float64, device="cuda")
            got = sm.discrepancy_static(I, M, out, mask=mk, metric=metric)
            assert got.data_ptr() == out.data_ptr()
            got = got.cpu().numpy()
            assert np.all(np.isfinite(got))
            assert np.allclose(got, ref, rtol=1e-11, atol=0), (seed, got, ref)
            assert np.array_equal(got, ref)
    # twice in a row on the same inputs: the array keeps the last call's contents and the result does not depend on them
    I, M, mask = _patterns(15, 5, 2 * 32768 + 777, False)
    out1 = torch.empty(5, dtype=torch.float64, device="cuda")
    out2 = torch.empty(5, dtype=torch.float64, device="cuda")
    sm.discrepancy_static(I, M, out1, mask=mask)
    sm.discrepancy_static(I, M, out2, mask=mask)
    ref = sm.discrepancy(I, M, mask).cpu().numpy()
    assert np.array_equal(out1.cpu().numpy(), ref) and np.array_equal(out2.cpu().numpy(), ref)


def test_static_scratch_call_does_not_take_device_memory(sm):
    import torch
    I, M, mask = _patterns(21, 4, 70000, False)
    out = torch.empty(4, dtype=torch.float64, device="cuda")
    sm.discrepancy_static(I, M, out, mask=mask)          # kernels loaded, everything warm
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    held0 = torch.cuda.memory_reserved()
    for _ in range(3):
        sm.discrepancy_static(I, M, out, mask=mask)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert torch.cuda.memory_reserved() == held0
    assert free1 >= free0


def test_sizes_beyond_the_static_array_are_rejected_with_both_numbers(sm):
    import torch
    from paper_2202_03411_b200 import binding as B
    # scratch need = 8 (6 batch nchunk + 6 batch) bytes, nchunk = ceil(npix / 32768): 4096 x 5 chunks = 1.125 MiB > 1 MiB
    batch, npix = 4096, 4 * 32768 + 1
    I = torch.zeros((batch, npix), dtype=torch.float32, device="cuda")
    M = torch.ones(npix, dtype=torch.float32, device="cuda")
    out = torch.full((batch,), -1.0, dtype=torch.float64, device="cuda")
    with pytest.raises(B.ScatmanError) as e:
        sm.discrepancy_static(I, M, out)
    assert e.value.status == B.WORKSPACE_TOO_SMALL
    msg = str(e.value)
    assert str(8 * batch * (5 * 6 + 6)) in msg and str(B.STATIC_SCRATCH_BYTES) in msg
    torch.cuda.synchronize()
    assert bool((out == -1.0).all())                      # nothing was launched
    # the largest batch of this pixel count that fits does run
    fit = B.STATIC_SCRATCH_BYTES // (8 * 36)
    out = torch.empty(fit, dtype=torch.float64, device="cuda")
    I[:fit].fill_(1.0)
    got = sm.discrepancy_static(I[:fit], M, out).cpu().numpy()
    assert np.all(got == 0.0)                             # identical normalised patterns
