"""bb_kmeans_levels_static — the level-interval estimate for callers that cannot allocate.

Some users of this library may not call cudaMalloc when they ask for level intervals: an imaging service that fixed
its whole GPU memory layout at start-up, a process in which PyTorch's (or another framework's) pool already owns
nearly all of HBM so that a raw cudaMalloc can fail, or a latency-bound loop for which the device-wide stall of
cudaMalloc / cudaFree is not acceptable. For them the library keeps the k-means scratch tables in a fixed array
inside its own image (about 170 KB per GPU, problems up to 1024 eigenvalues) and takes inputs and outputs as device
pointers. This file checks that entry point against the allocating one, bb_kmeans_levels, which the oracle-based
test in test_gpu_edges.py covers: same kernel, so the intervals must agree to the last bit.

The file is named test_zz_* so that pytest collects it last: under `pytest -x` a failure here hides no other test.
It needs nothing from the tests before it and nothing after it depends on it (own buffers, own stream order).
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def bb():
    import torch
    assert torch.cuda.is_available()
    from paper_2310_09200_b200 import binding
    binding.load_library()
    return binding


def spectra():
    """Eigenvalue lists shaped like the library's use: a decaying positive spectrum with a noise floor and a few
    non-positive values (dropped by the method), at the size limit, at an awkward size, tiny, and with ties."""
    rng = np.random.default_rng(20231009)
    big = np.concatenate([rng.lognormal(2.0, 2.5, 1000), 0.5 + 0.01 * rng.random(20), [-3.0, 0.0, -1e-9, 0.0]])   # n = 1024
    mid = np.concatenate([rng.lognormal(0.0, 3.0, 37), [-1.0, 0.0]])
    tied = np.array([1.0, 1.0, 1.0, 4.0, 4.0, 9.0, 9.0, 9.0, 9.0, 16.0, -2.0, 0.0])
    small = np.arange(1.0, 15.0)
    return [(big, 8, True), (mid, 5, False), (big, 32, False), (tied, 3, True), (small, 2, False), (mid, 7, True)]


def run_static(bb, torch, lam, k, logd, stale=None):
    """One call through the no-allocation entry point; all buffers are torch tensors made by the caller (here)."""
    lam_d = torch.from_numpy(np.ascontiguousarray(lam, dtype=np.float64)).cuda()
    iv_d = torch.full((2, k), -7.0, dtype=torch.float64, device="cuda")     # (2, k) row-major = k x 2 column-major, ld = k
    st_d = torch.full((1,), -1, dtype=torch.int32, device="cuda")
    stream = torch.cuda.current_stream()
    bb.kmeans_levels_static(0, stream.cuda_stream, lam_d.data_ptr(), lam_d.numel(), k, logd, iv_d.data_ptr(), k, st_d.data_ptr())
    stream.synchronize()
    return int(st_d.item()), iv_d.cpu().numpy().T.copy()


def test_static_scratch_kmeans_matches_the_allocating_path(bb):
    import torch
    ctx = bb.Context(0)
    cases = spectra()
    # the existing path first, so that the static calls below run back to back with nothing in between
    want = [ctx.kmeans_levels(lam, k, logd) for lam, k, logd in cases]
    # back-to-back calls that share the scratch array: a large problem, then small ones that would pick up its
    # leftovers if the kernel read a table entry it had not written, then the large one again
    for rep in range(2):
        for (lam, k, logd), ref in zip(cases, want):
            status, got = run_static(bb, torch, lam, k, logd)
            assert status == 0
            assert got.shape == ref.shape == (k, 2)
            assert np.array_equal(got, ref), (rep, lam.size, k, logd, np.max(np.abs(got - ref)))


def test_static_scratch_kmeans_limits_and_errors(bb):
    import torch
    rng = np.random.default_rng(5)
    # at the limit: accepted; one above: refused before anything is launched, outputs untouched
    lam = rng.lognormal(0.0, 2.0, bb.KMEANS_STATIC_MAX_N + 1)
    status, _ = run_static(bb, torch, lam[:-1], 4, True)
    assert status == 0
    lam_d = torch.from_numpy(lam).cuda()
    iv_d = torch.full((2, 4), -7.0, dtype=torch.float64, device="cuda")
    st_d = torch.full((1,), -1, dtype=torch.int32, device="cuda")
    with pytest.raises(bb.BluebildError) as e:
        bb.kmeans_levels_static(0, 0, lam_d.data_ptr(), lam_d.numel(), 4, True, iv_d.data_ptr(), 4, st_d.data_ptr())
    assert e.value.code == 7 and "1024" in str(e.value)        # BB_EUNSUPPORTED, with the limit in the message
    torch.cuda.synchronize()
    assert int(st_d.item()) == -1 and bool((iv_d == -7.0).all())
    # host memory is refused (staging it would need an allocation), as are the usual bad sizes
    host = np.ones(8)
    with pytest.raises(bb.BluebildError) as e:
        bb.kmeans_levels_static(0, 0, host.ctypes.data, 8, 2, True, iv_d.data_ptr(), 4, st_d.data_ptr())
    assert e.value.code == 1
    for n, k, ld in ((0, 1, 1), (8, 9, 9), (8, 2, 1), (8, 33, 33)):
        with pytest.raises(bb.BluebildError) as e:
            bb.kmeans_levels_static(0, 0, lam_d.data_ptr(), n, k, True, iv_d.data_ptr(), ld, st_d.data_ptr())
        assert e.value.code == 1
    # fewer positive eigenvalues than levels: reported through the device status word, intervals left alone
    status, iv = run_static(bb, torch, np.array([1.0, -1.0, 0.0]), 2, True)
    assert status == 1 and np.all(iv == -7.0)
    # and the entry point still works after the refusals
    status, iv = run_static(bb, torch, np.arange(1.0, 15.0), 3, False)
    assert status == 0 and iv[0, 1] == np.finfo(np.float64).max and iv[2, 0] == 0.0
