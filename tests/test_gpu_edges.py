"""GPU edge cases of the hot path through the C ABI: ragged tiles, odd eigen counts, many levels,
negative weights, queue overflow, determinism, argument validation."""
import numpy as np
import pytest

from helpers import assert_parity

pytestmark = pytest.mark.gpu

VARIANTS = ["fp32", "tf32x3", "fp16x3"]


@pytest.fixture(scope="module")
def bb():
    import torch
    assert torch.cuda.is_available()
    from paper_2310_09200_b200 import binding
    binding.load_library()
    return binding


@pytest.fixture(scope="module")
def ctx(bb):
    return bb.Context(0)


def random_case(seed, n_ant, n_eig, n_levels, n_pix, extent=3000.0, fov=0.25, signed=False):
    rng = np.random.default_rng(seed)
    B = ((rng.normal(size=(n_ant, n_eig)) + 1j * rng.normal(size=(n_ant, n_eig))) / np.sqrt(n_ant)).astype(np.complex64)
    D = rng.uniform(0.1, 3.0, size=(n_levels, n_eig)) * (rng.random((n_levels, n_eig)) < 0.5)
    if signed:
        D *= rng.choice([-1.0, 1.0], size=D.shape)
    xyz = rng.uniform(-extent, extent, size=(n_ant, 3)) + np.array([6.1e6, -2.3e5, 1.7e6])   # far from the origin
    lm = rng.uniform(-fov, fov, size=(n_pix, 2))
    c = np.array([0.3, -0.5, np.sqrt(1 - 0.34)])
    e1 = np.cross(c, [0, 0, 1.0]); e1 /= np.linalg.norm(e1)
    e2 = np.cross(c, e1)
    pix = lm[:, :1] * e1 + lm[:, 1:] * e2 + np.sqrt(1 - np.sum(lm * lm, axis=1))[:, None] * c
    return dict(B=np.asfortranarray(B), D=np.asfortranarray(D.astype(np.float32)), xyz=np.asfortranarray(xyz),
                pix=np.asfortranarray(pix), wavelength=2.7)


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("n_ant,n_eig,n_levels,n_pix", [
    (1, 1, 1, 1), (16, 8, 2, 1000), (37, 5, 3, 513), (50, 13, 4, 777), (33, 16, 1, 257), (70, 31, 5, 300),
    (64, 33, 2, 129), (40, 64, 8, 255), (48, 65, 3, 200), (20, 130, 2, 150), (24, 7, 32, 100),
    (40, 64, 32, 300)])      # most shared memory: 32 levels x 64 eigenpairs
def test_shapes_ragged_and_padded(bb, ctx, oracle, variant, n_ant, n_eig, n_levels, n_pix):
    c = random_case(1000 + n_ant + n_eig, n_ant, n_eig, n_levels, n_pix, signed=True)
    ref = oracle.synth(c["B"], c["D"], c["xyz"], c["pix"], c["wavelength"])
    s = bb.StandardSynthesis(ctx, c["pix"], n_levels, variant)
    s.collect_eig(c["B"], c["D"], c["xyz"], c["wavelength"])
    got = s.images()
    scale = np.max(np.abs(ref))
    for l in range(n_levels):       # signed weights: measure against the overall peak
        assert np.max(np.abs(got[l] - ref[l])) <= 1e-4 * scale, (l, np.max(np.abs(got[l] - ref[l])) / scale)


@pytest.mark.parametrize("variant", VARIANTS)
def test_leading_dimensions_and_device_pointers(bb, ctx, oracle, variant):
    import torch
    c = random_case(7, 21, 6, 2, 300)
    ref = oracle.synth(c["B"], c["D"], c["xyz"], c["pix"], c["wavelength"])
    # padded leading dimensions on the device side
    def padded(a, dtype, extra):
        rows, cols = a.shape
        t = torch.zeros((cols, rows + extra), dtype=dtype, device="cuda:0")
        t[:, :rows] = torch.from_numpy(np.ascontiguousarray(a.T)).to("cuda:0")
        m = bb.DeviceMatrix(t, rows, cols)
        m.ld = rows + extra
        return m
    s = bb.StandardSynthesis(ctx, padded(c["pix"], torch.float64, 11), 2, variant)
    s.collect_eig(padded(c["B"], torch.complex64, 3), padded(c["D"], torch.float32, 5), padded(c["xyz"], torch.float64, 2),
                  c["wavelength"])
    out = torch.empty(300, dtype=torch.float32, device="cuda:0")
    got = np.stack([s.get(l, out).cpu().numpy().copy() for l in range(2)])
    assert_parity(got, ref, "ld")


@pytest.mark.parametrize("variant", VARIANTS)
def test_queue_overflow_additivity_reset_and_determinism(bb, ctx, oracle, variant):
    c = random_case(11, 18, 8, 2, 400)
    rng = np.random.default_rng(5)
    ref = np.zeros((2, 400))
    s = bb.StandardSynthesis(ctx, c["pix"], 2, variant)
    cases = []
    for e in range(70):             # more collects than the queue holds: several launches accumulate
        B = np.asfortranarray((c["B"] * np.exp(1j * rng.uniform(0, 6.28, size=8))).astype(np.complex64))
        xyz = np.asfortranarray(c["xyz"] + rng.normal(0, 5.0, size=c["xyz"].shape))
        cases.append((B, xyz))
        oracle.synth(B, c["D"], xyz, c["pix"], c["wavelength"], img=ref)
        s.collect_eig(B, c["D"], xyz, c["wavelength"])
    a = s.images()
    assert_parity(a, ref, "70 collects")
    s.reset()
    assert np.all(s.images() == 0)
    for B, xyz in cases:
        s.collect_eig(B, c["D"], xyz, c["wavelength"])
    assert np.array_equal(s.images(), a)        # bit-exact run to run
    # mixed shapes flush the queue and keep accumulating
    c2 = random_case(12, 9, 3, 2, 400)
    s.collect_eig(c2["B"], c2["D"], c2["xyz"], c2["wavelength"])
    oracle.synth(c2["B"], c2["D"], c2["xyz"], c["pix"], c2["wavelength"], img=ref)
    assert_parity(s.images(), ref, "mixed shapes")


@pytest.mark.parametrize("variant", VARIANTS)
def test_zero_weights_give_exact_zero_and_nonnegativity(bb, ctx, variant):
    c = random_case(13, 30, 12, 3, 500)
    c["D"][1, :] = 0
    s = bb.StandardSynthesis(ctx, c["pix"], 3, variant)
    s.collect_eig(c["B"], c["D"], c["xyz"], c["wavelength"])
    img = s.images()
    assert np.all(img[1] == 0) and np.all(img >= 0) and img[0].max() > 0


def test_argument_validation(bb, ctx):
    c = random_case(14, 10, 4, 2, 50)
    with pytest.raises(bb.BluebildError) as e:
        bb.StandardSynthesis(ctx, c["pix"], 0)
    assert e.value.code == 1
    with pytest.raises(bb.BluebildError):
        bb.StandardSynthesis(ctx, c["pix"], 33)
    s = bb.StandardSynthesis(ctx, c["pix"], 2)
    with pytest.raises(bb.BluebildError) as e:
        s.collect_eig(c["B"], c["D"], c["xyz"], -1.0)
    assert e.value.code == 1
    with pytest.raises(bb.BluebildError):
        s.get(2)
    with pytest.raises(bb.BluebildError):        # n_eig > n_beam
        s.collect(np.eye(4, dtype=np.complex64), None, c["xyz"][:4], 2.0, 5, np.array([[0.0, 1.0], [1.0, 2.0]]))
    # a failed call leaves the images unchanged and the handle usable
    assert np.all(s.images() == 0)
    s.collect_eig(c["B"], c["D"], c["xyz"], c["wavelength"])
    assert s.images().max() > 0
    # Gram not positive definite: two coincident antennas
    xyz = np.asfortranarray(np.zeros((4, 3)))
    with pytest.raises(bb.BluebildError) as e:
        s.collect(np.eye(4, dtype=np.complex64), None, xyz, 2.0, 2, np.array([[0.0, 1.0], [1.0, 2.0]]))
    assert e.value.code == 4


def test_empty_image(bb, ctx):
    s = bb.StandardSynthesis(ctx, np.zeros((0, 3)), 1)
    c = random_case(15, 5, 2, 1, 4)
    s.collect_eig(c["B"], c["D"], c["xyz"], c["wavelength"])
    s.flush()
    assert s.get(0).shape == (0,)


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("extent,wavelength,fov", [
    (60000.0, 1.0, 0.35),      # 120 km array at 1 m: |p'| up to 1e5 wavelengths, phases of ~3e4 turns
    (35000.0, 2.5, 0.26),      # config-4-like extremes
    (300.0, 15.0, 1.0)])       # compact array, pixels all over the hemisphere (|r - r_c| ~ 1)
def test_phase_generator_range(bb, ctx, oracle, variant, extent, wavelength, fov):
    """The range reduction (fp64 in the FP32 kernel, integer + tensor-core mini-GEMM in the tensor kernels) must
    hold its precision for very long baselines and for pixel sets far from the field centre."""
    c = random_case(4242, 96, 24, 3, 1500, extent=extent, fov=min(fov, 0.7))
    if fov >= 1.0:             # unit vectors over a wide cap instead of a small tangent patch
        rng = np.random.default_rng(7)
        v = rng.normal(size=(1500, 3)); v[:, 2] = np.abs(v[:, 2]) + 0.2
        c["pix"] = np.asfortranarray(v / np.linalg.norm(v, axis=1, keepdims=True))
    ref = oracle.synth(c["B"], c["D"], c["xyz"], c["pix"], wavelength)
    s = bb.StandardSynthesis(ctx, c["pix"], 3, variant)
    s.collect_eig(c["B"], c["D"], c["xyz"], wavelength)
    assert_parity(s.images(), ref, "%s extent %g" % (variant, extent))


@pytest.mark.parametrize("variant", VARIANTS)
def test_column_magnitudes_span_many_decades(bb, ctx, oracle, variant):
    """Eigenvector columns of very different size (and one all-zero column): the FP16 variant rescales each
    column by a power of two and folds it into the weights; the result must not depend on the magnitudes."""
    c = random_case(99, 80, 12, 2, 700)
    scale = np.array([1e-9, 1e-6, 1e-3, 1.0, 37.0, 1e3, 1e5, 3e-12, 0.0, 2.0, 1e-1, 5e6], dtype=np.float64)
    B = (c["B"].astype(np.complex128) * scale[None, :]).astype(np.complex64)
    D = c["D"].astype(np.float64)
    D[:, scale > 0] /= scale[scale > 0][None, :] ** 2          # keep every column's contribution O(1)
    B, D = np.asfortranarray(B), np.asfortranarray(D.astype(np.float32))
    ref = oracle.synth(B, D, c["xyz"], c["pix"], c["wavelength"])
    s = bb.StandardSynthesis(ctx, c["pix"], 2, variant)
    s.collect_eig(B, D, c["xyz"], c["wavelength"])
    assert_parity(s.images(), ref, variant)


def test_interference_probe(bb, ctx):
    """bb_probe_peak kinds 4-7: fp64 FMA chains slow down under a concurrent tcgen05.mma stream on the same SM
    (the reason the tensor variants reduce phases in integer arithmetic), integer multiply-adds do not."""
    dfma_alone, _ = ctx.probe_peak(4)
    dfma_mma, _ = ctx.probe_peak(5)
    imad_alone, _ = ctx.probe_peak(6)
    imad_mma, _ = ctx.probe_peak(7)
    assert min(dfma_alone, dfma_mma, imad_alone, imad_mma) > 0
    assert dfma_mma < 0.8 * dfma_alone, (dfma_alone, dfma_mma)
    assert imad_mma > 0.8 * imad_alone, (imad_alone, imad_mma)


def test_parameter_estimation_matches_oracle(bb, ctx, oracle):
    """bb_estimate_n_eig / bb_kmeans_levels (device glue) against the oracle: the counts must be
    equal, the level edges equal to rounding (same fp64 expression on both sides)."""
    from paper_2310_09200_b200 import workloads
    w = workloads.make_workload(3)
    lam_all = []
    for n in (0, w.mid_collect(), w.cfg.n_collects - 1):
        ci = w.collect_inputs(n)
        lam, _ = ctx.eig(ci["S"], ci["W"], ci["xyz"], ci["wavelength"], 512, want_B=False)
        lam_all.append(lam)
    lam_all = np.concatenate(lam_all)                       # 1536 eigenvalues pooled from three epochs
    for frac in (0.5, 0.9, 0.99, 1.0):
        assert ctx.estimate_n_eig(lam_all[:512], frac) == oracle.estimate_n_eig(lam_all[:512], frac)
    for logd in (True, False):
        for k in (1, 2, 4, 8):
            got = ctx.kmeans_levels(lam_all, k, logd)
            ref = oracle.kmeans_levels(lam_all, k, logd)
            assert np.allclose(got, ref, rtol=1e-12, atol=0), (logd, k, got, ref)
    rng = np.random.default_rng(3)
    odd = np.concatenate([rng.lognormal(0, 3, 37), [-1.0, 0.0]])
    assert np.allclose(ctx.kmeans_levels(odd, 5, True), oracle.kmeans_levels(odd, 5, True), rtol=1e-12)
    with pytest.raises(bb.BluebildError):
        ctx.kmeans_levels(np.array([1.0, -1.0, 0.0]), 2)
