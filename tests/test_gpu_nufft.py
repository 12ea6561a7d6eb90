"""NUFFT Synthesis on the device (bb_nufft_*, csrc/nufft.cu; Section 2.5 Eq. 17-21, Section 3.4 Eq. 32-36, Alg. 3)
against the oracle's direct baseline-domain double sum (oracle.nufft_direct = Eq. 19 written out, pinned in
tests/test_oracle_pins.py to Standard Synthesis and a hand-typed fringe). The NUFFT is an approximation to a requested
tolerance eps: the gate is north_star's (rel-L2 <= 1e-4, max-abs <= 1e-3 x peak) at eps = 1e-6, and the error must follow eps."""
import numpy as np
import pytest

from helpers import assert_parity, parity_numbers

pytestmark = pytest.mark.gpu


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


def case(seed, n_ant, n_eig, n_levels, n_side, extent, fov, wavelength=2.0, flat=True):
    rng = np.random.default_rng(seed)
    B = ((rng.normal(size=(n_ant, n_eig)) + 1j * rng.normal(size=(n_ant, n_eig))) / np.sqrt(n_ant)).astype(np.complex64)
    D = (rng.uniform(0.5, 3.0, size=(n_levels, n_eig)) * (rng.integers(0, n_levels, size=n_eig)[None, :] == np.arange(n_levels)[:, None]))
    xyz = rng.uniform(-extent, extent, size=(n_ant, 3)) * np.array([1.0, 1.0, 0.02 if flat else 1.0]) + np.array([3.1e5, -2.2e5, 1.0e5])
    g = (np.arange(n_side) - n_side / 2) * (2 * np.sin(fov / 2) / n_side)
    l, m = np.meshgrid(g, g, indexing="xy")
    l, m = l.ravel(), m.ravel()
    c = np.array([0.2, -0.3, np.sqrt(1 - 0.13)])
    e1 = np.cross(c, [0, 0, 1.0]); e1 /= np.linalg.norm(e1)
    e2 = np.cross(c, e1)
    pix = l[:, None] * e1 + m[:, None] * e2 + np.sqrt(1 - l * l - m * m)[:, None] * c
    return dict(B=np.asfortranarray(B), D=np.asfortranarray(D.astype(np.float32)), xyz=np.asfortranarray(xyz),
                pix=np.asfortranarray(pix), wavelength=wavelength)


def test_config1_single_domain(bb, ctx, oracle):
    """Config 1 (16 antennas in a 200 m disk, 32 x 32 pixels over 10 degrees): one transform, no partitioning."""
    from paper_2310_09200_b200 import workloads
    w = workloads.make_workload(1)
    ci = w.collect_inputs(0)
    lam, B = oracle.eig_stage(ci["S"], ci["W"], ci["xyz"], ci["wavelength"], w.cfg.n_eig)
    iv = workloads.choose_intervals(lam, w.cfg.n_levels)
    D = oracle.level_weights(lam, iv)
    pix = w.pixels()
    ref, imag = oracle.nufft_direct(B.astype(np.complex64), D.astype(np.float32), ci["xyz"], pix, ci["wavelength"])
    assert imag <= 1e-9 * np.max(np.abs(ref))
    h = bb.NufftSynthesis(ctx, pix, w.cfg.n_levels, eps=1e-6)
    h.collect_eig(B.astype(np.complex64), D.astype(np.float32), ci["xyz"], ci["wavelength"])
    got = h.images()
    assert h.stats()["n_transforms"] == 1
    assert_parity(got, ref, "NUFFT synthesis config 1")
    # and the same images as the Standard Synthesizer's hot path on the same inputs
    s = bb.StandardSynthesis(ctx, pix, w.cfg.n_levels, "fp32")
    s.collect_eig(B.astype(np.complex64), D.astype(np.float32), ci["xyz"], ci["wavelength"])
    assert_parity(got, s.images().astype(np.float64), "NUFFT vs Standard Synthesis config 1")


@pytest.mark.parametrize("parts", [(1, 1), (2, 1), (1, 3), (4, 2), (3, 5)])
def test_domain_partitioning_gives_the_same_images(bb, ctx, oracle, parts):
    """Eq. 36: splitting the baselines into I cells and the pixels into O cells changes the grids, not the sum.
    40 antennas over +-400 wavelengths, 48 x 48 pixels over 12 degrees, 3 levels, two collects accumulated."""
    c1 = case(11, 40, 9, 3, 48, 800.0, np.deg2rad(12.0))
    c2 = case(12, 40, 9, 3, 48, 800.0, np.deg2rad(12.0))
    ref = oracle.nufft_direct(c1["B"], c1["D"], c1["xyz"], c1["pix"], c1["wavelength"])[0]
    ref = ref + oracle.nufft_direct(c2["B"], c2["D"], c2["xyz"], c1["pix"], c2["wavelength"])[0]
    h = bb.NufftSynthesis(ctx, c1["pix"], 3, eps=1e-6, n_part_in=parts[0], n_part_out=parts[1])
    h.collect_eig(c1["B"], c1["D"], c1["xyz"], c1["wavelength"])
    h.collect_eig(c2["B"], c2["D"], c2["xyz"], c2["wavelength"])
    assert h.stats()["n_transforms"] == 0                   # staged: the transforms run once, over both collects' baselines
    got = h.images()
    assert 1 <= h.stats()["n_transforms"] <= (parts[0] * parts[1]) ** 2
    assert_parity(got, ref, "NUFFT synthesis, partition %s" % (parts,))
    h.collect_eig(c1["B"], c1["D"], c1["xyz"], c1["wavelength"])        # a later collect accumulates into the same images
    ref2 = ref + oracle.nufft_direct(c1["B"], c1["D"], c1["xyz"], c1["pix"], c1["wavelength"])[0]
    assert_parity(h.images(), ref2, "NUFFT synthesis, partition %s, third collect" % (parts,))


def test_error_follows_the_requested_tolerance_and_grids_shrink_with_partitioning(bb, ctx, oracle):
    c = case(21, 32, 6, 2, 40, 600.0, np.deg2rad(10.0), flat=False)        # a genuinely 3-D baseline cloud
    ref = oracle.nufft_direct(c["B"], c["D"], c["xyz"], c["pix"], c["wavelength"])[0]
    errs, grids = [], []
    for eps, parts in ((1e-2, 2), (1e-4, 2), (1e-6, 2), (1e-6, 6)):
        h = bb.NufftSynthesis(ctx, c["pix"], 2, eps=eps, n_part_in=parts, n_part_out=parts)
        h.collect_eig(c["B"], c["D"], c["xyz"], c["wavelength"])
        errs.append(max(r for r, _ in parity_numbers(h.images(), ref)))
        grids.append(h.stats()["max_grid_points"])
        h.close()
    assert errs[0] <= 5e-2 and errs[1] <= 5e-4 and errs[2] <= 2e-5 and errs[3] <= 2e-5, errs
    assert errs[2] < errs[1] < errs[0], errs
    assert grids[3] < grids[2] / 4, grids                                   # Section 3.4.1 / Figure 1c: smaller FFT grids


def test_argument_validation_and_grid_limit(bb, ctx):
    c = case(31, 8, 4, 2, 8, 100.0, np.deg2rad(5.0))
    with pytest.raises(bb.BluebildError):
        bb.NufftSynthesis(ctx, c["pix"], 2, eps=1e-9)
    with pytest.raises(bb.BluebildError):
        bb.NufftSynthesis(ctx, c["pix"], 0)
    big = case(32, 8, 4, 2, 8, 4.0e5, np.deg2rad(40.0))                      # +-200 000 wavelengths over 40 degrees, one cell
    h = bb.NufftSynthesis(ctx, big["pix"], 2, eps=1e-6)
    h.collect_eig(big["B"], big["D"], big["xyz"], big["wavelength"])       # staged only
    with pytest.raises(bb.BluebildError) as e:
        h.images()                                                          # the transforms run here
    assert e.value.code == 7                                                # BB_EUNSUPPORTED: raise the partition counts


def test_algorithm3_from_S_config1_and_filters(bb, ctx, oracle):
    """bb_nufft_collect = Algorithm 3 as printed: Gram, generalized eigendecomposition, N_eig largest,
    intervals and filters, V per level, NUFFT. Reference: the oracle's Algorithm 1 from the same S (the two synthesizers
    compute the same image, Eq. 15/20 vs Eq. 17-19/21, pinned on the CPU side), with one LSQ filter and with (STD, LSQ)."""
    from paper_2310_09200_b200 import workloads
    w = workloads.make_workload(1)
    ci = w.collect_inputs(0)
    pix = w.pixels()
    lam, _ = oracle.eig_stage(ci["S"], ci["W"], ci["xyz"], ci["wavelength"], w.cfg.n_eig)
    iv = workloads.choose_intervals(lam, w.cfg.n_levels)
    ref = oracle.collect(ci["S"], ci["W"], ci["xyz"], ci["wavelength"], w.cfg.n_eig, iv, pix)
    h = bb.NufftSynthesis(ctx, pix, w.cfg.n_levels, eps=1e-6)
    h.collect(ci["S"], ci["W"], ci["xyz"], ci["wavelength"], w.cfg.n_eig, iv)
    h.collect(ci["S"], ci["W"], ci["xyz"], ci["wavelength"], w.cfg.n_eig, iv)          # two time steps staged, one set of transforms
    assert_parity(h.images(), 2 * ref, "Algorithm 3 from S, config 1")
    ref2 = oracle.collect(ci["S"], ci["W"], ci["xyz"], ci["wavelength"], w.cfg.n_eig, iv, pix, filt=("std", "lsq"))
    h2 = bb.NufftSynthesis(ctx, pix, 2 * w.cfg.n_levels, eps=1e-6)
    h2.collect(ci["S"], ci["W"], ci["xyz"], ci["wavelength"], w.cfg.n_eig, iv, filters=["std", "lsq"])
    assert_parity(h2.images(), ref2, "Algorithm 3 from S, config 1, filters (std, lsq)")
    with pytest.raises(bb.BluebildError):                                               # 3 levels cannot hold 2 filters x 2 intervals
        bb.NufftSynthesis(ctx, pix, 3, eps=1e-6).collect(ci["S"], ci["W"], ci["xyz"], ci["wavelength"], w.cfg.n_eig, iv, filters=["std", "lsq"])
    # a Gram matrix that is not positive definite (all antennas at the same place: all ones) is reported by the call itself
    xyz_bad = ci["xyz"].copy()
    xyz_bad[:] = xyz_bad[0]
    with pytest.raises(bb.BluebildError) as e:
        h.collect(ci["S"], ci["W"], np.asfortranarray(xyz_bad), ci["wavelength"], w.cfg.n_eig, iv)
    assert e.value.code == 4
    assert_parity(h.images(), 2 * ref, "images unchanged by the refused collect")


def test_algorithm3_from_S_config3_three_collects(bb, ctx, oracle):
    """Three collects of BASELINE config 3 (epochs 0, 50, 99) through bb_nufft_collect from S, 64 x 64 input cells, against the
    oracle's Algorithm 1 on the every-16th pixel subset (the device glue's eigenpairs, not the oracle's, feed the NUFFT)."""
    from paper_2310_09200_b200 import workloads
    from helpers import intervals_for
    w = workloads.make_workload(3)
    c = w.cfg
    iv = intervals_for(oracle, workloads, w, [0, 50, 99])
    sub = w.sample_pixels(16)
    ref = np.zeros((c.n_levels, sub.size))
    h = bb.NufftSynthesis(ctx, w.pixels(), c.n_levels, eps=1e-5, n_part_in=64, n_part_out=1)
    for n in (0, 50, 99):
        r = w.collect_inputs(n)
        oracle.collect(r["S"], r["W"], r["xyz"], r["wavelength"], c.n_eig, iv, w.pixels(sub), img=ref)
        h.collect(r["S"], r["W"], r["xyz"], r["wavelength"], c.n_eig, iv)
    assert_parity(h.images()[:, sub], ref, "Algorithm 3 from S, config 3")


def test_a_refused_flush_leaves_the_images_untouched(bb, ctx):
    """the grid limit is checked for ALL (input cell, output cell) pairs before any of them is transformed. Seven
    antennas within 50 m and one 570 km away, 2 x 2 input cells: the cells that hold only short baselines need tiny grids,
    the two that also hold the long ones exceed the limit. Whatever the order of the cells, a refused bb_nufft_get must not
    have run a single transform: the images are those of the earlier, good collect, bit for bit, and stay usable."""
    c = case(51, 8, 4, 2, 8, 50.0, np.deg2rad(40.0))
    h = bb.NufftSynthesis(ctx, c["pix"], 2, eps=1e-6, n_part_in=2, n_part_out=1)
    h.collect_eig(c["B"], c["D"], c["xyz"], c["wavelength"])
    good = h.images().copy()
    assert np.max(np.abs(good)) > 0
    for direction in ((1, 1, 0), (1, -1, 0), (1, 0, 1), (0, 1, -1), (1, 1, 1), (-1, 1, 1)):
        before = h.stats()["n_transforms"]
        far = c["xyz"].copy()
        far[7] += 4.0e5 * np.array(direction, dtype=np.float64)
        h.collect_eig(c["B"], c["D"], np.asfortranarray(far), c["wavelength"])     # staged only
        with pytest.raises(bb.BluebildError) as e:
            h.images()
        assert e.value.code == 7
        assert h.stats()["n_transforms"] == before, direction                     # no pair ran
        assert np.array_equal(h.images(), good), direction                         # staged collect dropped, images as before
    h.collect_eig(c["B"], c["D"], c["xyz"], c["wavelength"])                        # and the handle still works
    assert np.allclose(h.images(), 2 * good, rtol=1e-5, atol=1e-6 * np.max(np.abs(good)))


def test_staging_flushes_when_the_array_changes(bb, ctx, oracle):
    """Staged collects share one source list only while n_ant stays the same: a different array runs the pending transforms first."""
    ca = case(41, 12, 5, 2, 24, 300.0, np.deg2rad(8.0))
    cb = case(42, 20, 7, 2, 24, 500.0, np.deg2rad(8.0))
    pix = ca["pix"]
    ref = oracle.nufft_direct(ca["B"], ca["D"], ca["xyz"], pix, ca["wavelength"])[0]
    ref = ref + oracle.nufft_direct(cb["B"], cb["D"], cb["xyz"], pix, cb["wavelength"])[0]
    ref = ref + oracle.nufft_direct(ca["B"], ca["D"], ca["xyz"], pix, ca["wavelength"])[0]
    h = bb.NufftSynthesis(ctx, pix, 2, eps=1e-6, n_part_in=2, n_part_out=2)
    h.collect_eig(ca["B"], ca["D"], ca["xyz"], ca["wavelength"])
    assert h.stats()["n_transforms"] == 0
    h.collect_eig(cb["B"], cb["D"], cb["xyz"], cb["wavelength"])          # 20 antennas: the 12-antenna collect is transformed now
    assert h.stats()["n_transforms"] > 0
    h.collect_eig(ca["B"], ca["D"], ca["xyz"], ca["wavelength"])
    assert_parity(h.images(), ref, "NUFFT synthesis, arrays of 12 / 20 / 12 antennas")


def test_config3_two_collects_partitioned(bb, ctx, oracle):
    """BASELINE config 3 (512 stations to 35 km, 512 x 512 pixels over 15 degrees): unpartitioned, one transform would need a
    2.3e12-point fine grid per level (18 TB); 64 x 64 input cells bring the largest grid to 2e7 points (Section 3.4.1). Two collects
    are staged and transformed together; the whole image is synthesized, the every-16th subset + brightest-source pixels
    are compared with the oracle's Standard Synthesis (= Eq. 19, pinned)."""
    from paper_2310_09200_b200 import workloads
    from helpers import eig_inputs, intervals_for
    w = workloads.make_workload(3)
    iv = intervals_for(oracle, workloads, w, [0, 50])
    items = [eig_inputs(oracle, workloads, w, n, iv) for n in (0, 50)]        # 3 hours apart: the union of two baseline clouds
    plan1 = bb.nufft_plan(w.pixels(), items[0]["xyz"], items[0]["wavelength"], 1e-5, 1, 1)
    plan64 = bb.nufft_plan(w.pixels(), items[0]["xyz"], items[0]["wavelength"], 1e-5, 64, 1)
    assert plan1["max_grid_points"] > 1e12 and plan64["max_grid_points"] < 1e8 and plan64["nonempty_input_cells"] < 0.7
    sub = w.sample_pixels(16)
    ref = np.zeros((w.cfg.n_levels, sub.size))
    for it in items:
        oracle.synth(it["B"], it["D"], it["xyz"], w.pixels(sub), it["wavelength"], img=ref)
    h = bb.NufftSynthesis(ctx, w.pixels(), w.cfg.n_levels, eps=1e-5, n_part_in=64, n_part_out=1)
    for it in items:
        h.collect_eig(it["B"], it["D"], it["xyz"], it["wavelength"])
    got = h.images()
    assert_parity(got[:, sub], ref, "NUFFT synthesis config 3")
