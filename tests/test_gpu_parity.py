"""GPU parity: the CUDA path (through the C ABI) against the fp64 oracle, element by element.

Tolerance (north_star): per level, relative L2 <= 1e-4 and max-abs <= 1e-3 x level peak.
Gate G1 feeds the oracle's B and D (rounded once to complex64 / float32) to both sides
(`collect_eig`, the hot path); gate G2 runs the whole `collect` (device fp64 glue + hot path).
"""
import numpy as np
import pytest

from helpers import assert_parity, eig_inputs, intervals_for, parity_numbers

pytestmark = pytest.mark.gpu

VARIANTS = ["fp32", "tf32x3", "fp16x3"]


@pytest.fixture(scope="module")
def bb():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2310_09200_b200 import binding
    binding.load_library()          # raises if the extension is missing: no fallback
    return binding


@pytest.fixture(scope="module")
def ctx(bb):
    return bb.Context(0)


@pytest.fixture(scope="module")
def wl():
    from paper_2310_09200_b200 import workloads
    return workloads


def oracle_images(oracle, items, pix, n_levels):
    img = np.zeros((n_levels, pix.shape[0]))
    for it in items:
        oracle.synth(it["B"], it["D"], it["xyz"], pix, it["wavelength"], img=img)
    return img


# ------------------------------------------------------------------------------------ config 1
@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("device_inputs", [False, True])
def test_cfg1_collect_eig(bb, ctx, wl, oracle, variant, device_inputs):
    w = wl.make_workload(1)
    iv = intervals_for(oracle, wl, w, [0])
    it = eig_inputs(oracle, wl, w, 0, iv)
    pix = w.pixels()
    ref = oracle_images(oracle, [it], pix, 2)
    if device_inputs:
        s = bb.StandardSynthesis(ctx, bb.DeviceMatrix.from_numpy(pix, np.float64), 2, variant)
        s.collect_eig(bb.DeviceMatrix.from_numpy(it["B"], np.complex64), bb.DeviceMatrix.from_numpy(it["D"], np.float32),
                      bb.DeviceMatrix.from_numpy(it["xyz"], np.float64), it["wavelength"])
    else:
        s = bb.StandardSynthesis(ctx, pix, 2, variant)
        s.collect_eig(it["B"], it["D"], it["xyz"], it["wavelength"])
    got = s.images()
    assert_parity(got, ref, "cfg1")
    assert int(np.argmax(got[0])) == int(np.argmax(ref[0]))
    assert s.launches() >= 2


@pytest.mark.parametrize("variant", VARIANTS)
def test_cfg1_full_collect_with_device_glue(bb, ctx, wl, oracle, variant):
    w = wl.make_workload(1)
    iv = intervals_for(oracle, wl, w, [0])
    ci = w.collect_inputs(0)
    pix = w.pixels()
    ref = oracle.collect(ci["S"], ci["W"], ci["xyz"], ci["wavelength"], 8, iv, pix)
    s = bb.StandardSynthesis(ctx, pix, 2, variant)
    s.collect(ci["S"], ci["W"], ci["xyz"], ci["wavelength"], 8, iv)
    assert_parity(s.images(), ref, "cfg1 full collect")
    lam, B = ctx.eig(ci["S"], ci["W"], ci["xyz"], ci["wavelength"], 8)
    lam_ref, _ = oracle.eig_stage(ci["S"], ci["W"], ci["xyz"], ci["wavelength"], 8)
    assert np.allclose(lam, lam_ref, rtol=1e-9)
    t = s.timings()
    assert t["gram_ms"] > 0 and t["eig_ms"] > 0 and t["synth_ms"] > 0


# ------------------------------------------------------------------------------------ config 2
@pytest.mark.parametrize("variant", VARIANTS)
def test_cfg2_lofar_like_three_epochs_full_image(bb, ctx, wl, oracle, variant):
    w = wl.make_workload(2)
    collects = [0, 30, 59]
    iv = intervals_for(oracle, wl, w, collects)
    items = [eig_inputs(oracle, wl, w, n, iv) for n in collects]
    pix = w.pixels()
    ref = oracle_images(oracle, items, pix, 4)
    s = bb.StandardSynthesis(ctx, pix, 4, variant)
    for it in items:
        s.collect_eig(it["B"], it["D"], it["xyz"], it["wavelength"])
    assert_parity(s.images(), ref, "cfg2")
    # G2: whole collect with beamforming W through the device glue, same three epochs
    s2 = bb.StandardSynthesis(ctx, pix, 4, variant)
    for it in items:
        r = it["raw"]
        s2.collect(r["S"], r["W"], r["xyz"], r["wavelength"], 12, iv)
    assert_parity(s2.images(), ref, "cfg2 full collect")


# ------------------------------------------------------------------------------------ config 3
@pytest.mark.parametrize("variant", VARIANTS)
def test_cfg3_ska_low_like_sampled(bb, ctx, wl, oracle, variant):
    w = wl.make_workload(3)
    collects = [0, 50, 99]
    iv = intervals_for(oracle, wl, w, collects)
    items = [eig_inputs(oracle, wl, w, n, iv) for n in collects]
    sub = w.sample_pixels(8)
    ref = oracle_images(oracle, items, w.pixels(sub), 4)
    s = bb.StandardSynthesis(ctx, w.pixels(), 4, variant)      # full 512^2 image on the GPU
    for it in items:
        s.collect_eig(it["B"], it["D"], it["xyz"], it["wavelength"])
    assert_parity(s.images()[:, sub], ref, "cfg3")
    s2 = bb.StandardSynthesis(ctx, w.pixels(sub), 4, variant)  # G2 on the pixel subset
    for it in items:
        r = it["raw"]
        s2.collect(r["S"], r["W"], r["xyz"], r["wavelength"], 32, iv)
    assert_parity(s2.images(), ref, "cfg3 full collect")


# ------------------------------------------------------------------------------------ config 4 (bench workload, full size)
@pytest.mark.parametrize("variant", VARIANTS)
def test_cfg4_full_size_bench_configuration(bb, ctx, wl, oracle, variant):
    w = wl.make_workload(4)
    collects = list(range(20))
    iv = intervals_for(oracle, wl, w, collects)
    items = [eig_inputs(oracle, wl, w, n, iv) for n in collects]
    sub = w.sample_pixels(32)
    ref = oracle_images(oracle, items, w.pixels(sub), 8)
    s = bb.StandardSynthesis(ctx, w.pixels(), 8, variant)      # full 1024^2, all 20 epochs, one launch
    for it in items:
        s.collect_eig(it["B"], it["D"], it["xyz"], it["wavelength"])
    got = s.images()
    assert_parity(got[:, sub], ref, "cfg4")
    assert np.all(got >= 0)                                    # invariant I2 holds bit-for-bit
    print("cfg4 parity (rel-L2, max-abs/peak) per level:", parity_numbers(got[:, sub], ref))


# ------------------------------------------------------------------------------------ config 5 (reduced epochs, full image)
@pytest.mark.parametrize("variant", VARIANTS)
def test_cfg5_multichannel_two_epochs_full_image(bb, ctx, wl, oracle, variant):
    w = wl.make_workload(5)
    collects = [n for t in (0, 49) for n in range(t * 16, t * 16 + 16, 5)]   # channels 0,5,10,15 of 2 epochs
    iv = intervals_for(oracle, wl, w, collects)
    items = [eig_inputs(oracle, wl, w, n, iv) for n in collects]
    sub = w.sample_pixels(64)
    ref = oracle_images(oracle, items, w.pixels(sub), 8)
    s = bb.StandardSynthesis(ctx, w.pixels(), 8, variant)      # full 2048^2
    for it in items:
        s.collect_eig(it["B"], it["D"], it["xyz"], it["wavelength"])
    assert_parity(s.images()[:, sub], ref, "cfg5")


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("gram", ["sinc", "identity"])
def test_collect_ex_filters_and_gram_mode(bb, ctx, oracle, variant, gram):
    """N_f = 2 filters (STD, LSQ) x 2 intervals through bb_synth_collect_ex, with the sinc
    Gram and with G := I (dirty-image eigendecomposition), against the oracle's Algorithm 1."""
    from paper_2310_09200_b200 import workloads
    w = workloads.make_workload(1)
    ci = w.collect_inputs(0)
    pix = w.pixels()
    lam, _ = oracle.eig_stage(ci["S"], ci["W"], ci["xyz"], ci["wavelength"], w.cfg.n_eig, gram_identity=(gram == "identity"))
    iv = workloads.choose_intervals(lam, 2)
    ref = oracle.collect(ci["S"], ci["W"], ci["xyz"], ci["wavelength"], w.cfg.n_eig, iv, pix, filt=("std", "lsq"),
                         gram_identity=(gram == "identity"))
    s = bb.StandardSynthesis(ctx, pix, 4, variant)
    s.collect(ci["S"], ci["W"], ci["xyz"], ci["wavelength"], w.cfg.n_eig, iv, filters=["std", "lsq"], gram=gram)
    assert_parity(s.images(), ref, "%s %s" % (variant, gram))
    # wrong level count for the filter list is rejected and leaves the images untouched
    s3 = bb.StandardSynthesis(ctx, pix, 3, variant)
    with pytest.raises(bb.BluebildError):
        s3.collect(ci["S"], ci["W"], ci["xyz"], ci["wavelength"], w.cfg.n_eig, iv, filters=["std", "lsq"])
    assert not s3.images().any()


# ------------------------------------------------------------------------------------ batched glue
@pytest.mark.parametrize("cfg_idx,collects,n_sub", [(2, [0, 20, 40, 59], 4), (3, list(range(0, 100, 5)), 16)])
def test_collect_batch_matches_oracle(bb, ctx, wl, oracle, cfg_idx, collects, n_sub):
    """bb_synth_collect_batch (batched Gram / Cholesky / XsyevBatched, 16 eigenproblems per solve) against the
    oracle's Algorithm 1 run collect by collect: beamformed with a W per epoch (config 2) and 20 epochs in two
    batched groups with W = I (config 3), on a pixel subset."""
    w = wl.make_workload(cfg_idx)
    c = w.cfg
    iv = intervals_for(oracle, wl, w, collects[:3])
    raws = [w.collect_inputs(n) for n in collects]
    sub = w.sample_pixels(n_sub)
    pix = w.pixels(sub)
    ref = np.zeros((c.n_levels, pix.shape[0]))
    for r in raws:
        oracle.collect(r["S"], r["W"], r["xyz"], r["wavelength"], c.n_eig, iv, pix, img=ref)
    S = np.stack([r["S"] for r in raws])
    X = np.stack([r["xyz"] for r in raws])
    W = None if raws[0]["W"] is None else np.stack([r["W"] for r in raws])
    s = bb.StandardSynthesis(ctx, pix, c.n_levels, "fp16x3")
    s.collect_batch(S, W, X, [r["wavelength"] for r in raws], c.n_eig, iv)
    assert_parity(s.images(), ref, "cfg%d batch" % cfg_idx)
    t = s.timings()
    assert t["eig_ms"] > 0 and t["gram_ms"] > 0
