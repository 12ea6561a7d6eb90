"""GPU parity: the CUDA path (through the C ABI) against the fp64 oracle, element by element.

Tolerance (north_star): per level, relative L2 <= 1e-4 and max-abs <= 1e-3 x level peak.
Gate G1 feeds the oracle's B and D (rounded once to complex64 / float32) to both sides
(`collect_eig`, the hot path); gate G2 runs the whole `collect` (device fp64 glue + hot path).
"""
import numpy as np
import pytest

from helpers import assert_parity, eig_inputs, intervals_for, parity_numbers

pytestmark = pytest.mark.gpu

VARIANTS = ["fp32", "tf32x3", "fp16x3", "fp16fp8"]


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


# ------------------------------------------------------------------------------------ configs 2-5, ALL collects
# SURVEY 8(d) "Oracle timing beside it": full image for config 2, the every-8th / every-16th pixel subset
# (+ the pixels nearest the 10 brightest sources + 1280 consecutive pixels: whole tiles) for configs 3, 4 and 5 — over EVERY collect of the config, because
# every time step and band accumulates into the same images. The oracle side (eigen stage of
# each collect, then Alg. 2) is computed once per config and shared by the three variants.
_FULL = {2: dict(stride=None), 3: dict(stride=8), 4: dict(stride=16), 5: dict(stride=16)}
_cache = {}


def oracle_case(oracle, wl, cfg_idx):
    """-> dict(w, items [all collects: B, D, lam, xyz, wavelength], iv, sub (pixel indices or None), ref (L, n))."""
    if cfg_idx in _cache:
        return _cache[cfg_idx]
    from helpers import assert_well_posed, attach_weights, eig_inputs_many, intervals_from_items
    w = wl.make_workload(cfg_idx)
    c = w.cfg
    items = eig_inputs_many(cfg_idx, range(c.n_collects))
    iv = intervals_from_items(wl, w, items, items[w.mid_collect()])
    assert_well_posed(items, iv)
    attach_weights(oracle, items, iv)
    stride = _FULL[cfg_idx]["stride"]
    # + four whole consecutive 256-pixel tiles and the image's last tile: every thread / TMEM lane of a tile at full size
    sub = None if stride is None else w.sample_pixels(stride, full_tiles=True)
    ref = oracle_images(oracle, items, w.pixels(sub), c.n_levels)
    _cache[cfg_idx] = dict(w=w, items=items, iv=iv, sub=sub, ref=ref)
    return _cache[cfg_idx]


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("cfg_idx", [2, 3, 4, 5])
def test_G1_all_collects(bb, ctx, wl, oracle, cfg_idx, variant):
    """Hot path (collect_eig, the oracle's B and D) over all collects of the config, full-size image on the GPU, in
    the launch configuration bench.py times; compared on the oracle's pixels."""
    from helpers import record_parity
    case = oracle_case(oracle, wl, cfg_idx)
    w, items, sub, ref = case["w"], case["items"], case["sub"], case["ref"]
    s = bb.StandardSynthesis(ctx, w.pixels(), w.cfg.n_levels, variant)
    for it in items:
        s.collect_eig(it["B"], it["D"], it["xyz"], it["wavelength"])
    got = s.images()
    assert np.all(got >= 0)                                    # invariant I2 (all D >= 0) holds bit-for-bit
    got = got if sub is None else got[:, sub]
    record_parity(cfg_idx, "G1 collect_eig", variant, got, ref, len(items), ref.shape[1])
    assert_parity(got, ref, "cfg%d G1 %s" % (cfg_idx, variant))
    s.close()


# config 5: 9 epochs x 16 channels = 144 collects = one FULL glue group of 128 staged collects + a partial one of 16
_G2_COLLECTS = {2: None, 3: None, 4: None, 5: [n for t in (0, 6, 12, 18, 24, 30, 36, 42, 49) for n in range(t * 16, t * 16 + 16)]}


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("api", ["collect", "collect_batch"])
@pytest.mark.parametrize("cfg_idx", [2, 3, 4, 5])
def test_G2_device_glue(bb, ctx, wl, oracle, cfg_idx, api, variant):
    """Algorithm 1 end to end on the device (batched fp64 Gram / Cholesky / eigensolve, level weights, hot path)
    from S, W, xyz and the intervals, through bb_synth_collect and bb_synth_collect_batch, on the oracle's pixel
    subset: all collects of configs 2-4, 9 epochs x 16 channels of config 5 (a full 128-collect glue group and a partial one)."""
    from helpers import record_parity
    case = oracle_case(oracle, wl, cfg_idx)
    w, iv, sub = case["w"], case["iv"], case["sub"]
    c = w.cfg
    pix = w.pixels(sub)
    collects = _G2_COLLECTS[cfg_idx]
    if collects is None:
        collects, ref = list(range(c.n_collects)), case["ref"]
    else:
        key = ("g2ref", cfg_idx)
        if key not in _cache:
            _cache[key] = oracle_images(oracle, [case["items"][n] for n in collects], pix, c.n_levels)
        ref = _cache[key]
    s = bb.StandardSynthesis(ctx, pix, c.n_levels, variant)
    rkey = ("raw", cfg_idx)
    if rkey not in _cache:
        _cache[rkey] = {n: w.collect_inputs(n) for n in collects}
    raw = _cache[rkey]
    if api == "collect":
        for n in collects:
            r = raw[n]
            s.collect(r["S"], r["W"], r["xyz"], r["wavelength"], c.n_eig, iv)
    else:
        for k in range(0, len(collects), 24):                 # several calls, groups that do not align with the queue
            raws = [raw[n] for n in collects[k:k + 24]]
            S = np.stack([r["S"] for r in raws])
            X = np.stack([r["xyz"] for r in raws])
            W = None if raws[0]["W"] is None else np.stack([r["W"] for r in raws])
            s.collect_batch(S, W, X, [r["wavelength"] for r in raws], c.n_eig, iv)
    got = s.images()
    s.status()
    record_parity(cfg_idx, "G2 " + api, variant, got, ref, len(collects), ref.shape[1])
    assert_parity(got, ref, "cfg%d G2 %s %s" % (cfg_idx, api, variant))
    t = s.timings()
    assert t["eig_ms"] > 0 and t["gram_ms"] > 0 and t["synth_ms"] > 0
    s.close()


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


# ------------------------------------------------------------------------------------ uniform weighting (Section 3.5)
@pytest.mark.parametrize("variant", ["fp32", "fp16fp8"])
@pytest.mark.parametrize("cfg_idx,collects,stride", [(1, [0], None), (3, [0, 50, 99], 16)])
def test_uniform_weighting_matches_oracle(bb, ctx, wl, oracle, cfg_idx, collects, stride, variant):
    """bb_uvgrid_* + bb_synth_set_weighting against the oracle's Section 3.5: density on the 1/FoV uv grid over the
    given collects, S_pq divided by the density of its cell before the eigendecomposition (weighted matrices may be
    indefinite: the level edges are placed between signed eigenvalues)."""
    from helpers import assert_well_posed, record_parity
    w = wl.make_workload(cfg_idx)
    c = w.cfg
    cell = 1.0 / (c.n_side * w.pix_step)                          # 1 / FoV, the extent of the image in direction cosines
    raws = [w.collect_inputs(n) for n in collects]
    dens = oracle.uv_density([(r["xyz"], r["wavelength"]) for r in raws], w.e_l, w.e_m, cell)
    wts = [oracle.uniform_weights(r["xyz"], r["wavelength"], w.e_l, w.e_m, cell, dens) for r in raws]
    items = []
    for n, r, wt in zip(collects, raws, wts):
        lam, _ = oracle.eig_stage(r["S"], None, r["xyz"], r["wavelength"], min(c.n_eig + 1, c.n_beam), vis_weights=wt)
        items.append(dict(n=n, lam=lam[:c.n_eig], lam_next=float(lam[c.n_eig]) if lam.size > c.n_eig else None))
    mid = items[len(items) // 2]["lam"]
    L = c.n_levels
    edges = [0.5 * (mid[(q * c.n_eig) // L - 1] + mid[(q * c.n_eig) // L]) for q in range(1, L)]
    bounds = [1e30] + edges + [-1e30]
    iv = np.array([[bounds[l + 1], bounds[l]] for l in range(L)])
    assert_well_posed(items, iv[:, :][np.abs(iv) < 1e29].reshape(-1, 1) if L > 1 else np.zeros((0, 1)))
    pix = w.pixels(None if stride is None else w.sample_pixels(stride))
    ref = np.zeros((L, pix.shape[0]))
    for r, wt in zip(raws, wts):
        oracle.collect(r["S"], None, r["xyz"], r["wavelength"], c.n_eig, iv, pix, img=ref, vis_weights=wt)
    max_uv = max(np.max(np.abs(r["xyz"] @ e)) for r in raws for e in (w.e_l, w.e_m)) * 2.0 / min(r["wavelength"] for r in raws)
    grid = bb.UVGrid(ctx, cell, w.e_l, w.e_m, max_uv)
    for r in raws:
        grid.add(r["xyz"], r["wavelength"])
    s = bb.StandardSynthesis(ctx, pix, L, variant)
    s.set_weighting(grid)
    for r in raws:
        s.collect(r["S"], None, r["xyz"], r["wavelength"], c.n_eig, iv)
    got = s.images()
    s.status()
    record_parity(cfg_idx, "G2 uniform weighting", variant, got, ref, len(collects), ref.shape[1])
    for l in range(L):                                            # signed eigenvalues: measure against the level's own peak
        peak = np.max(np.abs(ref[l]))
        assert np.linalg.norm(got[l] - ref[l]) <= 1e-4 * np.linalg.norm(ref[l]) and np.max(np.abs(got[l] - ref[l])) <= 1e-3 * peak, (l,)
    # natural weighting again on the same handle: different images
    s.set_weighting(None)
    s.reset()
    for r in raws:
        s.collect(r["S"], None, r["xyz"], r["wavelength"], c.n_eig, iv)
    assert np.max(np.abs(s.images() - got)) > 1e-3 * np.max(np.abs(got))
    s.close()
    grid.close()
