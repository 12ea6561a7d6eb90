"""Host logic of the collect-range split (csrc/kernels_tc.cu bb_collect_split, through the host-only ABI query
bb_plan_collect_split; no GPU needed): which launches are split, and that a split always pays in wave efficiency."""
import numpy as np
import pytest

from paper_2310_09200_b200 import binding

SM = 148
# (variant, pixels per CTA, resident CTAs per SM) as the kernels are built: tensor variants 256 / 1; FP32 depends on n_eig
TENSOR = ("tf32x3", "fp16x3", "fp16fp8")


def eff(tiles, split, slots):
    ctas = tiles * split
    return ctas / (-(-ctas // slots) * slots)


def test_baseline_configs():
    shapes = {1: (32 * 32, 16, 8, 2, 1), 2: (256 * 256, 1776, 12, 4, 60), 3: (512 * 512, 512, 32, 4, 100),
              4: (1024 * 1024, 512, 64, 8, 20), 5: (2048 * 2048, 512, 64, 8, 128)}
    for v in TENSOR:
        got = {k: binding.plan_collect_split(v, *s) for k, s in shapes.items()}
        assert got == {1: 1, 2: 4, 3: 1, 4: 1, 5: 1}, (v, got)      # config 2: 256 tiles x 4 = 6.92 waves of 148 SMs
    got = {k: binding.plan_collect_split("fp32", *s) for k, s in shapes.items()}
    assert got[1] == 1 and got[2] == 2 and got[4] == 1 and got[5] == 1, got


def test_split_rules():
    rng = np.random.default_rng(5)
    for _ in range(400):
        n_pix = int(rng.integers(1, 600_000)); n_col = int(rng.integers(1, 129)); sm = int(rng.choice([148, 132, 80, 16]))
        s = binding.plan_collect_split("fp16fp8", n_pix, 64, 16, 2, n_col, sm)
        tiles = -(-n_pix // 256)
        assert 1 <= s <= 8
        if s > 1:
            assert n_col // s >= 4                                   # every range keeps at least 4 collects
            assert (s - 1) * -(-n_col // s) < n_col, (n_col, s)      # ... and, with ranges of ceil(n / s), the LAST one is not empty
            assert eff(tiles, s, sm) > eff(tiles, 1, sm) + 0.05      # a split must pay
            assert eff(tiles, 1, sm) < 0.95
        if n_col < 8 or eff(tiles, 1, sm) >= 0.95:
            assert s == 1
    assert binding.plan_collect_split("fp16fp8", 0, 64, 16, 2, 10, 148) == 0      # invalid arguments
    # ranges are ceil(n / s) collects long: 25 collects in 6 ranges of 5, or 33 in 8 ranges of 5, would leave trailing
    # ranges empty (or of negative length) whose CTAs address weights beyond the queued collects: never chosen
    for variant in TENSOR + ("fp32",):
        for n_col in range(1, 129):
            for n_pix in (256 * 25, 256 * 19, 256 * 37, 256 * 150, 65536, 40000):
                for sm in (148, 132, 16):
                    s = binding.plan_collect_split(variant, n_pix, 64, 16, 2, n_col, sm)
                    assert s >= 1 and (s - 1) * -(-n_col // s) < n_col, (variant, n_col, n_pix, sm, s)


def test_nufft_plan_domain_partitioning():
    """bb_nufft_plan (host only): Section 3.4.1 — partitioning the baselines shrinks the FFT grids by orders of magnitude and
    leaves a growing share of the partition cells empty (Figure 1c-d), on the synthetic SKA-Low layout of config 3."""
    from paper_2310_09200_b200 import workloads
    w1 = workloads.make_workload(1)
    p = binding.nufft_plan(w1.pixels(), w1.xyz(0), 2.0, 1e-6, 1, 1)
    assert p["n_transforms"] == 1 and p["max_grid_points"] < 1e6 and p["nonempty_input_cells"] == 1.0
    w3 = workloads.make_workload(3)
    pix, xyz = w3.pixels(), w3.xyz(0)
    prev = None
    for parts in (1, 4, 16, 64):
        p = binding.nufft_plan(pix, xyz, 3.0, 1e-4, parts, 1)
        assert p["n_transforms"] <= parts * parts
        if prev is not None:
            assert p["max_grid_points"] < prev["max_grid_points"] / 8 and p["nonempty_input_cells"] <= prev["nonempty_input_cells"]
        prev = p
    assert binding.nufft_plan(pix, xyz, 3.0, 1e-4, 1, 1)["max_grid_points"] > 1e12          # 18 TB per level: does not fit anywhere
    assert prev["max_grid_points"] < 5e7 and 0.3 < prev["nonempty_input_cells"] < 0.7
    # output partitioning multiplies the transforms and shrinks the grids further
    q = binding.nufft_plan(pix, xyz, 3.0, 1e-4, 16, 4)
    assert q["n_transforms"] == 16 * binding.nufft_plan(pix, xyz, 3.0, 1e-4, 16, 1)["n_transforms"]
    assert q["max_grid_points"] < binding.nufft_plan(pix, xyz, 3.0, 1e-4, 16, 1)["max_grid_points"] / 4
    with pytest.raises(binding.BluebildError):
        binding.nufft_plan(pix, xyz, 3.0, 1e-9, 1, 1)
