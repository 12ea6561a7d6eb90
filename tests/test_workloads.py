"""Synthetic workload generators: determinism, shapes, structure (no GPU)."""
import numpy as np
import pytest

from paper_2310_09200_b200 import workloads as wl


@pytest.mark.parametrize("idx", [1, 2, 3])
def test_shapes_and_determinism(idx):
    a, b = wl.make_workload(idx), wl.make_workload(idx)
    c = a.cfg
    ia, ib = a.collect_inputs(a.mid_collect()), b.collect_inputs(b.mid_collect())
    assert ia["S"].shape == (c.n_beam, c.n_beam) and ia["S"].dtype == np.complex64
    assert ia["xyz"].shape == (c.n_ant, 3) and ia["xyz"].dtype == np.float64
    assert np.array_equal(ia["S"], ib["S"]) and np.array_equal(ia["xyz"], ib["xyz"])
    assert np.array_equal(ia["S"], ia["S"].conj().T)                       # exactly Hermitian
    if c.beamformed:
        W = ia["W"]
        assert W.shape == (c.n_ant, c.n_beam) and W.dtype == np.complex64
        nz = np.abs(W) > 0
        assert np.all(nz.sum(axis=1) == 1) and np.all(nz.sum(axis=0) == 48)  # block diagonal
        assert np.allclose(np.abs(W[nz]), 1.0, atol=1e-6)                  # unit modulus
    else:
        assert ia["W"] is None


def test_pixel_grid_unit_vectors_and_centre():
    w = wl.make_workload(3)
    pix = w.pixels()
    assert pix.shape == (512 * 512, 3) and pix.flags.f_contiguous
    assert np.allclose(np.linalg.norm(pix, axis=1), 1.0, atol=1e-14)
    centre = 256 + 512 * 256
    assert np.allclose(pix[centre], w.r_c, atol=1e-15)                     # a pixel sits on r_c
    sub = w.sample_pixels(16)
    assert sub.size >= 32 * 32 and np.all(np.diff(sub) > 0)
    full = w.sample_pixels(16, full_tiles=True)
    assert np.all(np.diff(full) > 0) and np.all(np.isin(sub, full)) and full[-1] == 512 * 512 - 1
    runs = np.split(full, np.where(np.diff(full) != 1)[0] + 1)
    longest = max(runs, key=len)
    assert len(longest) >= 1024 and longest[0] % 256 == 0            # four whole 256-pixel tiles, tile-aligned
    assert set(full[-256:] % 256) == set(range(256))                 # the last tile: every lane


def test_earth_rotation_preserves_geometry():
    w = wl.make_workload(3)
    x0, x1 = w.xyz(0), w.xyz(99)
    d0 = np.linalg.norm(x0[:20, None] - x0[None, :20], axis=-1)
    d1 = np.linalg.norm(x1[:20, None] - x1[None, :20], axis=-1)
    assert np.allclose(d0, d1, atol=1e-7) and not np.allclose(x0, x1)
    assert np.allclose(x0[:, 2], x1[:, 2])                                 # rotation about the pole
    r = np.linalg.norm(w.enu[:, :2], axis=1)
    assert (r < 1000.0).sum() >= 224 and r.max() > 30000.0                 # core + arms


def test_cfg1_sources_on_pixel_centres():
    w = wl.make_workload(1)
    assert np.allclose(w.pixels()[w.src_pixel], w.src_dir, atol=1e-15)
    d = np.linalg.norm(w.enu[:, None, :2] - w.enu[None, :, :2], axis=-1) + 1e9 * np.eye(16)
    assert d.min() >= 5.0 and np.linalg.norm(w.enu[:, :2], axis=1).max() <= 100.0


def test_choose_intervals_structure():
    mu = np.array([74.3, 67.1, 20.2, 0.1033, 0.1030, 0.1021, 0.1015, 0.1010])
    iv = wl.choose_intervals(mu, 2)
    assert iv.shape == (2, 2) and iv[0, 1] == 2 * mu[0] and iv[1, 0] == mu[-1] / 2
    assert iv[0, 0] == iv[1, 1] and 0.1033 < iv[0, 0] < 20.2               # the widest gap
    mu = np.exp(-np.arange(64) / 9.0)
    iv = wl.choose_intervals(mu, 8, lam_max=3.0, lam_min=1e-4)
    assert np.all(iv[:, 0] < iv[:, 1]) and np.all(iv[1:, 1] == iv[:-1, 0])
    counts = [(np.sum((mu >= lo) & (mu <= hi))) for lo, hi in iv]
    assert sum(counts) == 64 and min(counts) >= 1
