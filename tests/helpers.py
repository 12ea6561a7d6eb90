"""Shared by the parity tests: oracle-side preparation of collect_eig inputs and the tolerance."""
import numpy as np

REL_L2_TOL = 1e-4       # north_star: per level, relative L2 <= 1e-4 ...
MAX_ABS_TOL = 1e-3      # ... and max-abs <= 1e-3 x level-image peak, against the fp64 oracle


def eig_inputs(oracle, wl_mod, w, n, intervals):
    """Oracle eigen stage of collect n -> the exact arrays handed to BOTH sides (rounded once)."""
    ci = w.collect_inputs(n)
    lam, B = oracle.eig_stage(ci["S"], ci["W"], ci["xyz"], ci["wavelength"], w.cfg.n_eig)
    D = oracle.level_weights(lam, intervals)
    return dict(B=np.asfortranarray(B.astype(np.complex64)), D=np.asfortranarray(D.astype(np.float32)),
                xyz=ci["xyz"], wavelength=ci["wavelength"], lam=lam, raw=ci)


def intervals_for(oracle, wl_mod, w, collects):
    """Level edges per DESIGN.md recipe, from the oracle's eigenvalues (mid collect + range over `collects`)."""
    c = w.cfg
    ci = w.collect_inputs(w.mid_collect())
    mu, _ = oracle.eig_stage(ci["S"], ci["W"], ci["xyz"], ci["wavelength"], c.n_eig)
    lo, hi = mu[-1], mu[0]
    for n in collects:
        ci = w.collect_inputs(n)
        lam, _ = oracle.eig_stage(ci["S"], ci["W"], ci["xyz"], ci["wavelength"], c.n_eig)
        lo, hi = min(lo, lam[-1]), max(hi, lam[0])
    return wl_mod.choose_intervals(mu, c.n_levels, lam_max=hi, lam_min=lo)


def assert_parity(got, ref, what=""):
    """got: (L, n) float32 from the CUDA path; ref: (L, n) float64 from the oracle."""
    got = np.asarray(got, dtype=np.float64)
    assert got.shape == ref.shape, (got.shape, ref.shape)
    for l in range(ref.shape[0]):
        peak = np.max(np.abs(ref[l]))
        if peak == 0.0:
            assert np.all(got[l] == 0.0), "%s level %d: expected an all-zero image" % (what, l)
            continue
        rel = np.linalg.norm(got[l] - ref[l]) / np.linalg.norm(ref[l])
        mx = np.max(np.abs(got[l] - ref[l])) / peak
        assert rel <= REL_L2_TOL and mx <= MAX_ABS_TOL, "%s level %d: rel-L2 %.3e, max-abs/peak %.3e" % (what, l, rel, mx)
    return True


def parity_numbers(got, ref):
    got = np.asarray(got, dtype=np.float64)
    out = []
    for l in range(ref.shape[0]):
        peak = np.max(np.abs(ref[l])) or 1.0
        out.append((np.linalg.norm(got[l] - ref[l]) / (np.linalg.norm(ref[l]) or 1.0), np.max(np.abs(got[l] - ref[l])) / peak))
    return out
