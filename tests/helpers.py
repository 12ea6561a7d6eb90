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


# ------------------------------------------------------------------------------------ oracle eigen stage, many collects
def _eig_worker(args):
    """One collect's oracle eigen stage (a separate process: numpy only, one BLAS thread)."""
    cfg_idx, n = args
    import os
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    if root not in sys.path:
        sys.path.insert(0, root)
    from oracle import bluebild_oracle as oracle
    from paper_2310_09200_b200 import workloads
    try:
        from threadpoolctl import threadpool_limits
        limit = threadpool_limits(limits=1)
    except Exception:
        limit = None
    w = _eig_worker.cache.get(cfg_idx)
    if w is None:
        w = _eig_worker.cache[cfg_idx] = workloads.make_workload(cfg_idx)
    ci = w.collect_inputs(n)
    k = w.cfg.n_eig
    lam, B = oracle.eig_stage(ci["S"], ci["W"], ci["xyz"], ci["wavelength"], min(k + 1, w.cfg.n_beam))
    out = dict(n=n, lam=lam[:k].copy(), lam_next=(float(lam[k]) if lam.size > k else None),
               B=np.asfortranarray(B[:, :k].astype(np.complex64)), xyz=ci["xyz"], wavelength=ci["wavelength"])
    if limit is not None:
        limit.restore_original_limits() if hasattr(limit, "restore_original_limits") else None
    return out


_eig_worker.cache = {}


def eig_inputs_many(cfg_idx, collects, workers=None):
    """Oracle eigen stage (Alg. 1 l.2-4) of many collects, in parallel processes (the oracle itself is called as it
    stands; only the loop over collects is spread). Returns a list of dicts {n, lam (n_eig, desc), lam_next
    (eigenvalue N_eig + 1, for the cut guard), B complex64, xyz, wavelength} in the order of `collects`."""
    import os
    collects = list(collects)
    if workers is None:
        workers = min(len(collects), max(1, (os.cpu_count() or 2)))
    if workers <= 1 or len(collects) < 8:
        return [_eig_worker((cfg_idx, n)) for n in collects]
    import multiprocessing as mp
    with mp.get_context("spawn").Pool(workers) as pool:
        return pool.map(_eig_worker, [(cfg_idx, n) for n in collects], chunksize=max(1, len(collects) // (4 * workers)))


def intervals_from_items(wl_mod, w, items, mid_item):
    """Level edges per DESIGN.md recipe from the eigenvalues of the middle collect and the range over all `items`."""
    lo = min(float(it["lam"][-1]) for it in items)
    hi = max(float(it["lam"][0]) for it in items)
    return wl_mod.choose_intervals(mid_item["lam"], w.cfg.n_levels, lam_max=hi, lam_min=lo)


def assert_well_posed(items, intervals):
    """SURVEY 8(d) harness guard: level images are ill-conditioned (not wrong) when an eigenvalue sits on a level edge
    or when the N_eig cut falls inside a cluster, so the synthetic workloads must keep away from both: no selected
    eigenvalue within 1e-6 (relative) of an edge, and a gap at the cut above 1e-9 lambda_max."""
    edges = np.unique(np.asarray(intervals, dtype=np.float64).ravel())
    for it in items:
        lam = np.asarray(it["lam"], dtype=np.float64)
        rel = np.abs(lam[:, None] - edges[None, :]) / np.maximum(np.abs(edges[None, :]), 1e-300)
        assert rel.min() > 1e-6, "collect %s: eigenvalue within 1e-6 of a level edge" % it.get("n")
        if it.get("lam_next") is not None:
            assert lam[-1] - it["lam_next"] > 1e-9 * lam[0], "collect %s: no gap at the N_eig cut" % it.get("n")


def attach_weights(oracle, items, intervals, filt="lsq"):
    for it in items:
        it["D"] = np.asfortranarray(oracle.level_weights(it["lam"], intervals, filt).astype(np.float32))
    return items


# ------------------------------------------------------------------------------------ achieved-error record
PARITY_RECORDS = []


def record_parity(config, gate, variant, got, ref, collects, pixels):
    """Keeps (rel-L2, max-abs/peak) per level of one parity comparison; tests/conftest.py writes all of them to
    $BB_PARITY_JSON (default gpurun_out/parity_errors.json) at the end of the session."""
    nums = parity_numbers(got, ref)
    PARITY_RECORDS.append(dict(config=config, gate=gate, variant=variant, collects=int(collects), pixels=int(pixels),
                               rel_l2=[float(a) for a, _ in nums], max_abs_over_peak=[float(b) for _, b in nums]))
    return nums


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


# ------------------------------------------------------------------------------------ k-means level validity
def kmeans_partition_check(lam, iv, k, log_domain):
    """Properties that hold for ANY correct solution of PAPER.md:164 under reading Q16 (no reference to how the
    solver works): every positive eigenvalue lies in exactly one closed interval, level 0 is the highest-energy
    one, outer edges are 0 and DBL_MAX, adjacent intervals share their edge and the edge is the midpoint of the
    two adjacent cluster centroids (mapped back from the log domain). Returns the within-cluster sum of squares
    of the induced partition, computed directly from its definition."""
    lam = np.asarray(lam, dtype=np.float64)
    iv = np.asarray(iv, dtype=np.float64)
    pos = lam[lam > 0.0]
    x = np.log(pos) if log_domain else pos
    assert iv.shape == (k, 2)
    member = (pos[None, :] >= iv[:, :1]) & (pos[None, :] <= iv[:, 1:])
    assert np.all(member.sum(axis=0) == 1), "an eigenvalue lies in no level or in two"
    lab = np.argmax(member, axis=0)
    assert iv[0, 1] == np.finfo(np.float64).max and iv[k - 1, 0] == 0.0
    cen = []
    for l in range(k):
        assert np.any(lab == l), "empty level"
        cen.append(float(np.mean(x[lab == l])))
    for l in range(k - 1):
        assert iv[l, 0] == iv[l + 1, 1]                                   # shared edge
        assert pos[lab == l].min() > pos[lab == l + 1].max()              # level 0 = highest energy
        e = 0.5 * (cen[l] + cen[l + 1])
        e = np.exp(e) if log_domain else e
        assert abs(iv[l, 0] - e) <= 1e-9 * abs(e), "edge is not the midpoint of the adjacent centroids"
    return float(sum(np.sum((x[lab == l] - cen[l]) ** 2) for l in range(k)))


def kmeans_brute_contiguous(x_sorted, k):
    """Minimum within-cluster sum of squares over ALL partitions of the sorted values into k contiguous,
    non-empty groups, each group's cost computed from the definition sum (x - mean)^2."""
    import itertools
    x = np.asarray(x_sorted, dtype=np.float64)
    n = len(x)
    best = np.inf
    for cuts in itertools.combinations(range(1, n), k - 1):
        b = (0,) + cuts + (n,)
        sse = 0.0
        for a, c in zip(b[:-1], b[1:]):
            seg = x[a:c]
            sse += float(np.sum((seg - seg.mean()) ** 2))
        best = min(best, sse)
    return best
