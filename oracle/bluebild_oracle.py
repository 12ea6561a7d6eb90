"""ORACLE — TEST INFRASTRUCTURE, NOT PRODUCT CODE.

A plain, slow, fp64 CPU implementation of the Bluebild Standard Synthesis path, written from
/root/reference/PAPER.md (arXiv 2310.09200) and from nothing else. Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may
import it. It shares no code with ``paper_2310_09200_b200`` (the CUDA path) and never imports it.

Functions and the passage each follows:

===================  ==========================================================================
``gram``             Eq. 11 Psi_pq = sinc(2 ||b_pq||), b = (f/c)(x_p - x_q), sinc
                     normalized; Eq. 24 G = W^H Psi W.
``geig``             Eq. 13 V alpha = lambda G alpha, solved as G = L L^H,
                     C = L^-1 S L^-H, Hermitian eig of C, alpha = L^-H Q  (so alpha^H G alpha = I).
``select``           Alg. 1 line 4: keep the N_eig largest eigenvalues.
``level_weights``    Alg. 1 lines 7-8: D[l,k] = d_f(lambda_k) if lambda_k in
                     [min_l, max_l] else 0; LSQ filter d = lambda, STD filter d = 1.
``synth``            Alg. 2 + Alg. 1 line 9 (C++: oracle/synth.cpp).
``brute``            the literal definition, tiny inputs (C++: oracle/brute.cpp).
``collect``          Alg. 1 end to end.
``estimate_n_eig``   PAPER.md:152: minimum number of leading eigenvalues holding a given fraction
                     of the total (positive) energy.
``kmeans_levels``    PAPER.md:164: k-means clustering of the eigenvalues into energy levels; in one
                     dimension the global optimum is found by dynamic programming over the sorted
                     values (readings in DESIGN.md Q16).
``gram_corrected_visibilities``  Eq. 17 / Eq. 21: V'_l = A Lambda_l A^H per level.
``nufft_direct``     Eq. 18-19: the NUFFT-synthesis image as the literal double sum over
                     baselines and pixels (what a type-3 NUFFT approximates); tiny inputs only.
``uv_density``       Section 3.5 "uniform" weighting: the sampling density function on a
``uniform_weights``  uv grid of cell 1/FoV; "each visibility is then weighted with the inverse of its
                     sampling density" before the eigendecomposition (readings in DESIGN.md Q17).
===================  ==========================================================================

Library primitives used as steps: numpy.linalg.cholesky, numpy.linalg.eigh, numpy.linalg.solve,
numpy.sinc. Pins: tests/test_oracle_pins.py (P1-P6, I1-I8 of DESIGN.md). Parity unpinned: none.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "liboracle.so")
_SOURCES = ["synth.cpp", "brute.cpp"]
_lib = None

C_LIGHT = 299792458.0  # m/s; wavelength = c / f (reading Q3: PAPER.md:117 prints "f/c")


def build(force: bool = False, sanitize: bool = False) -> str:
    """Compile oracle/*.cpp into oracle/liboracle.so (g++ -O2, no fast-math). sanitize=True builds
    oracle/liboracle_san.so with AddressSanitizer + UndefinedBehaviorSanitizer instead (tests/test_sanitizers.py)."""
    srcs = [os.path.join(_HERE, s) for s in _SOURCES]
    out = os.path.join(_HERE, "liboracle_san.so") if sanitize else _LIB_PATH
    if (not force and os.path.exists(out)
            and all(os.path.getmtime(out) >= os.path.getmtime(s) for s in srcs)):
        return out
    flags = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"] if sanitize else ["-O2"]
    cmd = ["g++"] + flags + ["-std=c++17", "-fPIC", "-shared", "-pthread", "-o", out] + srcs
    subprocess.run(cmd, check=True)
    return out


def _load():
    global _lib
    if _lib is None:
        path = build(sanitize=True) if os.environ.get("BB_ORACLE_SANITIZE") else build()
        lib = ctypes.CDLL(path)
        dp = ctypes.POINTER(ctypes.c_double)
        lib.oracle_synth.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int64,
                                     dp, ctypes.c_int, dp, ctypes.c_int, dp, ctypes.c_int,
                                     dp, ctypes.c_int64, ctypes.c_double, dp, ctypes.c_int]
        lib.oracle_synth.restype = ctypes.c_int
        lib.oracle_brute.argtypes = lib.oracle_synth.argtypes[:-1]
        lib.oracle_brute.restype = ctypes.c_int
        lib.oracle_hardware_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def hardware_threads() -> int:
    return int(_load().oracle_hardware_threads())


def _f(a, dtype):
    return np.asfortranarray(np.asarray(a, dtype=dtype))


def _dptr(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


# ---------------------------------------------------------------------------------- glue steps
def gram(xyz, W, wavelength):
    """Eq. 11 + Eq. 24. xyz (n_ant,3) metres; W (n_ant,n_beam) complex or None (identity)."""
    xyz = np.asarray(xyz, dtype=np.float64)
    diff = xyz[:, None, :] - xyz[None, :, :]
    dist = np.sqrt(np.sum(diff * diff, axis=-1))           # ||x_p - x_q||
    psi = np.sinc(2.0 * dist / wavelength)                 # sinc(2 ||b_pq||), np.sinc is normalized
    if W is None:
        return psi.astype(np.complex128)
    W = np.asarray(W, dtype=np.complex128)
    return W.conj().T @ psi @ W


def geig(S, G):
    """Eq. 13: S v = lambda G v with V^H G V = I. Returns (lambda ascending, V columns)."""
    S = np.asarray(S, dtype=np.complex128)
    G = np.asarray(G, dtype=np.complex128)
    S = 0.5 * (S + S.conj().T)                             # reading Q10
    G = 0.5 * (G + G.conj().T)
    L = np.linalg.cholesky(G)                              # G = L L^H
    Y = np.linalg.solve(L, S)                              # L^-1 S
    C = np.linalg.solve(L, Y.conj().T).conj().T            # L^-1 S L^-H
    C = 0.5 * (C + C.conj().T)
    lam, Q = np.linalg.eigh(C)
    V = np.linalg.solve(L.conj().T, Q)                     # L^-H Q
    return lam, V


def select(lam, V, n_eig):
    """Alg. 1 line 4: N_eig largest eigenvalues (by signed value, reading Q6), descending."""
    order = np.argsort(lam, kind="stable")[::-1][:n_eig]
    return lam[order], V[:, order]


def level_weights(lam, intervals, filt="lsq"):
    """D[l,k] for closed intervals [min_l, max_l] (reading Q7), LSQ (d = lambda) or STD (d = 1).
    `filt` may also be a sequence of filters (Alg. 1 l.6: N_f filters): the blocks are stacked, row
    f * N_i + i belonging to (filter f, interval i) = B^(n_i, n_f) of Alg. 1 l.9."""
    if not isinstance(filt, str):
        return np.vstack([level_weights(lam, intervals, f) for f in filt])
    assert filt in ("lsq", "std")
    lam = np.asarray(lam, dtype=np.float64)
    intervals = np.asarray(intervals, dtype=np.float64).reshape(-1, 2)
    inside = (lam[None, :] >= intervals[:, :1]) & (lam[None, :] <= intervals[:, 1:])
    d = lam if filt == "lsq" else np.ones_like(lam)
    return np.where(inside, d[None, :], 0.0)


# ---------------------------------------------------------------------------------- parameter estimation
def estimate_n_eig(lam, fraction):
    """Smallest m such that the m largest eigenvalues hold >= fraction of the sum of the positive ones."""
    lam = np.sort(np.asarray(lam, dtype=np.float64))[::-1]
    pos = np.where(lam > 0.0, lam, 0.0)
    total = 0.0
    for x in pos:
        total = total + x
    target = fraction * total
    run = 0.0
    for a, x in enumerate(pos):
        run = run + x
        if run >= target:
            return a + 1
    return len(pos)


def kmeans_levels(lam, n_levels, log_domain=True):
    """Exact 1-D k-means of the positive eigenvalues (optionally of their logarithms): minimise the
    within-cluster sum of squares over all partitions of the sorted values into n_levels contiguous
    groups (optimal k-means clusters in one dimension are contiguous). Returns intervals
    (n_levels, 2), level 0 = highest energy: edges at the midpoints between adjacent centroids
    (mapped back from the log domain), lowest edge 0, highest the largest finite double."""
    lam = np.asarray(lam, dtype=np.float64)
    x = np.sort(np.log(lam[lam > 0.0]) if log_domain else lam[lam > 0.0])
    n, k = len(x), int(n_levels)
    if n < k:
        raise ValueError("fewer positive eigenvalues than levels")
    p1 = np.zeros(n + 1)
    p2 = np.zeros(n + 1)
    for i in range(n):
        p1[i + 1] = p1[i] + x[i]
        p2[i + 1] = p2[i] + x[i] * x[i]

    def cost(i, j):                                         # sum of squared deviations of x[i:j]; i may be an array
        s1 = p1[j] - p1[i]
        s2 = p2[j] - p2[i]
        return s2 - (s1 * s1) / (j - i)

    big = np.finfo(np.float64).max
    prev = np.full(n + 1, big)
    for j in range(1, n + 1):
        prev[j] = cost(0, j)
    arg = np.zeros((k, n + 1), dtype=np.int64)
    for c in range(1, k):
        cur = np.full(n + 1, big)
        for j in range(c + 1, n + 1):
            i = np.arange(c, j)
            v = prev[c:j] + cost(i, j)
            b = int(np.argmin(v))                           # first minimum: the earliest split
            cur[j] = v[b]
            arg[c, j] = c + b
        prev = cur
    start = [0] * (k + 1)
    start[k] = n
    for c in range(k - 1, 0, -1):
        start[c] = int(arg[c, start[c + 1]])
    cen = [(p1[start[c + 1]] - p1[start[c]]) / (start[c + 1] - start[c]) for c in range(k)]
    iv = np.zeros((k, 2))
    for l in range(k):
        c = k - 1 - l
        lo, hi = 0.0, big
        if c > 0:
            e = 0.5 * (cen[c - 1] + cen[c])
            lo = np.exp(e) if log_domain else e
        if c < k - 1:
            e = 0.5 * (cen[c] + cen[c + 1])
            hi = np.exp(e) if log_domain else e
        iv[l] = (lo, hi)
    return iv


# ---------------------------------------------------------------------------------- image weighting (Section 3.5)
def _uv_cells(xyz, wavelength, e_u, e_v, cell):
    """Integer uv cell of every antenna pair (p, q): baseline b_pq = (x_p - x_q) / lambda_w, projected
    on the image-plane axes e_u, e_v; cell index = nearest integer of u / cell (the cell centred on the origin)."""
    xyz = np.asarray(xyz, dtype=np.float64)
    pu = (xyz @ np.asarray(e_u, dtype=np.float64)) / wavelength
    pv = (xyz @ np.asarray(e_v, dtype=np.float64)) / wavelength
    cu = np.rint((pu[:, None] - pu[None, :]) / cell).astype(np.int64)
    cv = np.rint((pv[:, None] - pv[None, :]) / cell).astype(np.int64)
    return cu, cv


def uv_density(collects, e_u, e_v, cell):
    """Sampling density function: number of visibilities (all antenna pairs, p = q included, of all the given
    collects = [(xyz, wavelength), ...]) in each uv cell of side `cell` = 1 / FoV. Returns {(cu, cv): count}."""
    density = {}
    for xyz, wavelength in collects:
        cu, cv = _uv_cells(xyz, wavelength, e_u, e_v, cell)
        for a, b in zip(cu.ravel().tolist(), cv.ravel().tolist()):
            density[(a, b)] = density.get((a, b), 0) + 1
    return density


def uniform_weights(xyz, wavelength, e_u, e_v, cell, density):
    """(n_ant, n_ant) real weights 1 / density(cell of b_pq); the visibility matrix is multiplied by them entry by
    entry before the eigendecomposition (W = I only: a beamformed visibility has no single baseline)."""
    cu, cv = _uv_cells(xyz, wavelength, e_u, e_v, cell)
    w = np.empty(cu.shape, dtype=np.float64)
    for p in range(cu.shape[0]):
        for q in range(cu.shape[1]):
            w[p, q] = 1.0 / density[(int(cu[p, q]), int(cv[p, q]))]
    return w


# ---------------------------------------------------------------------------------- synthesis
def synth(B, D, xyz, pix, wavelength, img=None, n_threads=0):
    """I_l(r_j) += sum_k D[l,k] |sum_i conj(B_ik) exp(+j 2 pi <p_i,r_j>/lambda_w)|^2 (Alg. 2)."""
    B = _f(B, np.complex128)
    D = _f(np.atleast_2d(D), np.float64)
    xyz = _f(xyz, np.float64)
    pix = _f(pix, np.float64)
    n_ant, n_eig = B.shape
    n_levels = D.shape[0]
    n_pix = pix.shape[0]
    assert D.shape[1] == n_eig and xyz.shape == (n_ant, 3) and pix.shape[1] == 3
    if img is None:
        img = np.zeros((n_levels, n_pix), dtype=np.float64)
    assert img.shape == (n_levels, n_pix) and img.dtype == np.float64 and img.flags.c_contiguous
    rc = _load().oracle_synth(n_ant, n_eig, n_levels, n_pix, _dptr(B), max(n_ant, 1),
                              _dptr(D), max(n_levels, 1), _dptr(xyz), max(n_ant, 1), _dptr(pix),
                              max(n_pix, 1), float(wavelength), _dptr(img), int(n_threads))
    if rc != 0:
        raise ValueError("oracle_synth: invalid arguments")
    return img


def brute(B, D, xyz, pix, wavelength):
    """Literal triple sum with the exponential in the innermost loop (tiny inputs only)."""
    B = _f(B, np.complex128)
    D = _f(np.atleast_2d(D), np.float64)
    xyz = _f(xyz, np.float64)
    pix = _f(pix, np.float64)
    n_ant, n_eig = B.shape
    n_levels, n_pix = D.shape[0], pix.shape[0]
    img = np.zeros((n_levels, n_pix), dtype=np.float64)
    _load().oracle_brute(n_ant, n_eig, n_levels, n_pix, _dptr(B), max(n_ant, 1),
                         _dptr(D), max(n_levels, 1), _dptr(xyz), max(n_ant, 1), _dptr(pix),
                         max(n_pix, 1), float(wavelength), _dptr(img))
    return img


# ---------------------------------------------------------------------------------- NUFFT synthesis, direct form
def gram_corrected_visibilities(B, D):
    """Eq. 17 with the level selection of Eq. 21: V'_l = B diag(D[l, :]) B^H, one (n_ant, n_ant) matrix per level
    ("constructed by setting eigenvalues which fall outside the interval to zero"; B = W alpha, Eq. 22-24)."""
    B = np.asarray(B, dtype=np.complex128)
    D = np.atleast_2d(np.asarray(D, dtype=np.float64))
    return np.stack([(B * D[l][None, :]) @ B.conj().T for l in range(D.shape[0])])


def nufft_direct(B, D, xyz, pix, wavelength):
    """Eq. 18-19: I_l(r_j) = sum_p sum_q V'_l,pq exp(-2 pi i <b_pq, r_j>), b_pq = (x_p - x_q) / lambda_w — the sum a
    type-3 NUFFT evaluates approximately, written out over all N_A^2 baselines. Returns (images (L, n_pix) real part,
    largest |imaginary part|): the sum is real because V' is Hermitian and b_qp = -b_pq."""
    V = gram_corrected_visibilities(B, D)
    xyz = np.asarray(xyz, dtype=np.float64)
    pix = np.asarray(pix, dtype=np.float64)
    n_ant = xyz.shape[0]
    img = np.zeros((V.shape[0], pix.shape[0]), dtype=np.complex128)
    for p in range(n_ant):
        for q in range(n_ant):
            b = (xyz[p] - xyz[q]) / wavelength
            img += V[:, p, q][:, None] * np.exp(-2j * np.pi * (pix @ b))[None, :]
    return img.real, float(np.max(np.abs(img.imag)))


# ---------------------------------------------------------------------------------- Alg. 1
def eig_stage(S, W, xyz, wavelength, n_eig, gram_identity=False, vis_weights=None):
    """Alg. 1 lines 2-4 and U = W alpha. Returns (lambda desc (n_eig,), B (n_ant,n_eig)).
    vis_weights: optional (n_beam, n_beam) real weights applied to S entry by entry first (Section 3.5)."""
    n_ant = np.asarray(xyz).shape[0]
    if vis_weights is not None:
        assert W is None, "uniform weighting is defined on antenna baselines (W = I)"
        S = np.asarray(S, dtype=np.complex128) * np.asarray(vis_weights, dtype=np.float64)
    if gram_identity:                                       # G := I special case
        G = np.eye(np.asarray(S).shape[0], dtype=np.complex128)
    else:
        G = gram(xyz, W, wavelength)
    lam, V = geig(S, G)
    lam, V = select(lam, V, n_eig)
    B = V if W is None else np.asarray(W, dtype=np.complex128) @ V
    assert B.shape[0] == n_ant
    return lam, B


def collect(S, W, xyz, wavelength, n_eig, intervals, pix, img=None, filt="lsq",
            gram_identity=False, n_threads=0, vis_weights=None):
    """Algorithm 1 for one time step / channel; accumulates into img."""
    lam, B = eig_stage(S, W, xyz, wavelength, n_eig, gram_identity, vis_weights)
    D = level_weights(lam, intervals, filt)
    return synth(B, D, xyz, pix, wavelength, img=img, n_threads=n_threads)
