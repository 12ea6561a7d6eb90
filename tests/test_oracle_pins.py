"""Pins for the oracle (no GPU): closed forms, brute force, invariants.

The paper prints no worked numeric example of the method, so the oracle is
pinned by what the mathematics fixes. Ids follow DESIGN.md / SURVEY.md section 8c (P1-P6, I1-I8).
Each test builds its own inputs with plain numpy (not with oracle helpers) wherever a plausible
mistake in the oracle - dropped conjugate, wrong sign, transposed operand, wrong sinc
convention, wrong normalisation - must show up.
"""
import numpy as np
import pytest


def unit(v):
    v = np.asarray(v, dtype=np.float64)
    return v / np.linalg.norm(v, axis=-1, keepdims=True)


def steering(xyz, dirs, wl):
    """a_i(r) = exp(+j 2 pi <p_i, r>/lambda_w)  (Eq. 3), shape (n_ant, n_dir)."""
    return np.exp(2j * np.pi * (xyz @ np.atleast_2d(dirs).T) / wl)


def grid_dirs(n, fov_deg):
    step = 2.0 * np.sin(np.radians(fov_deg) / 2.0) / n
    g = (np.arange(n) - n // 2) * step
    l, m = np.tile(g, n), np.repeat(g, n)
    return np.column_stack([l, m, np.sqrt(1.0 - l * l - m * m)])


def rand_layout(rng, n, extent):
    return np.column_stack([rng.uniform(-extent, extent, n), rng.uniform(-extent, extent, n), rng.normal(0, 1, n)])


# ------------------------------------------------------------------------------------------ P1
@pytest.mark.parametrize("n_ant,n_eig,n_lev,n_pix,wl", [(1, 1, 1, 5, 2.0), (8, 3, 2, 64, 1.7), (16, 8, 2, 40, 3.1)])
def test_P1_synth_equals_brute(oracle, n_ant, n_eig, n_lev, n_pix, wl):
    rng = np.random.default_rng(100 + n_ant)
    B = rng.normal(size=(n_ant, n_eig)) + 1j * rng.normal(size=(n_ant, n_eig))
    D = rng.normal(size=(n_lev, n_eig))
    xyz = rand_layout(rng, n_ant, 80.0)
    pix = unit(rng.normal(size=(n_pix, 3)))
    a = oracle.synth(B, D, xyz, pix, wl)
    b = oracle.brute(B, D, xyz, pix, wl)
    assert np.max(np.abs(a - b)) <= 1e-12 * np.max(np.abs(b))
    # and against the definition retyped with numpy matrices (different code again)
    E = B.conj().T @ steering(xyz, pix, wl)
    c = D @ (np.abs(E) ** 2)
    assert np.max(np.abs(a - c)) <= 1e-11 * np.max(np.abs(c))


def test_P1_conjugation_matters(oracle):
    """The un-conjugated contraction is a different image (reading Q1): make sure the pin sees it."""
    rng = np.random.default_rng(7)
    B = rng.normal(size=(6, 2)) + 1j * rng.normal(size=(6, 2))
    xyz = rand_layout(rng, 6, 30.0)
    pix = unit(rng.normal(size=(9, 3)))
    good = oracle.synth(B, np.ones((1, 2)), xyz, pix, 2.0)
    wrong = np.sum(np.abs(B.T @ steering(xyz, pix, 2.0)) ** 2, axis=0)
    assert np.max(np.abs(good[0] - wrong)) > 1e-3 * np.max(good)


# ------------------------------------------------------------------------------------------ P6
def test_P6_two_element_interferometer(oracle):
    d, wl = 37.5, 2.5
    xyz = np.array([[-d / 2, 0, 0], [d / 2, 0, 0]])
    B = np.ones((2, 1)) / np.sqrt(2.0)
    l = np.linspace(-0.3, 0.3, 101)
    pix = np.column_stack([l, np.zeros_like(l), np.sqrt(1 - l * l)])
    img = oracle.synth(B, [[1.0]], xyz, pix, wl)[0]
    assert np.allclose(img, 1.0 + np.cos(2 * np.pi * d * l / wl), rtol=0, atol=1e-12)


def test_P6_uniform_line_array_dirichlet(oracle):
    n, d, wl = 12, 1.3, 2.0
    xyz = np.column_stack([np.arange(n) * d, np.zeros(n), np.zeros(n)])
    B = np.ones((n, 1)) / np.sqrt(n)
    l = np.linspace(-0.45, 0.45, 200) + 1e-3      # avoid l = 0 (0/0 in the closed form)
    pix = np.column_stack([l, np.zeros_like(l), np.sqrt(1 - l * l)])
    img = oracle.synth(B, [[1.0]], xyz, pix, wl)[0]
    x = np.pi * d * l / wl
    assert np.allclose(img, np.sin(n * x) ** 2 / (n * np.sin(x) ** 2), rtol=0, atol=1e-11)


def test_P6_single_antenna_constant(oracle):
    B = np.array([[0.3 - 0.4j, 2.0 + 1.0j]])
    D = np.array([[2.0, 0.0], [0.5, 3.0]])
    pix = unit(np.random.default_rng(3).normal(size=(11, 3)))
    img = oracle.synth(B, D, [[12.0, -7.0, 3.0]], pix, 1.9)
    expect = D @ (np.abs(B[0]) ** 2)
    assert np.allclose(img, expect[:, None] * np.ones(11), rtol=1e-14)


def test_P6_phase_sign_asymmetric_array(oracle):
    """A beam steered to +l0 must peak at +l0, not -l0: pins the sign of the exponent together
    with the conjugate (a transposed/unconjugated operand moves the peak to -l0)."""
    n, d, wl, l0 = 16, 1.0, 2.0, 0.2
    xyz = np.column_stack([np.arange(n) * d + 0.37 * np.arange(n) ** 1.5, np.zeros(n), np.zeros(n)])
    r0 = np.array([l0, 0.0, np.sqrt(1 - l0 * l0)])
    B = steering(xyz, r0, wl)                      # B_i = a_i(r0)  =>  E(r) = a(r0)^H a(r)
    l = np.linspace(-0.4, 0.4, 161)
    pix = np.column_stack([l, np.zeros_like(l), np.sqrt(1 - l * l)])
    img = oracle.synth(B, [[1.0]], xyz, pix, wl)[0]
    assert abs(l[np.argmax(img)] - l0) < 1e-9 and np.isclose(img.max(), n * n, rtol=1e-12)


# ---------------------------------------------------------------------------------- P2 / P3
def _tiny_case(rng, n_ant=16, n=32, fov=10.0, wl=2.0):
    xyz = rand_layout(rng, n_ant, 70.0)
    pix = grid_dirs(n, fov)
    return xyz, pix, wl


def test_P2_point_source_identity_gram(oracle):
    rng = np.random.default_rng(11)
    xyz, pix, wl = _tiny_case(rng)
    j0, sigma = 13 + 32 * 21, 3.0
    a0 = steering(xyz, pix[j0], wl)[:, 0]
    S = sigma * np.outer(a0, a0.conj())
    img = oracle.collect(S, None, xyz, wl, 1, [[0.0, 1e9]], pix, gram_identity=True)[0]
    assert int(np.argmax(img)) == j0                                   # Cauchy-Schwarz
    assert np.isclose(img[j0], sigma * 16 ** 2, rtol=1e-10)
    expect = sigma * np.abs(a0.conj() @ steering(xyz, pix, wl)) ** 2
    assert np.allclose(img, expect, rtol=0, atol=1e-10 * expect.max())


def test_P3_point_source_real_gram(oracle):
    rng = np.random.default_rng(12)
    xyz, pix, wl = _tiny_case(rng)
    # close antennas so that G is far from the identity
    xyz[:8] *= 0.02
    j0, sigma = 500, 2.5
    A = steering(xyz, pix, wl)
    a0 = A[:, j0]
    S = sigma * np.outer(a0, a0.conj())
    # Gram retyped here independently: sinc(2 d / wl) with the NORMALIZED sinc sin(pi x)/(pi x)
    d = np.linalg.norm(xyz[:, None, :] - xyz[None, :, :], axis=-1)
    x = 2.0 * d / wl
    G = np.where(x == 0, 1.0, np.sin(np.pi * np.where(x == 0, 1, x)) / (np.pi * np.where(x == 0, 1, x)))
    assert np.allclose(oracle.gram(xyz, None, wl).real, G, atol=1e-14) and np.linalg.cond(G) > 3
    Ginv_a0 = np.linalg.solve(G, a0)
    expect = sigma * np.abs(Ginv_a0.conj() @ A) ** 2                   # sigma |a0^H G^-1 a(r)|^2
    img = oracle.collect(S, None, xyz, wl, 1, [[0.0, 1e12]], pix)[0]
    assert np.allclose(img, expect, rtol=0, atol=1e-9 * expect.max())
    assert np.isclose(img[j0], sigma * np.real(a0.conj() @ Ginv_a0) ** 2, rtol=1e-9)
    lam, _ = oracle.eig_stage(S, None, xyz, wl, 1)
    assert np.isclose(lam[0], sigma * np.real(a0.conj() @ Ginv_a0), rtol=1e-10)


# ---------------------------------------------------------------------------------- P4 / P5
def _random_sky_S(rng, xyz, wl, n_src=5, noise=0.3, W=None):
    dirs = unit(np.column_stack([rng.uniform(-0.08, 0.08, n_src), rng.uniform(-0.08, 0.08, n_src), np.ones(n_src)]))
    A = steering(xyz, dirs, wl)
    flux = rng.uniform(1, 5, n_src)
    S = (A * flux) @ A.conj().T + noise * np.eye(xyz.shape[0])
    if W is not None:
        S = W.conj().T @ S @ W
    return 0.5 * (S + S.conj().T)


@pytest.mark.parametrize("beamformed", [False, True])
def test_P4_sum_of_levels_is_least_squares_image(oracle, beamformed):
    rng = np.random.default_rng(21 + beamformed)
    xyz, pix, wl = _tiny_case(rng, n_ant=12, n=12)
    xyz[:5] *= 0.03
    W = None
    if beamformed:
        W = (rng.normal(size=(12, 5)) + 1j * rng.normal(size=(12, 5))) / 3.0
    S = _random_sky_S(rng, xyz, wl, W=W)
    nb = S.shape[0]
    d = np.linalg.norm(xyz[:, None, :] - xyz[None, :, :], axis=-1)
    Psi = np.sinc(2.0 * d / wl)
    G = Psi if W is None else W.conj().T @ Psi @ W
    A = steering(xyz, pix, wl)
    aW = A if W is None else W.conj().T @ A                            # a_W = W^H a(r)  (Q12)
    X = np.linalg.solve(G, aW)                                         # G^-1 a_W
    expect = np.real(np.sum(X.conj() * (S @ X), axis=0))              # a^H G^-1 S G^-1 a (Eq. 9)
    lam, _ = oracle.eig_stage(S, W, xyz, wl, nb)
    edges = [[np.median(lam), 2 * lam.max()], [lam.min() - 1.0, np.median(lam) * (1 - 1e-9)]]
    img = oracle.collect(S, W, xyz, wl, nb, edges, pix)
    assert np.allclose(img.sum(axis=0), expect, rtol=0, atol=1e-10 * np.abs(expect).max())


def test_P5_identity_gram_gives_dirty_image(oracle):
    rng = np.random.default_rng(31)
    xyz, pix, wl = _tiny_case(rng, n_ant=10, n=10)
    S = _random_sky_S(rng, xyz, wl)
    expect = np.zeros(pix.shape[0])
    for p in range(10):                                               # Eq. 26 written out
        for q in range(10):
            expect += np.real(S[p, q] * np.exp(-2j * np.pi * ((xyz[p] - xyz[q]) @ pix.T) / wl))
    img = oracle.collect(S, None, xyz, wl, 10, [[-1e9, 1e9]], pix, gram_identity=True)[0]
    assert np.allclose(img, expect, rtol=0, atol=1e-10 * expect.max())


# ---------------------------------------------------------------------------------- invariants
def test_I1_hermitian_inputs_real_gram(oracle):
    rng = np.random.default_rng(41)
    xyz = rand_layout(rng, 9, 20.0)
    G = oracle.gram(xyz, None, 2.2)
    assert np.allclose(G.imag, 0) and np.allclose(G, G.T) and np.allclose(np.diag(G).real, 1.0)
    W = rng.normal(size=(9, 4)) + 1j * rng.normal(size=(9, 4))
    GW = oracle.gram(xyz, W, 2.2)
    assert np.allclose(GW, GW.conj().T, atol=1e-13)
    lam, V = oracle.geig(_random_sky_S(rng, xyz, 2.2, W=W), GW)
    assert np.allclose(V.conj().T @ GW @ V, np.eye(4), atol=1e-11)     # V^H G V = I (reading Q5)
    assert np.all(np.diff(lam) >= 0)


def test_I1_geig_matches_scipy_generalized_solver(oracle):
    scipy_linalg = pytest.importorskip("scipy.linalg")
    rng = np.random.default_rng(42)
    xyz = rand_layout(rng, 14, 15.0)
    G = oracle.gram(xyz, None, 3.0)
    S = _random_sky_S(rng, xyz, 3.0)
    lam, V = oracle.geig(S, G)
    lam2 = scipy_linalg.eigh(S, G, eigvals_only=True)
    assert np.allclose(lam, lam2, rtol=1e-10)
    assert np.allclose(S @ V, (G @ V) * lam, atol=1e-9 * np.abs(lam).max())


def test_I2_nonnegative_for_nonnegative_weights(oracle):
    rng = np.random.default_rng(43)
    B = rng.normal(size=(7, 4)) + 1j * rng.normal(size=(7, 4))
    img = oracle.synth(B, rng.uniform(0, 2, size=(3, 4)), rand_layout(rng, 7, 50), unit(rng.normal(size=(50, 3))), 2.0)
    assert np.all(img >= 0)


def test_I3_sum_over_levels_independent_of_level_count(oracle):
    """The paper's own check (Table 2)."""
    rng = np.random.default_rng(44)
    xyz, pix, wl = _tiny_case(rng, n_ant=16, n=8)
    S = _random_sky_S(rng, xyz, wl, n_src=6)
    lam, _ = oracle.eig_stage(S, None, xyz, wl, 16)
    ref = None
    for L in (1, 2, 4, 8):
        cuts = [2 * lam[0]] + [np.sqrt(lam[q * 16 // L - 1] * lam[q * 16 // L]) for q in range(1, L)] + [lam[-1] / 2]
        iv = [[cuts[l + 1], cuts[l]] for l in range(L)]
        tot = oracle.collect(S, None, xyz, wl, 16, iv, pix).sum(axis=0)
        ref = tot if ref is None else ref
        assert np.allclose(tot, ref, rtol=0, atol=1e-13 * ref.max())


def test_I4_unit_phase_on_eigenvector_columns(oracle):
    rng = np.random.default_rng(45)
    B = rng.normal(size=(7, 4)) + 1j * rng.normal(size=(7, 4))
    D = rng.uniform(0, 2, size=(2, 4))
    xyz, pix = rand_layout(rng, 7, 50), unit(rng.normal(size=(20, 3)))
    a = oracle.synth(B, D, xyz, pix, 2.0)
    b = oracle.synth(B * np.exp(1j * rng.uniform(0, 6.28, size=4)), D, xyz, pix, 2.0)
    assert np.allclose(a, b, rtol=0, atol=1e-13 * a.max())


def test_I5_image_independent_of_eigensolver(oracle):
    scipy_linalg = pytest.importorskip("scipy.linalg")
    rng = np.random.default_rng(46)
    xyz, pix, wl = _tiny_case(rng, n_ant=12, n=8)
    S = _random_sky_S(rng, xyz, wl)
    iv = [[1.0, 1e6], [1e-3, 1.0]]
    a = oracle.collect(S, None, xyz, wl, 6, iv, pix)
    lam, V = scipy_linalg.eigh(S, oracle.gram(xyz, None, wl))          # a different solver
    lam, V = lam[::-1][:6], V[:, ::-1][:, :6]
    b = oracle.synth(V, oracle.level_weights(lam, iv), xyz, pix, wl)
    assert np.allclose(a, b, rtol=0, atol=1e-10 * a.max())


def test_I6_additive_over_collects_and_linear_in_D(oracle):
    rng = np.random.default_rng(47)
    xyz, pix = rand_layout(rng, 6, 40), unit(rng.normal(size=(17, 3)))
    B1 = rng.normal(size=(6, 3)) + 1j * rng.normal(size=(6, 3))
    B2 = rng.normal(size=(6, 3)) + 1j * rng.normal(size=(6, 3))
    D1, D2 = rng.normal(size=(2, 3)), rng.normal(size=(2, 3))
    acc = oracle.synth(B1, D1, xyz, pix, 2.0)
    acc = oracle.synth(B2, D2, xyz, pix, 2.0, img=acc)
    sep = oracle.synth(B1, D1, xyz, pix, 2.0) + oracle.synth(B2, D2, xyz, pix, 2.0)
    assert np.allclose(acc, sep, rtol=0, atol=1e-13 * np.abs(sep).max())
    lin = oracle.synth(B1, 2 * D1 + D2, xyz, pix, 2.0)
    assert np.allclose(lin, 2 * oracle.synth(B1, D1, xyz, pix, 2.0) + oracle.synth(B1, D2, xyz, pix, 2.0),
                       rtol=0, atol=1e-12 * np.abs(lin).max())


def test_I7_translation_invariance(oracle):
    rng = np.random.default_rng(48)
    xyz, pix, wl = _tiny_case(rng, n_ant=10, n=8)
    S = _random_sky_S(rng, xyz, wl)   # built from sources: S changes by a diagonal similarity only
    iv = [[0.0, 1e9]]
    a = oracle.collect(S, None, xyz, wl, 10, iv, pix)
    shift = np.array([1234.5, -987.25, 333.0])
    # S for shifted antennas: a_i -> a_i * exp(j 2 pi <shift, r_q>/wl) per source, i.e. S is unchanged
    # only when rebuilt from the sources; rebuild it.
    rng2 = np.random.default_rng(48)
    _tiny_case(rng2, n_ant=10, n=8)
    S2 = _random_sky_S(rng2, xyz + shift, wl)
    b = oracle.collect(S2, None, xyz + shift, wl, 10, iv, pix)
    assert np.allclose(a, b, rtol=0, atol=1e-9 * a.max())
    # the synthesizer alone: a common shift multiplies E_kj by a unit phasor per pixel
    B = rng.normal(size=(10, 3)) + 1j * rng.normal(size=(10, 3))
    c = oracle.synth(B, np.ones((1, 3)), xyz, pix, wl)
    d = oracle.synth(B, np.ones((1, 3)), xyz + shift, pix, wl)
    assert np.allclose(c, d, rtol=0, atol=1e-10 * c.max())


def test_I8_rotation_and_pixel_subset(oracle):
    rng = np.random.default_rng(49)
    xyz, pix = rand_layout(rng, 8, 60), unit(rng.normal(size=(30, 3)))
    B = rng.normal(size=(8, 3)) + 1j * rng.normal(size=(8, 3))
    D = rng.uniform(0, 1, size=(2, 3))
    Q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
    a = oracle.synth(B, D, xyz, pix, 2.0)
    b = oracle.synth(B, D, xyz @ Q.T, pix @ Q.T, 2.0)
    assert np.allclose(a, b, rtol=0, atol=1e-12 * a.max())
    sub = np.array([3, 17, 4, 29])
    assert np.array_equal(oracle.synth(B, D, xyz, pix[sub], 2.0), a[:, sub])
    # thread count changes nothing (pixels are independent)
    assert np.array_equal(oracle.synth(B, D, xyz, pix, 2.0, n_threads=1), oracle.synth(B, D, xyz, pix, 2.0, n_threads=5))


# ------------------------------------------------------------------------------ level weights
def test_level_weights_closed_overlapping_uncovered(oracle):
    lam = np.array([10.0, 5.0, 2.0, 1.0, -0.5])
    iv = [[5.0, 10.0], [2.0, 5.0], [-1.0, -0.5]]                      # closed; 5.0 in two; 1.0 in none
    D = oracle.level_weights(lam, iv)
    assert np.array_equal(D, [[10, 5, 0, 0, 0], [0, 5, 2, 0, 0], [0, 0, 0, 0, -0.5]])
    assert np.array_equal(oracle.level_weights(lam, iv, "std"), (D != 0).astype(float))


def test_select_largest_signed(oracle):
    lam = np.array([-9.0, 0.1, 3.0, 2.0])
    V = np.arange(16.0).reshape(4, 4)
    l, v = oracle.select(lam, V, 2)
    assert np.array_equal(l, [3.0, 2.0]) and np.array_equal(v, V[:, [2, 3]])


# ---------------------------------------------------------------------------------- filters
@pytest.mark.parametrize("beamformed", [False, True])
def test_P7_standardized_filter_sums_to_inverse_gram_form(oracle, beamformed):
    """STD filter (d = 1) over ALL eigenpairs: sum_k |v_k^H a_W|^2 = a_W^H G^-1 a_W because the
    G-orthonormal eigenvectors satisfy V V^H = G^-1 -- a linear solve, no eigensolver."""
    rng = np.random.default_rng(41 + beamformed)
    xyz, pix, wl = _tiny_case(rng, n_ant=12, n=12)
    W = (rng.normal(size=(12, 5)) + 1j * rng.normal(size=(12, 5))) / 3.0 if beamformed else None
    S = _random_sky_S(rng, xyz, wl, W=W)
    nb = S.shape[0]
    d = np.linalg.norm(xyz[:, None, :] - xyz[None, :, :], axis=-1)
    Psi = np.sinc(2.0 * d / wl)
    G = Psi if W is None else W.conj().T @ Psi @ W
    A = steering(xyz, pix, wl)
    aW = A if W is None else W.conj().T @ A
    expect = np.real(np.sum(aW.conj() * np.linalg.solve(G, aW), axis=0))
    img = oracle.collect(S, W, xyz, wl, nb, [[-1e9, 1e9]], pix, filt="std")[0]
    assert np.allclose(img, expect, rtol=0, atol=1e-10 * expect.max())


def test_P7_standardized_identity_gram_is_constant(oracle):
    """G := I, W = I, STD filter, all eigenpairs: sum_k |v_k^H a|^2 = |a|^2 = N_ant at every pixel."""
    rng = np.random.default_rng(43)
    xyz, pix, wl = _tiny_case(rng, n_ant=9, n=8)
    S = _random_sky_S(rng, xyz, wl)
    img = oracle.collect(S, None, xyz, wl, 9, [[-1e9, 1e9]], pix, filt="std", gram_identity=True)[0]
    assert np.allclose(img, 9.0, rtol=0, atol=1e-10)


def test_filters_stack_as_interval_blocks(oracle):
    """N_f filters (Alg. 1 l.6-12): image f * N_i + i is (filter f, interval i), each block equal to the
    single-filter run; LSQ and STD blocks differ exactly by the eigenvalue weights."""
    rng = np.random.default_rng(44)
    xyz, pix, wl = _tiny_case(rng, n_ant=10, n=6)
    S = _random_sky_S(rng, xyz, wl)
    lam, B = oracle.eig_stage(S, None, xyz, wl, 6)
    iv = [[lam[2] * 0.999, 2 * lam[0]], [0.0, lam[3] * 1.001]]
    both = oracle.collect(S, None, xyz, wl, 6, iv, pix, filt=("std", "lsq"))
    assert both.shape[0] == 4
    assert np.array_equal(both[:2], oracle.collect(S, None, xyz, wl, 6, iv, pix, filt="std"))
    assert np.array_equal(both[2:], oracle.collect(S, None, xyz, wl, 6, iv, pix, filt="lsq"))
    D = oracle.level_weights(lam, iv, ("std", "lsq"))
    assert np.array_equal(D[2:], D[:2] * lam[None, :])


# ---------------------------------------------------------------------------------- parameter estimation
def test_estimate_n_eig_geometric_spectrum(oracle):
    """lambda_a = 2^-a: the m leading values hold 1 - 2^-m of the (infinite) total, so 90 % needs m = 4 and
    99.9 % needs m = 10; non-positive values carry no energy."""
    lam = np.concatenate([2.0 ** -np.arange(1, 40), [-3.0, 0.0]])
    rng = np.random.default_rng(5)
    rng.shuffle(lam)
    assert oracle.estimate_n_eig(lam, 0.9) == 4
    assert oracle.estimate_n_eig(lam, 0.999) == 10
    assert oracle.estimate_n_eig(lam, 1.0) <= 39


@pytest.mark.parametrize("log_domain", [False, True])
def test_kmeans_levels_is_the_global_optimum(oracle, log_domain):
    """Brute force over ALL k^n assignments of 9 values to 3 clusters (not only contiguous ones): the dynamic
    programme must reach the same minimum within-cluster sum of squares, and its edges must separate the
    optimal clusters."""
    import itertools
    rng = np.random.default_rng(17 + log_domain)
    lam = np.concatenate([rng.uniform(90, 110, 3), rng.uniform(9, 12, 3), rng.uniform(0.8, 1.3, 3)]) * rng.uniform(0.5, 2)
    x = np.log(lam) if log_domain else lam
    best, best_lab = np.inf, None
    for lab in itertools.product(range(3), repeat=9):
        lab = np.array(lab)
        if len(set(lab)) < 3:
            continue
        sse = sum(np.sum((x[lab == c] - x[lab == c].mean()) ** 2) for c in range(3))
        if sse < best:
            best, best_lab = sse, lab
    iv = oracle.kmeans_levels(lam, 3, log_domain)
    got = np.array([[l for l in range(3) if iv[l, 0] <= v <= iv[l, 1]] for v in lam]).ravel()
    assert got.size == 9                                            # every value in exactly one level
    sse = sum(np.sum((x[got == l] - x[got == l].mean()) ** 2) for l in range(3))
    assert abs(sse - best) <= 1e-12 * best
    assert iv[0, 1] == np.finfo(np.float64).max and iv[2, 0] == 0.0 and iv[0, 0] == iv[1, 1] and iv[1, 0] == iv[2, 1]
    assert lam[got == 0].min() > lam[got == 1].max() > lam[got == 2].max()     # level 0 = highest energy


def _kmeans_spectra():
    """Spectra for the contiguous-partition brute force: random, log-spread, exactly tied, nearly tied (1e-13
    apart), and values that fall on what would be an edge of a coarser clustering."""
    rng = np.random.default_rng(164)
    out = []
    for n in (5, 8, 11, 14):
        out.append(rng.uniform(0.1, 10.0, n))
        out.append(np.exp(rng.normal(0.0, 3.0, n)))
        t = rng.uniform(1.0, 5.0, n)
        t[1] = t[0]; t[-1] = t[-2]                                # exact ties
        out.append(t)
        nt = rng.uniform(1.0, 5.0, n)
        nt[2] = nt[3] * (1.0 + 1e-13)                             # near tie
        out.append(nt)
        out.append(np.arange(1, n + 1, dtype=np.float64))         # equally spaced: many equal-cost splits
        out.append(np.concatenate([[1.0, 2.0, 3.0], 3.0 + 2.0 ** -np.arange(n - 3)]))
    out.append(np.array([1.0, 1.0, 1.0, 4.0, 4.0, 9.0, 9.0, 9.0, 9.0, 16.0, -2.0, 0.0]))
    return out


@pytest.mark.parametrize("log_domain", [False, True])
@pytest.mark.parametrize("k", [2, 3, 4, 5])
def test_kmeans_levels_reaches_the_brute_force_minimum_over_contiguous_partitions(oracle, k, log_domain):
    """PAPER.md:164, reading Q16. For n <= 14 every contiguous partition is enumerated with the cost written out
    from its definition (helpers.kmeans_brute_contiguous); the oracle's intervals must induce a partition whose
    cost equals that minimum and must be a valid level structure (helpers.kmeans_partition_check). An off-by-one
    anywhere in a split search or its back-tracking yields a non-optimal or invalid partition and fails here."""
    from helpers import kmeans_brute_contiguous, kmeans_partition_check
    for lam in _kmeans_spectra():
        pos = np.sort(lam[lam > 0])
        if len(np.unique(pos)) < k:
            continue
        x = np.log(pos) if log_domain else pos
        best = kmeans_brute_contiguous(x, k)
        iv = oracle.kmeans_levels(lam, k, log_domain)
        sse = kmeans_partition_check(lam, iv, k, log_domain)
        assert sse <= best + 1e-12 * max(best, 1e-30) + 1e-13 * float(np.sum(x * x)), (k, log_domain, lam, sse, best)


def test_kmeans_levels_all_assignments_four_clusters(oracle):
    """All 4^8 assignments (contiguous or not) of 8 log-spread values to 4 clusters: the contiguity theorem the
    oracle and the enumeration above rely on, checked where it can be."""
    import itertools
    from helpers import kmeans_partition_check
    rng = np.random.default_rng(8)
    lam = np.exp(rng.normal(0.0, 2.0, 8))
    best = np.inf
    for lab in itertools.product(range(4), repeat=8):
        lab = np.array(lab)
        if len(set(lab.tolist())) < 4:
            continue
        best = min(best, sum(np.sum((lam[lab == c] - lam[lab == c].mean()) ** 2) for c in range(4)))
    sse = kmeans_partition_check(lam, oracle.kmeans_levels(lam, 4, False), 4, False)
    assert abs(sse - best) <= 1e-12 * best


def test_kmeans_levels_needs_enough_positive_values(oracle):
    with pytest.raises(ValueError):
        oracle.kmeans_levels([1.0, -2.0, 0.0], 2)


# ---------------------------------------------------------------------------------- uniform weighting (Section 3.5)
def test_uniform_weights_hand_computed_line_array(oracle):
    """Three antennas on a line at spacing d, cell = d: the uv cells hold {0: 3 autocorrelations, +-d: 2 each,
    +-2d: 1 each}, so the weights are 1/3 on the diagonal, 1/2 next to it and 1 in the corners — worked by hand."""
    d, wl = 7.0, 2.0
    xyz = np.array([[0.0, 0, 0], [d, 0, 0], [2 * d, 0, 0]])
    e_u, e_v = np.array([1.0, 0, 0]), np.array([0, 1.0, 0])
    dens = oracle.uv_density([(xyz, wl)], e_u, e_v, d / wl)
    assert dens == {(0, 0): 3, (1, 0): 2, (-1, 0): 2, (2, 0): 1, (-2, 0): 1}
    w = oracle.uniform_weights(xyz, wl, e_u, e_v, d / wl, dens)
    assert np.allclose(w, [[1 / 3, 1 / 2, 1], [1 / 2, 1 / 3, 1 / 2], [1, 1 / 2, 1 / 3]], rtol=0, atol=1e-15)
    # the density accumulates over collects: the same epoch twice halves every weight
    dens2 = oracle.uv_density([(xyz, wl), (xyz, wl)], e_u, e_v, d / wl)
    assert np.allclose(oracle.uniform_weights(xyz, wl, e_u, e_v, d / wl, dens2), w / 2)


def test_uniform_weighting_with_one_visibility_per_cell_is_natural_weighting(oracle):
    """If no two baselines share a uv cell (and the N autocorrelations are the only visibilities at the origin), the
    off-diagonal weights are 1 and the diagonal 1/N: S' = S - (1 - 1/N) diag(S). With a constant density (every
    weight equal to c) the weighted problem is c S: eigenvalues scale by c, eigenvectors and hence the STD-filter image
    do not change, the LSQ image scales by c."""
    rng = np.random.default_rng(35)
    xyz, dirs, wl = _tiny_case(rng, n_ant=7, n=8)
    e_u, e_v = np.array([1.0, 0, 0]), np.array([0, 1.0, 0])
    cell = 1e-3                                                     # far smaller than any baseline difference
    dens = oracle.uv_density([(xyz, wl)], e_u, e_v, cell)
    w = oracle.uniform_weights(xyz, wl, e_u, e_v, cell, dens)
    assert np.array_equal(w, np.where(np.eye(7, dtype=bool), 1.0 / 7.0, 1.0))
    assert np.array_equal(w, w.T)
    S = _random_sky_S(rng, xyz, wl)
    lam_w, B_w = oracle.eig_stage(S, None, xyz, wl, 7, vis_weights=np.full((7, 7), 0.25))
    lam_n, B_n = oracle.eig_stage(S, None, xyz, wl, 7)
    assert np.allclose(lam_w, 0.25 * lam_n, rtol=1e-12)
    iv = np.array([[0.0, 1e9]])
    img_w = oracle.collect(S, None, xyz, wl, 7, iv, dirs, vis_weights=np.full((7, 7), 0.25))
    img_n = oracle.collect(S, None, xyz, wl, 7, iv, dirs)
    assert np.allclose(img_w, 0.25 * img_n, rtol=1e-10)
    std_w = oracle.collect(S, None, xyz, wl, 7, iv, dirs, filt="std", vis_weights=np.full((7, 7), 0.25))
    std_n = oracle.collect(S, None, xyz, wl, 7, iv, dirs, filt="std")
    assert np.allclose(std_w, std_n, rtol=1e-10)


def test_uniform_weighting_equals_linear_solve_form(oracle):
    """P4 with weights: with all eigenpairs kept, the sum over levels equals a^H G^-1 (S o Wt) G^-1 a computed by a
    linear solve — the weights act on the visibilities and on nothing else. Also: the density is symmetric under
    b -> -b, so the weights are symmetric and S o Wt stays Hermitian."""
    rng = np.random.default_rng(36)
    xyz, dirs, wl = _tiny_case(rng, n_ant=9, n=8)
    e_u, e_v = np.array([1.0, 0, 0]), np.array([0, 1.0, 0])
    cell = 20.0                                                     # coarse: several baselines per cell
    dens = oracle.uv_density([(xyz, wl)], e_u, e_v, cell)
    assert all(dens[(-a, -b)] == c for (a, b), c in dens.items()) and max(dens.values()) > 2
    Wt = oracle.uniform_weights(xyz, wl, e_u, e_v, cell, dens)
    assert np.array_equal(Wt, Wt.T)
    S = _random_sky_S(rng, xyz, wl)
    lam, _ = oracle.eig_stage(S, None, xyz, wl, 9, vis_weights=Wt)
    iv = np.array([[min(lam.min(), 0) * 2 - 1, 0.0], [np.nextafter(0.0, 1), lam.max() * 2]])   # a negative and a positive level
    img = oracle.collect(S, None, xyz, wl, 9, iv, dirs, vis_weights=Wt)
    G = oracle.gram(xyz, None, wl)
    A = steering(xyz, dirs, wl)                                     # (n_ant, n_pix)
    X = np.linalg.solve(G, A)
    want = np.real(np.einsum("ij,ik,kj->j", X.conj(), S.astype(np.complex128) * Wt, X))
    assert np.allclose(img.sum(axis=0), want, rtol=1e-9, atol=1e-9 * np.abs(want).max())


# ---------------------------------------------------------------------------------- NUFFT synthesis, direct form (oracle slice)
def test_nufft_direct_equals_standard_synthesis(oracle):
    """Eq. 16: Psi V' Psi^* = sum_a lambda_a |eps_a|^2 — the baseline-domain double sum (Eq. 18-19, 21) and Standard
    Synthesis (Eq. 15, 20) evaluate the same images; also with a beamforming matrix and a standardized filter."""
    rng = np.random.default_rng(44)
    xyz, pix, wl = _tiny_case(rng, n_ant=6, n=6)
    Wb = (rng.normal(size=(6, 4)) + 1j * rng.normal(size=(6, 4)))
    for W in (None, Wb):
        S = _random_sky_S(rng, xyz, wl, W=W)
        lam, B = oracle.eig_stage(S, W, xyz, wl, S.shape[0])
        iv = np.array([[lam[1] * 0.999, 1e9], [0.0, lam[1] * 0.999]])
        for filt in ("lsq", "std"):
            D = oracle.level_weights(lam, iv, filt)
            want = oracle.synth(B, D, xyz, pix, wl)
            got, imag = oracle.nufft_direct(B, D, xyz, pix, wl)
            assert np.allclose(got, want, rtol=1e-11, atol=1e-11 * np.abs(want).max())
            assert imag <= 1e-11 * np.abs(want).max()


def test_nufft_direct_two_antennas_by_hand(oracle):
    """V' = [[a, c], [conj(c), b]], baseline d along x: I(l) = a + b + 2 Re(c exp(-2 pi i d l / lambda)) — typed by hand."""
    d, wl = 9.0, 3.0
    xyz = np.array([[d, 0.0, 0.0], [0.0, 0.0, 0.0]])
    l = np.linspace(-0.3, 0.3, 25)
    pix = np.column_stack([l, np.zeros_like(l), np.sqrt(1 - l * l)])
    B = np.array([[0.7 + 0.2j, 0.1 - 0.4j], [-0.3 + 0.5j, 0.6 + 0.1j]])
    D = np.array([[2.0, 0.5]])
    V = oracle.gram_corrected_visibilities(B, D)[0]
    assert np.allclose(V, V.conj().T)
    want = V[0, 0].real + V[1, 1].real + 2 * np.real(V[0, 1] * np.exp(-2j * np.pi * d * l / wl))
    got, imag = oracle.nufft_direct(B, D, xyz, pix, wl)
    assert np.allclose(got[0], want, rtol=1e-13, atol=1e-13) and imag < 1e-13
