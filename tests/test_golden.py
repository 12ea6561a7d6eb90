"""Stored fixtures under tests/golden/ (written by tests/golden/make_golden.py, which calls only oracle/)."""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.join(HERE, "golden"))


def _load(name):
    return np.loadtxt(os.path.join(HERE, "golden", name), comments="#", ndmin=2)


def test_oracle_matches_its_stored_tiny_case(oracle):
    """Regression guard: the oracle's arithmetic has not drifted since the fixture was written."""
    import make_golden
    B, D, xyz, pix, wl = make_golden.tiny_case()
    ref = _load("oracle_tiny_case.txt")
    got = oracle.synth(B, D, xyz, pix, wl)
    assert got.shape == ref.shape
    assert np.allclose(got, ref, rtol=1e-13, atol=0)
    assert np.allclose(oracle.brute(B, D, xyz, pix, wl), ref, rtol=1e-12, atol=0)


def test_oracle_reproduces_tabulated_closed_forms(oracle):
    """closed_forms.txt holds textbook values (fringe of a two-element interferometer, Dirichlet kernel of a
    uniform line array) that were NOT computed by the oracle."""
    tab = _load("closed_forms.txt")
    l = tab[:, 0]
    pix = np.column_stack([l, np.zeros_like(l), np.sqrt(1 - l * l)])
    two = np.array([[-3.5, 0, 0], [3.5, 0, 0]])
    img = oracle.synth(np.ones((2, 1)) / np.sqrt(2.0), [[1.0]], two, pix, 2.0)[0]
    assert np.allclose(img, tab[:, 1], rtol=0, atol=1e-12)
    line = np.column_stack([1.5 * np.arange(8), np.zeros(8), np.zeros(8)])
    img = oracle.synth(np.ones((8, 1)) / np.sqrt(8.0), [[1.0]], line, pix, 2.0)[0]
    assert np.allclose(img, tab[:, 2], rtol=0, atol=1e-11)
