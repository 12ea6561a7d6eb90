"""Writes tests/golden/*.txt. Calls ONLY oracle/ (never the CUDA path): the stored values are the oracle's own,
kept so that an unintended change of the oracle's arithmetic shows up as a diff (tests/test_golden.py).
The paper prints no worked numeric example of Standard Synthesis, so there is no
paper-valued fixture; the closed-form fixture below is the textbook two-element fringe and the uniform-line-array
Dirichlet kernel (the forms pinned in tests/test_oracle_pins.py P6), tabulated to 17 digits.

    python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))
from oracle import bluebild_oracle as oracle  # noqa: E402


def tiny_case():
    """Deterministic 6-antenna, 3-eigenpair, 2-level, 5-pixel case with round numbers (no random generator)."""
    xyz = np.array([[0, 0, 0], [10, 0, 0], [0, 14, 1], [-7, 5, 0], [3, -9, 2], [12, 11, -1]], dtype=np.float64)
    k = np.arange(6)[:, None] + 1.0
    c = np.arange(3)[None, :] + 1.0
    B = (np.cos(0.7 * k * c) + 1j * np.sin(0.3 * k + c)) / 4.0
    D = np.array([[2.0, 0.0, 0.5], [0.0, 1.25, 0.0]])
    lm = np.array([[0.0, 0.0], [0.05, -0.02], [-0.08, 0.03], [0.01, 0.09], [-0.04, -0.07]])
    pix = np.column_stack([lm, np.sqrt(1.0 - np.sum(lm * lm, axis=1))])
    return B, D, xyz, pix, 3.0


def main():
    B, D, xyz, pix, wl = tiny_case()
    img = oracle.synth(B, D, xyz, pix, wl)
    with open(os.path.join(HERE, "oracle_tiny_case.txt"), "w") as f:
        f.write("# oracle.synth on make_golden.tiny_case(): rows = levels, columns = pixels (PAPER.md Alg. 2, Eq. 20)\n")
        for row in img:
            f.write(" ".join("%.17e" % v for v in row) + "\n")
    # closed forms (not computed by the oracle): two-element fringe 1 + cos(2 pi d l / lambda) and the Dirichlet kernel
    d, wl2, n = 7.0, 2.0, 8
    l = np.linspace(-0.3, 0.3, 7)
    fringe = 1.0 + np.cos(2.0 * np.pi * d * l / wl2)
    with np.errstate(invalid="ignore", divide="ignore"):
        x = np.pi * 1.5 * l / wl2
        dirichlet = np.where(np.abs(np.sin(x)) < 1e-300, float(n), np.sin(n * x) ** 2 / (n * np.sin(x) ** 2))
    with open(os.path.join(HERE, "closed_forms.txt"), "w") as f:
        f.write("# l, two-element fringe (d = 7 m, lambda = 2 m), 8-element line array at 1.5 m spacing (lambda = 2 m)\n")
        for a, b, c in zip(l, fringe, dirichlet):
            f.write("%.17e %.17e %.17e\n" % (a, b, c))


if __name__ == "__main__":
    main()
