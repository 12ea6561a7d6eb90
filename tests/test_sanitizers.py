"""the C++ oracle under AddressSanitizer + UndefinedBehaviorSanitizer. compute-sanitizer is
closed on the GPU pool, so the CUDA path has no sanitizer run; the oracle that judges it does."""
import glob
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

SCRIPT = r"""
import numpy as np
from oracle import bluebild_oracle as o
rng = np.random.default_rng(5)
for n_ant, n_eig, L, n_pix, threads in ((1, 1, 1, 1, 1), (7, 3, 2, 33, 3), (16, 8, 2, 257, 0), (5, 5, 4, 64, 8)):
    B = rng.normal(size=(n_ant, n_eig)) + 1j * rng.normal(size=(n_ant, n_eig))
    D = rng.uniform(0, 2, size=(L, n_eig))
    xyz = rng.uniform(-50, 50, size=(n_ant, 3))
    v = rng.normal(size=(n_pix, 3)); pix = v / np.linalg.norm(v, axis=1, keepdims=True)
    a = o.synth(B, D, xyz, pix, 2.0, n_threads=threads)
    b = o.brute(B, D, xyz, pix, 2.0)
    assert np.allclose(a, b, rtol=1e-11, atol=1e-11 * np.abs(b).max())
o.synth(np.zeros((3, 2), complex), np.zeros((1, 2)), np.zeros((3, 3)), np.zeros((0, 3)), 1.0)      # empty image
print("sanitized oracle ok")
"""


def _asan_runtime():
    out = subprocess.run(["g++", "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip()
    return out if os.path.isabs(out) and os.path.exists(out) else None


def test_oracle_under_asan_and_ubsan():
    rt = _asan_runtime()
    if rt is None:
        pytest.skip("g++ has no libasan on this machine")
    env = dict(os.environ, BB_ORACLE_SANITIZE="1", LD_PRELOAD=rt, ASAN_OPTIONS="detect_leaks=0:abort_on_error=0:exitcode=99",
               UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1", PYTHONPATH=ROOT)
    r = subprocess.run([sys.executable, "-c", SCRIPT], cwd=ROOT, env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0 and "sanitized oracle ok" in r.stdout, (r.returncode, r.stdout[-2000:], r.stderr[-4000:])
    assert "ERROR: AddressSanitizer" not in r.stderr and "runtime error" not in r.stderr, r.stderr[-4000:]
