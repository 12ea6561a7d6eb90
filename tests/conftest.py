import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def oracle():
    from oracle import bluebild_oracle
    bluebild_oracle.build()
    return bluebild_oracle


def pytest_sessionfinish(session, exitstatus):
    """Achieved parity errors (tests/helpers.record_parity) -> one JSON file, so that the numbers behind the
    pass/fail verdicts are on file (profiles/ holds the copy of the last GPU run)."""
    try:
        import helpers
    except Exception:
        return
    if not helpers.PARITY_RECORDS:
        return
    import json
    path = os.environ.get("BB_PARITY_JSON", os.path.join(ROOT, "gpurun_out", "parity_errors.json"))
    os.makedirs(os.path.dirname(path), exist_ok=True)
    with open(path, "w") as f:
        json.dump({"tolerance": {"rel_l2": helpers.REL_L2_TOL, "max_abs_over_peak": helpers.MAX_ABS_TOL},
                   "records": helpers.PARITY_RECORDS}, f, indent=1)
