import sys
from fractions import Fraction
from pathlib import Path

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parent.parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

GOLDEN = Path(__file__).resolve().parent / "golden"


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


def _num(tok: str) -> float:
    return float(Fraction(tok))


def load_golden(name: str) -> dict:
    """Parse a tests/golden/*.txt fixture (see tests/golden/README.md)."""
    out = {}
    for line in (GOLDEN / name).read_text().splitlines():
        line = line.split("#", 1)[0].strip()
        if not line:
            continue
        key, *vals = line.split()
        out[key] = np.array([_num(v) for v in vals], dtype=np.float64)
    n = out["mass"].shape[0]
    for k in ("pos", "vel", "acc", "acc_newton", "acc_cross_star", "acc_cross_full"):
        if k in out:
            out[k] = out[k].reshape(n, 3)
    if "cross_star" in out:  # [a_i]_Cross of the stars only (bodies 1 .. N-1)
        out["cross_star"] = out["cross_star"].reshape(n - 1, 3)
    for k in ("G", "c", "eps", "eps2", "energy", "energy_newton"):
        if k in out:
            out[k] = float(out[k][0])
    if "eps" not in out:
        out["eps"] = float(np.sqrt(out["eps2"]))
    return out


GOLDEN_CASES = ["n2_circular.txt", "n2_oblique.txt", "n3_345.txt", "n3_345_softened.txt"]


@pytest.fixture(params=GOLDEN_CASES)
def golden_case(request):
    return load_golden(request.param)


def rel_err_rows(a, ref):
    """DESIGN.md reading R10: err_i = max_k |a_ik - ref_ik| / ||ref_i||_2."""
    a, ref = np.asarray(a), np.asarray(ref)
    nrm = np.linalg.norm(ref, axis=1)
    nrm = np.where(nrm > 0, nrm, 1.0)
    return np.abs(a - ref).max(axis=1) / nrm
