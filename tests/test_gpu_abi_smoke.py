"""The plain-C client of include/pn.h (tests/abi_smoke.c) built with gcc -std=c11 -pedantic and run on the GPU: header and
library agree on every argument type of the calls a user makes, and the hand values of tests/golden/n2_circular.txt come
back through the C entry points."""
import subprocess

import pytest

from tests.test_host_abi import _build_abi_smoke

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


def test_c_client_runs_the_golden_case(tmp_path):
    exe = _build_abi_smoke(tmp_path)
    r = subprocess.run([str(exe)], capture_output=True, text=True, timeout=120)
    assert r.returncode == 0, r.stderr
    assert r.stdout.startswith("ABI_SMOKE_OK")
