"""CPU-only checks of the C-ABI library: it builds, loads, exports every symbol include/pn.h
declares, and refuses to work (loudly) without a GPU -- no CPU fallback.  No compute calls."""
import ctypes
import re
from pathlib import Path

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def lib():
    from paper_1801_07986_b200 import build

    build.build()
    from paper_1801_07986_b200 import binding

    return binding.load_library()


def _declared_symbols():
    text = (ROOT / "include" / "pn.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(pn_[a-z_0-9]+)\s*\(", text)))


def test_header_symbols_all_exported(lib):
    from paper_1801_07986_b200 import binding

    declared = _declared_symbols()
    assert len(declared) >= 15
    assert sorted(binding.EXPORTS) == declared
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in pn.h but not exported by libpn.so"


def test_version_string(lib):
    assert b"sm_100a" in lib.pn_version()


def test_create_validates_arguments_before_touching_cuda(lib):
    from paper_1801_07986_b200 import binding

    ctx = ctypes.c_void_p(None)
    m = np.array([1.0, 1e-3])
    bad = [
        (1, m, 1.0, 10.0, 0.0),  # N < 2
        (2, np.array([1.0, -1.0]), 1.0, 10.0, 0.0),  # negative mass
        (2, np.array([0.0, 1.0]), 1.0, 10.0, 0.0),  # M <= 0
        (2, m, 0.0, 10.0, 0.0),  # G <= 0
        (2, m, 1.0, 0.0, 0.0),  # c <= 0
        (2, m, 1.0, float("nan"), 0.0),  # c NaN
        (2, m, 1.0, 10.0, -1.0),  # eps < 0
    ]
    for n, mm, G, c, eps in bad:
        rc = lib.pn_create(ctypes.byref(ctx), n, mm.ctypes.data, G, c, eps)
        assert rc == binding.PN_EINVAL
        assert not ctx.value
        assert len(lib.pn_last_error(None)) > 0


def test_no_cpu_fallback_without_gpu(lib):
    import torch

    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_1801_07986_b200 import binding

    ctx = ctypes.c_void_p(None)
    m = np.array([1.0, 1e-3])
    rc = lib.pn_create(ctypes.byref(ctx), 2, m.ctypes.data, 1.0, 10.0, 0.0)
    assert rc == binding.PN_ECUDA and not ctx.value
    assert b"no CUDA device" in lib.pn_last_error(None)


def test_null_context_is_rejected(lib):
    from paper_1801_07986_b200 import binding

    assert lib.pn_step(None, 1e-3, 1) == binding.PN_EINVAL
    assert lib.pn_destroy(None) == binding.PN_OK


def test_product_path_does_not_reference_oracle():
    """The oracle is test infrastructure: nothing in the product package may import or link it."""
    pkg = ROOT / "paper_1801_07986_b200"
    for p in list(pkg.rglob("*.py")) + list(pkg.rglob("*.cu")) + list(pkg.rglob("*.cuh")):
        text = p.read_text()
        code = "\n".join(l for l in text.splitlines() if not l.strip().startswith(("#", "//", "*", "/*")))
        assert "import oracle" not in code and "from oracle" not in code and "liboracle" not in code, p
    for p in (ROOT / "oracle").rglob("*"):
        if p.suffix in (".py", ".c", ".h"):
            for line in p.read_text().splitlines():
                if re.match(r"\s*(#\s*include|import|from)\b", line):
                    assert "paper_1801_07986_b200" not in line and "csrc" not in line and "pn.h" not in line, (p, line)


# ------------------------------------------------------------------ the header as a C header; the bench-only probe library
def _build_abi_smoke(tmp_path):
    """gcc -std=c11 -pedantic: pn.h must be a self-sufficient C header; linking checks the symbols a C client needs."""
    import subprocess

    from paper_1801_07986_b200 import build

    build.build()
    exe = tmp_path / "abi_smoke"
    cmd = ["gcc", "-std=c11", "-Wall", "-Wextra", "-Werror", "-pedantic", f"-I{ROOT / 'include'}", str(ROOT / "tests" / "abi_smoke.c"),
           f"-L{build.LIB.parent}", "-lpn", f"-Wl,-rpath,{build.LIB.parent}", "-lm", "-o", str(exe)]
    subprocess.run(cmd, check=True)
    return exe


def test_c_client_compiles_links_and_refuses_to_run_without_a_gpu(tmp_path):
    import subprocess

    import torch

    exe = _build_abi_smoke(tmp_path)
    if torch.cuda.is_available():
        pytest.skip("a GPU is present: tests/test_gpu_abi_smoke.py runs the client")
    r = subprocess.run([str(exe)], capture_output=True, text=True)
    assert r.returncode == 3 and "no CUDA device" in r.stderr  # no CPU fallback behind the C entry points either


def test_bench_probe_library_is_separate_and_exports_its_header():
    from paper_1801_07986_b200 import build

    build.build()
    text = re.sub(r"/\*.*?\*/", "", (ROOT / "include" / "pn_bench.h").read_text(), flags=re.S)
    declared = sorted(set(re.findall(r"\b(pn_bench_[a-z_0-9]+)\s*\(", text)))
    assert declared == ["pn_bench_fp32_peak", "pn_bench_fp64_peak", "pn_bench_operand_probe"]
    blib = ctypes.CDLL(str(build.BENCH_LIB))
    for name in declared:
        assert hasattr(blib, name)
    plib = ctypes.CDLL(str(build.LIB))
    for name in declared + ["pn_measure_fp64_peak"]:
        assert not hasattr(plib, name), f"{name} must not be part of the product library"
