"""Build libpn.so (the C-ABI CUDA library) and libpn_bench.so (bench.py's pipe-peak probes, include/pn_bench.h) in-tree
for sm_100a with nvcc.

    python -m paper_1801_07986_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The shared object lands next to this file (git-ignored,
but it travels to the GPU box with the working tree).
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys
from pathlib import Path

PKG = Path(__file__).resolve().parent
CSRC = PKG / "csrc"
INCLUDE = PKG.parent / "include"
LIB = PKG / "libpn.so"
SOURCES = [CSRC / "pn_api.cu", CSRC / "pn_noalloc.cu"]
HEADERS = sorted(CSRC.glob("*.cuh")) + [INCLUDE / "pn.h"]
BENCH_LIB = PKG / "libpn_bench.so"  # roofline-denominator probes for bench.py; not linked into or loaded by the product
BENCH_SOURCES = [CSRC / "pn_bench.cu"]
BENCH_HEADERS = [INCLUDE / "pn_bench.h"]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17",
    "--fmad=true",  # fp64 contraction is part of the kernel design; the oracle is built with -ffp-contract=off
    "-Xcompiler", "-fPIC,-O2,-Wall",
    "-shared",
]


def nvcc_path() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and Path(cand).exists():
            return cand
    raise RuntimeError("nvcc not found; the CUDA library cannot be built (there is no CPU fallback)")


def _stale(lib: Path, deps) -> bool:
    if not lib.exists():
        return True
    t = lib.stat().st_mtime
    return any(p.stat().st_mtime > t for p in list(deps) + [Path(__file__)])


def needs_build() -> bool:
    return _stale(LIB, SOURCES + HEADERS) or _stale(BENCH_LIB, BENCH_SOURCES + BENCH_HEADERS)


def _nvcc(sources, out: Path, verbose: bool) -> None:
    tmp = out.with_suffix(f".tmp{os.getpid()}.so")
    cmd = [nvcc_path(), *NVCC_FLAGS, f"-I{INCLUDE}", *(["-Xptxas", "-v"] if verbose else []),
           *map(str, sources), "-o", str(tmp)]
    if verbose:
        print(" ".join(cmd), file=sys.stderr)
    subprocess.run(cmd, check=True)
    os.replace(tmp, out)


def build(force: bool = False, verbose: bool = False) -> Path:
    if force or _stale(LIB, SOURCES + HEADERS):
        _nvcc(SOURCES, LIB, verbose)
    if force or _stale(BENCH_LIB, BENCH_SOURCES + BENCH_HEADERS):
        _nvcc(BENCH_SOURCES, BENCH_LIB, verbose)
    return LIB


if __name__ == "__main__":
    out = build(force="--force" in sys.argv, verbose="--verbose" in sys.argv)
    print(out)
