"""ctypes loader for the CPU oracle (oracle/pn_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It never touches CUDA and never
imports the product package.

Two builds of the SAME source:
  "ref"  : real = long double, -O2 -ffp-contract=off          -> parity oracle
  "fast" : real = double, -O3 -march=native (-DORACLE_FAST)   -> timed CPU baseline
Both are compiled with OpenMP over the independent outer index only.  The shared objects are
built on demand next to the source (git-ignored); the "fast" build is keyed by the host's CPU
flags so an object built on another machine is never loaded.
"""
from __future__ import annotations

import ctypes
import hashlib
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "pn_oracle.c"
_LIBS: dict[str, ctypes.CDLL] = {}

# `terms` bit mask of the NEXT rows; 0 = the hot path
CROSS_STAR = 1  # [a_i]_Cross, Eq. 2.6
CROSS_BH = 2    # [a_1]_Cross, Eq. 2.3

N_ENERGY_TERMS = 11
ENERGY_TERM_NAMES = ("T1", "T2", "T3", "T4", "P1", "P2", "P3", "P4", "P5", "P6", "P7")


def _cpu_key() -> str:
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("flags"):
                    return hashlib.sha1(line.encode()).hexdigest()[:10]
    except OSError:
        pass
    return "generic"


def lib_path(kind: str) -> Path:
    if kind == "ref":
        return _HERE / "liboracle_ref.so"
    if kind == "fast":
        return _HERE / f"liboracle_fast_{_cpu_key()}.so"
    raise ValueError(kind)


def build(kind: str = "ref", force: bool = False) -> Path:
    """Compile the oracle with gcc (idempotent)."""
    out = lib_path(kind)
    if not force and out.exists() and out.stat().st_mtime >= _SRC.stat().st_mtime:
        return out
    common = ["gcc", "-std=c11", "-shared", "-fPIC", "-fopenmp", "-Wall", "-Wextra"]
    if kind == "ref":
        flags = ["-O2", "-ffp-contract=off"]
    else:
        flags = ["-O3", "-march=native", "-DORACLE_FAST"]
    tmp = out.with_suffix(f".tmp{os.getpid()}.so")
    subprocess.run(common + flags + [str(_SRC), "-o", str(tmp), "-lm"], check=True)
    os.replace(tmp, out)
    return out


def _load(kind: str) -> ctypes.CDLL:
    if kind in _LIBS:
        return _LIBS[kind]
    lib = ctypes.CDLL(str(build(kind)))
    dp = ctypes.POINTER(ctypes.c_double)
    ip = ctypes.POINTER(ctypes.c_int64)
    i64, dbl = ctypes.c_int64, ctypes.c_double
    lib.oracle_accel.argtypes = [i64, dp, dbl, dbl, dbl, dp, dp, dp]
    lib.oracle_accel_rows.argtypes = [i64, dp, dbl, dbl, dbl, dp, dp, i64, ip, dp]
    lib.oracle_step.argtypes = [i64, dp, dbl, dbl, dbl, dp, dp, dbl, i64]
    lib.oracle_energy.argtypes = [i64, dp, dbl, dbl, dbl, dp, dp, dp, dp]
    lib.oracle_momentum.argtypes = [i64, dp, dbl, dbl, dbl, dp, dp, dp]
    lib.oracle_momentum.restype = ctypes.c_int
    lib.oracle_accel_rows_terms.argtypes = [i64, dp, dbl, dbl, dbl, dp, dp, i64, ip, ctypes.c_int, dp]
    lib.oracle_step_terms.argtypes = [i64, dp, dbl, dbl, dbl, dp, dp, dbl, i64, ctypes.c_int]
    for f in (lib.oracle_accel, lib.oracle_accel_rows, lib.oracle_step, lib.oracle_energy, lib.oracle_accel_rows_terms,
              lib.oracle_step_terms):
        f.restype = ctypes.c_int
    lib.oracle_set_threads.argtypes = [ctypes.c_int]
    lib.oracle_set_threads.restype = None
    _LIBS[kind] = lib
    return lib


def _d(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _prep(mass, pos, vel):
    mass = np.ascontiguousarray(mass, dtype=np.float64)
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    vel = np.ascontiguousarray(vel, dtype=np.float64)
    n = mass.shape[0]
    if pos.shape != (n, 3) or vel.shape != (n, 3):
        raise ValueError("pos and vel must have shape (N, 3) with N = len(mass)")
    return n, mass, pos, vel


def _check(rc: int, what: str):
    if rc != 0:
        raise ValueError(f"{what} failed with oracle error code {rc}")


class Oracle:
    """The paper's hot path on the host.  Body 0 is the massive object (mass[0] = M)."""

    def __init__(self, mass, G: float, c: float, softening: float, kind: str = "ref", threads: int | None = None,
                 terms: int = 0):
        self.kind = kind
        self.terms = int(terms)
        self.lib = _load(kind)
        self.mass = np.ascontiguousarray(mass, dtype=np.float64).copy()
        self.N = int(self.mass.shape[0])
        self.G, self.c, self.eps = float(G), float(c), float(softening)
        if threads is not None:
            self.lib.oracle_set_threads(int(threads))

    @property
    def max_threads(self) -> int:
        return int(self.lib.oracle_max_threads())

    @property
    def mantissa_bits(self) -> int:
        return int(self.lib.oracle_mantissa_bits())

    def accel(self, pos, vel) -> np.ndarray:
        return self.accel_rows(pos, vel, np.arange(self.N, dtype=np.int64))

    def accel_rows(self, pos, vel, rows) -> np.ndarray:
        n, m, pos, vel = _prep(self.mass, pos, vel)
        rows = np.ascontiguousarray(rows, dtype=np.int64)
        acc = np.empty((rows.shape[0], 3), dtype=np.float64)
        rp = rows.ctypes.data_as(ctypes.POINTER(ctypes.c_int64))
        _check(
            self.lib.oracle_accel_rows_terms(n, _d(m), self.G, self.c, self.eps, _d(pos), _d(vel), rows.shape[0], rp,
                                             self.terms, _d(acc)),
            "oracle_accel_rows_terms",
        )
        return acc

    def step(self, pos, vel, dt: float, nsteps: int = 1):
        """Returns (pos, vel) after nsteps classical-RK4 steps; inputs are not modified."""
        n, m, pos, vel = _prep(self.mass, pos, vel)
        pos, vel = pos.copy(), vel.copy()
        _check(self.lib.oracle_step_terms(n, _d(m), self.G, self.c, self.eps, _d(pos), _d(vel), float(dt), int(nsteps),
                                          self.terms), "oracle_step_terms")
        return pos, vel

    def momentum(self, pos, vel) -> np.ndarray:
        """Total 1PN momentum, Eq. 2.8 in the reading R16 of DESIGN.md."""
        n, m, pos, vel = _prep(self.mass, pos, vel)
        out = np.zeros(3, dtype=np.float64)
        _check(self.lib.oracle_momentum(n, _d(m), self.G, self.c, self.eps, _d(pos), _d(vel), _d(out)), "oracle_momentum")
        return out

    def energy(self, pos, vel, terms: bool = False):
        n, m, pos, vel = _prep(self.mass, pos, vel)
        e = ctypes.c_double(0.0)
        t = np.zeros(N_ENERGY_TERMS, dtype=np.float64)
        _check(
            self.lib.oracle_energy(n, _d(m), self.G, self.c, self.eps, _d(pos), _d(vel), ctypes.byref(e), _d(t)),
            "oracle_energy",
        )
        return (e.value, dict(zip(ENERGY_TERM_NAMES, t.tolist()))) if terms else e.value
