#!/usr/bin/env python
"""Writes the long-double oracle references of the full-size BASELINE.json configs 2, 3 and 4.

    python tests/make_fullsize_refs.py [--threads T] [--only config2|config3|config4]

Calls ONLY oracle/ (the parity oracle, long-double build) and the seeded input generators; never the CUDA path.
What it stores ("run it once per build and cache the result outside git"):

  tests/cache/config3_traj.npz   (git-ignored; travels to the GPU box with the working tree)
      config 3 as BASELINE.json states it: N = 1+65535, dt = 1e-5, 20 classical-RK4 steps of the oracle from the seeded
      initial state, the state rounded to fp64 after every step (as in the config-1 test); E (Eq. 2.7)
      of the initial state and after every step; x, v of a seeded subset of rows after every step; the full final state.
  tests/golden/config3_digest.npz  (committed; a subset of the same run: E[21] and 256 rows per step)
      used by the GPU test when the cache file is absent, so a fresh checkout never has to spend the ~1.5 h of host
      time the full run costs (3.4e11 long-double pair visits for the trajectory + 21 O(N^2) energies).
  tests/cache/config2_traj.npz, tests/golden/config2_digest.npz
      the same for config 2 as stated (N = 1+16383, dt = 1e-4, 50 steps; 5.4e10 pair visits + 51 energies, about half an
      hour of host time); the digest holds 128 rows per step.
  tests/golden/config4_energy.txt  (committed; one number)
      config 4: E of the full initial set, N = 1+262143 (6.9e10 ordered pairs in long double).

Every file carries a key = sha256 of (oracle/pn_oracle.c with comments and white space removed) + the input arrays; the
tests refuse a file whose key does not match the current oracle source and inputs.
The runs are resumable: progress is kept in tests/cache/_config<n>_partial.npz after every step.
"""
from __future__ import annotations

import argparse
import hashlib
import re
import sys
import time
from pathlib import Path

import numpy as np

HERE = Path(__file__).resolve().parent
ROOT = HERE.parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

CACHE = HERE / "cache"
GOLDEN = HERE / "golden"
N_ROWS_CACHE = 2048
N_ROWS_DIGEST = 256


def oracle_source_digest() -> str:
    src = (ROOT / "oracle" / "pn_oracle.c").read_text()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    src = re.sub(r"\s+", "", src)
    return hashlib.sha256(src.encode()).hexdigest()


def ref_key(p) -> str:
    h = hashlib.sha256()
    h.update(oracle_source_digest().encode())
    for a in (p.mass, p.pos, p.vel):
        h.update(np.ascontiguousarray(a, dtype=np.float64).tobytes())
    h.update(repr((p.G, p.c, p.softening, p.dt)).encode())
    return h.hexdigest()[:32]


def sample_rows(p, n: int, seed: int = 777) -> np.ndarray:
    """Seeded subset of body rows; always holds the massive object, the first / last star and the stars nearest to and
    farthest from the massive object.  The first N_ROWS_DIGEST entries of the cache's rows are the digest's rows."""
    rng = np.random.default_rng(seed)
    r = np.linalg.norm(p.pos[1:] - p.pos[0], axis=1)
    fixed = [0, 1, p.N - 1, 1 + int(np.argmin(r)), 1 + int(np.argmax(r))]
    rest = rng.permutation(np.arange(2, p.N - 1))
    rest = rest[~np.isin(rest, fixed)]
    return np.concatenate([fixed, rest[: n - len(fixed)]]).astype(np.int64)


def make_traj(cfg: int, threads: int | None, n_rows_digest: int = N_ROWS_DIGEST) -> None:
    """Config `cfg` as stated: p.nsteps RK4 steps of the oracle, E after every step, sampled rows after every step."""
    from oracle.pn_oracle import Oracle
    from paper_1801_07986_b200 import inputs

    p = inputs.config(cfg)
    name = f"config{cfg}"
    key = ref_key(p)
    o = Oracle(p.mass, p.G, p.c, p.softening, kind="ref", threads=threads)
    rows = sample_rows(p, N_ROWS_CACHE)
    CACHE.mkdir(exist_ok=True)
    part = CACHE / f"_{name}_partial.npz"
    n = p.nsteps
    E = np.full(n + 1, np.nan)
    xr = np.full((n, rows.size, 3), np.nan)
    vr = np.full((n, rows.size, 3), np.nan)
    x, v, done = p.pos.copy(), p.vel.copy(), 0
    if part.exists():
        z = np.load(part)
        if str(z["key"]) == key:
            E, xr, vr, x, v, done = z["E"], z["x_rows"], z["v_rows"], z["x"], z["v"], int(z["done"])
            print(f"{name}: resuming after step {done}", flush=True)
    t0 = time.perf_counter()
    if np.isnan(E[0]):
        E[0] = o.energy(p.pos, p.vel)
        print(f"{name}: E0 = {E[0]!r}  ({time.perf_counter() - t0:.0f} s)", flush=True)
    for s in range(done, n):
        x, v = o.step(x, v, p.dt, 1)
        E[s + 1] = o.energy(x, v)
        xr[s], vr[s] = x[rows], v[rows]
        np.savez(part, key=key, E=E, x_rows=xr, v_rows=vr, x=x, v=v, done=s + 1)
        print(f"{name}: step {s + 1}/{n}  E = {E[s + 1]!r}  drift {(E[s + 1] - E[0]) / abs(E[0]):.6e}  "
              f"({time.perf_counter() - t0:.0f} s)", flush=True)
    meta = dict(key=key, workload=p.name, dt=p.dt, nsteps=n, oracle="oracle/pn_oracle.c, long-double build (ref)",
                script="tests/make_fullsize_refs.py")
    np.savez(CACHE / f"{name}_traj.npz", E=E, rows=rows, x_rows=xr, v_rows=vr, x_final=x, v_final=v, **meta)
    d = n_rows_digest
    np.savez(GOLDEN / f"{name}_digest.npz", E=E, rows=rows[:d], x_rows=xr[:, :d], v_rows=vr[:, :d], **meta)
    part.unlink(missing_ok=True)
    print(f"{name}: written", flush=True)


def make_config4(threads: int | None) -> None:
    from oracle.pn_oracle import Oracle
    from paper_1801_07986_b200 import inputs

    p = inputs.config(4)
    key = ref_key(p)
    o = Oracle(p.mass, p.G, p.c, p.softening, kind="ref", threads=threads)
    t0 = time.perf_counter()
    e = o.energy(p.pos, p.vel)
    (GOLDEN / "config4_energy.txt").write_text(
        "# 1PN energy, Eq. 2.7 (PAPER.md:92-94), of the full initial set of BASELINE.json config 4 (N = 1+262143,\n"
        "# Plummer + BH 0.05, seed 3, c = 100, softening 1e-3): oracle/pn_oracle.c, long-double build, every ordered\n"
        "# pair.  Written by tests/make_fullsize_refs.py (calls only oracle/); key = oracle source + inputs.\n"
        f"key {key}\nenergy {e!r}\nenergy_hex {float(e).hex()}\n")
    print(f"config4: E0 = {e!r}  ({time.perf_counter() - t0:.0f} s)", flush=True)


if __name__ == "__main__":
    ap = argparse.ArgumentParser()
    ap.add_argument("--threads", type=int, default=None)
    ap.add_argument("--only", choices=["config2", "config3", "config4"], default=None)
    a = ap.parse_args()
    if a.only in (None, "config4"):
        make_config4(a.threads)
    if a.only in (None, "config2"):
        make_traj(2, a.threads, n_rows_digest=128)
    if a.only in (None, "config3"):
        make_traj(3, a.threads)
