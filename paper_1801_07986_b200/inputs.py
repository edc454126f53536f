"""Seeded synthetic inputs for the limited-1PN hot path (BASELINE.json configs 1-5).

This module serves BOTH the CUDA path's tests/bench and the CPU oracle's tests.  It contains
none of the method's arithmetic (no accelerations, no energies, no integrator) -- only the
recipes of DESIGN.md "Input recipe" that turn a seed into (mass, pos, vel) host arrays in
fp64.  numpy only; never imports the CUDA binding or the oracle.

Conventions (readings R7, R15): body 0 is the massive object ("#1" in the paper,
PAPER.md:41) of mass M, at the origin, at rest; stars are bodies 1..N_s and are recentred so
that sum m_i x_i = 0 and sum m_i v_i = 0 (the paper's equations assume the zero-momentum
frame).  G = 1 throughout.  The paper's own workloads are synthetic too (random spherical
shell), so these stand in for nothing external.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np


@dataclass
class Problem:
    """One workload: constants of pn_create + initial state + run parameters."""

    name: str
    mass: np.ndarray  # (N,)  mass[0] = M
    pos: np.ndarray  # (N, 3)
    vel: np.ndarray  # (N, 3)
    G: float
    c: float
    softening: float
    dt: float
    nsteps: int
    meta: dict = field(default_factory=dict)

    @property
    def N(self) -> int:
        return int(self.mass.shape[0])

    @property
    def n_stars(self) -> int:
        return self.N - 1

    @property
    def pairs_per_eval(self) -> int:
        """Ordered star-star pairs (i, j != i) visited by one force evaluation."""
        ns = self.n_stars
        return ns * (ns - 1)


def _isotropic(rng: np.random.Generator, n: int) -> np.ndarray:
    z = rng.uniform(-1.0, 1.0, n)
    phi = rng.uniform(0.0, 2.0 * np.pi, n)
    s = np.sqrt(1.0 - z * z)
    return np.stack([s * np.cos(phi), s * np.sin(phi), z], axis=1)


def _assemble(m_star: np.ndarray, x: np.ndarray, v: np.ndarray, M: float):
    """Recentre the stars (zero mass-weighted mean position and velocity), put the BH at the origin at rest."""
    w = m_star / m_star.sum()
    x = x - (w[:, None] * x).sum(axis=0)
    v = v - (w[:, None] * v).sum(axis=0)
    n = m_star.shape[0] + 1
    mass = np.empty(n)
    mass[0], mass[1:] = M, m_star
    pos = np.zeros((n, 3))
    vel = np.zeros((n, 3))
    pos[1:], vel[1:] = x, v
    return mass, np.ascontiguousarray(pos), np.ascontiguousarray(vel)


def plummer_stars(n_stars: int, rng: np.random.Generator):
    """Plummer sphere, scale radius a = 1, G M_tot = 1, isotropic equilibrium velocities
    (Aarseth-Henon-Wielen recipe): r = (u^(-2/3) - 1)^(-1/2);  speed = q sqrt(2) (1+r^2)^(-1/4)
    with q drawn by rejection from g(q) = q^2 (1-q^2)^(7/2) (accept if 0.1 u2 < g(u1)).  Untruncated."""
    u = rng.uniform(0.0, 1.0, n_stars)
    u = np.where(u <= 0.0, 0.5, u)
    r = 1.0 / np.sqrt(u ** (-2.0 / 3.0) - 1.0)
    x = r[:, None] * _isotropic(rng, n_stars)
    q = np.empty(n_stars)
    todo = np.arange(n_stars)
    while todo.size:
        u1 = rng.uniform(0.0, 1.0, todo.size)
        u2 = rng.uniform(0.0, 1.0, todo.size)
        ok = 0.1 * u2 < u1 * u1 * (1.0 - u1 * u1) ** 3.5
        q[todo[ok]] = u1[ok]
        todo = todo[~ok]
    speed = q * np.sqrt(2.0) * (1.0 + r * r) ** (-0.25)
    v = speed[:, None] * _isotropic(rng, n_stars)
    return x, v


def plummer_bh(n_stars: int, seed: int, M: float = 0.1, c: float = 100.0, softening: float = 1e-3,
               dt: float = 1e-4, nsteps: int = 100, name: str | None = None) -> Problem:
    """Configs 1, 2, 4: equal-mass Plummer sphere of total mass 1 + central BH of mass M."""
    rng = np.random.default_rng(seed)
    x, v = plummer_stars(n_stars, rng)
    m_star = np.full(n_stars, 1.0 / n_stars)
    mass, pos, vel = _assemble(m_star, x, v, M)
    return Problem(name or f"plummer_bh_N1+{n_stars}_seed{seed}", mass, pos, vel, 1.0, c, softening, dt, nsteps,
                   {"model": "plummer+bh", "seed": seed})


def cusp_sigma2(r: np.ndarray, M: float, n_stars: int, m: float, r_min: float) -> np.ndarray:
    """Isotropic Jeans dispersion for rho ~ r^(-7/4) on [r_min, 1] around a point mass M (G = 1):
    sigma^2(r) = r^(7/4) int_r^1 s^(-7/4) [M + M_*(<s)] s^(-2) ds,
    M_*(<s) = n m (s^(5/4) - b)/(1 - b),  b = r_min^(5/4);  closed form below."""
    b = r_min ** 1.25
    t1 = M / (2.75 * r) * (1.0 - r ** 2.75)
    t2 = (n_stars * m / (1.0 - b)) * r ** 1.75 * ((2.0 / 3.0) * (r ** -1.5 - 1.0) - (4.0 * b / 11.0) * (r ** -2.75 - 1.0))
    return t1 + t2


def cusp_bh(n_stars: int = 65535, seed: int = 2, M: float = 1.0, mass_ratio: float = 1e4, r_min: float = 1e-3,
            softening: float = 1e-4, dt: float = 1e-5, nsteps: int = 20, name: str | None = None) -> Problem:
    """Config 3: Bahcall-Wolf cusp rho ~ r^(-7/4), r in [r_min, 1], Gaussian isotropic velocities with the Jeans
    dispersion; c = 10 sqrt(G M / r_min) so the innermost circular speed is 0.1 c."""
    rng = np.random.default_rng(seed)
    m = M / mass_ratio
    b = r_min ** 1.25
    u = rng.uniform(0.0, 1.0, n_stars)
    r = (b + u * (1.0 - b)) ** 0.8
    x = r[:, None] * _isotropic(rng, n_stars)
    sig = np.sqrt(np.maximum(cusp_sigma2(r, M, n_stars, m, r_min), 0.0))
    v = sig[:, None] * rng.standard_normal((n_stars, 3))
    mass, pos, vel = _assemble(np.full(n_stars, m), x, v, M)
    c = 10.0 * np.sqrt(M / r_min)
    return Problem(name or f"cusp_bh_N1+{n_stars}_seed{seed}", mass, pos, vel, 1.0, float(c), softening, dt, nsteps,
                   {"model": "bahcall-wolf cusp+bh", "seed": seed})


def uniform_ball_bh(k: int, M: float = 0.1, c: float = 100.0, softening: float = 1e-3, sigma: float = 0.3,
                    name: str | None = None) -> Problem:
    """Config 5: N_s = 2^k - 1 stars uniform in the unit ball, Gaussian velocities, seed = k, total star mass 1."""
    n_stars = (1 << k) - 1
    rng = np.random.default_rng(k)
    r = rng.uniform(0.0, 1.0, n_stars) ** (1.0 / 3.0)
    x = r[:, None] * _isotropic(rng, n_stars)
    v = sigma * rng.standard_normal((n_stars, 3))
    mass, pos, vel = _assemble(np.full(n_stars, 1.0 / n_stars), x, v, M)
    return Problem(name or f"uniform_ball_bh_k{k}", mass, pos, vel, 1.0, c, softening, 0.0, 0,
                   {"model": "uniform ball+bh", "seed": k})


def cold_shell_bh(n_total: int = 10000, seed: int = 0, name: str | None = None) -> Problem:
    """The paper's own model as a stand-in for its timing runs, whose initial conditions are not
    given: N - 1 equal-mass stars, m = 1e-4, at rest, uniform in the shell 1 < r < 10; a massive object
    of mass M = 100 m = 0.01 at the origin; c = G = 1, softening 1e-3, dt = 2^-15.  (The paper draws the positions
    with an LCG whose constants it does not give; here numpy's PCG64 with the given seed.)"""
    n_stars = n_total - 1
    rng = np.random.default_rng(seed)
    r = (1.0 + rng.uniform(0.0, 1.0, n_stars) * (10.0 ** 3 - 1.0)) ** (1.0 / 3.0)
    x = r[:, None] * _isotropic(rng, n_stars)
    m = 1e-4
    mass = np.concatenate([[100.0 * m], np.full(n_stars, m)])
    pos = np.vstack([np.zeros(3), x])
    vel = np.zeros_like(pos)
    return Problem(name or f"cold_shell_N{n_total}_seed{seed}", mass, pos, vel, 1.0, 1.0, 1e-3, 2.0 ** -15, 32,
                   {"model": "cold shell+bh (paper)", "seed": seed})


def config(idx: int, **kw) -> Problem:
    """BASELINE.json configs by number (1-based, as SURVEY.md section 8(d) lists them)."""
    if idx == 1:
        return plummer_bh(1023, 0, M=0.1, dt=1e-4, nsteps=100, name="config1_plummer_N1+1023", **kw)
    if idx == 2:
        return plummer_bh(16383, 1, M=0.1, dt=1e-4, nsteps=50, name="config2_plummer_N1+16383", **kw)
    if idx == 3:
        return cusp_bh(65535, 2, name="config3_cusp_N1+65535", **kw)
    if idx == 4:
        return plummer_bh(262143, 3, M=0.05, dt=1e-4, nsteps=10, name="config4_plummer_N1+262143", **kw)
    raise ValueError("config index must be 1..4; use uniform_ball_bh(k) for the config-5 sweep")


def random_small(n_stars: int, seed: int, M: float = 1.0, m_scale: float = 1e-2, c: float = 10.0,
                 softening: float = 0.0, bh_moving: bool = False) -> Problem:
    """Tiny generic system for brute-force tests: unequal masses, O(1) separations, O(0.3) speeds."""
    rng = np.random.default_rng(seed)
    x = rng.uniform(-2.0, 2.0, (n_stars, 3))
    v = 0.3 * rng.standard_normal((n_stars, 3))
    m_star = m_scale * rng.uniform(0.5, 1.5, n_stars)
    mass, pos, vel = _assemble(m_star, x, v, M)
    if bh_moving:
        pos[0] = rng.uniform(-0.2, 0.2, 3)
        vel[0] = 0.05 * rng.standard_normal(3)
    return Problem(f"random_small_{n_stars}_seed{seed}", mass, pos, vel, 1.0, c, softening, 1e-3, 10,
                   {"model": "random small", "seed": seed})
