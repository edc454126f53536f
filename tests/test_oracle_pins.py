"""Pins for the CPU oracle (oracle/pn_oracle.c): every check compares it with something OTHER
than itself -- hand-evaluated values (tests/golden), textbook Newtonian gravity written
independently in numpy, the full N-body EIH theory in mpmath (tests/eih_reference.py), the
closed-form test-particle periastron advance, convergence order of classical RK4, and 1PN
two-body energy conservation.  CPU only.
"""
import math

import numpy as np
import pytest
from mpmath import mpf

from oracle.pn_oracle import Oracle
from paper_1801_07986_b200 import inputs
from tests import eih_reference as eih

KINDS = ["ref", "fast"]


# ------------------------------------------------------------------ hand-evaluated values
@pytest.mark.parametrize("kind", KINDS)
def test_golden_accel_and_energy(golden_case, kind):
    g = golden_case
    o = Oracle(g["mass"], g["G"], g["c"], g["eps"], kind=kind)
    acc = o.accel(g["pos"], g["vel"])
    np.testing.assert_allclose(acc, g["acc"], rtol=2e-15, atol=1e-18)
    assert o.energy(g["pos"], g["vel"]) == pytest.approx(g["energy"], rel=4e-15)
    # c = +inf is the pure Newtonian problem ("first term ... Newtonian gravity")
    oN = Oracle(g["mass"], g["G"], math.inf, g["eps"], kind=kind)
    assert oN.energy(g["pos"], g["vel"]) == pytest.approx(g["energy_newton"], rel=4e-15)
    if "acc_newton" in g:
        np.testing.assert_allclose(oN.accel(g["pos"], g["vel"]), g["acc_newton"], rtol=2e-15, atol=1e-18)


def test_schwarzschild_radius_constant():
    # M = 100 m = 0.01, c = G = 1  =>  R_Sch = 2GM/c^2 = 0.02
    G, c, M = 1.0, 1.0, 100 * 1e-4
    assert 2 * G * M / c**2 == pytest.approx(0.02)


# ------------------------------------------------------------------ Newtonian limit (textbook, numpy)
def _newton_numpy(mass, pos, G, eps):
    """Textbook softened Newtonian gravity, written independently of the oracle:
    a_a = G sum_b m_b (x_b - x_a) / d^3, d^2 = r^2 + eps^2 for star-star pairs, r^2 if a or b is body 0."""
    n = len(mass)
    d = pos[None, :, :] - pos[:, None, :]
    r2 = (d**2).sum(-1)
    soft = np.full((n, n), eps * eps)
    soft[0, :] = 0.0
    soft[:, 0] = 0.0
    r2 = r2 + soft
    np.fill_diagonal(r2, 1.0)
    w = G * mass[None, :] / r2**1.5
    np.fill_diagonal(w, 0.0)
    acc = (w[:, :, None] * d).sum(1)
    inv = 1.0 / np.sqrt(r2)
    np.fill_diagonal(inv, 0.0)
    pot = -0.5 * G * (mass[:, None] * mass[None, :] * inv).sum()
    return acc, pot


@pytest.mark.parametrize("kind", KINDS)
@pytest.mark.parametrize("eps", [0.0, 1e-3, 0.3])
def test_newtonian_limit_matches_textbook(kind, eps):
    p = inputs.plummer_bh(257, seed=11, M=0.1, softening=eps)
    o = Oracle(p.mass, p.G, math.inf, eps, kind=kind)
    accN, pot = _newton_numpy(p.mass, p.pos, p.G, eps)
    acc = o.accel(p.pos, p.vel)
    scale = np.linalg.norm(accN, axis=1, keepdims=True)
    assert np.max(np.abs(acc - accN) / scale) < 1e-12
    kin = 0.5 * (p.mass * (p.vel**2).sum(1)).sum()
    assert o.energy(p.pos, p.vel) == pytest.approx(kin + pot, rel=1e-12)


@pytest.mark.parametrize("kind", KINDS)
def test_newton_third_law_total_momentum(kind):
    # Newtonian parts only (c = inf): M a_1 + sum m_i a_i = 0.  NOT asserted for the 1PN parts (Eq. 2.8).
    p = inputs.random_small(40, seed=3, M=1.0, m_scale=0.05, softening=0.05)
    o = Oracle(p.mass, p.G, math.inf, p.softening, kind=kind)
    acc = o.accel(p.pos, p.vel)
    f = (p.mass[:, None] * acc).sum(0)
    fabs = (p.mass[:, None] * np.abs(acc)).sum(0)
    assert np.all(np.abs(f) < 1e-14 * fabs)


@pytest.mark.parametrize("kind", KINDS)
def test_softened_force_is_gradient_of_softened_potential(kind):
    # -dE/dx_i = m_i a_i at c = inf, including the eps^2 in rho_ij (Eq. 4.2) and none on BH-star.
    p = inputs.random_small(6, seed=5, M=1.0, m_scale=0.1, softening=0.4)
    o = Oracle(p.mass, p.G, math.inf, p.softening, kind=kind)
    acc = o.accel(p.pos, p.vel)
    h = 1e-5
    for a in range(p.N):
        for k in range(3):
            xp, xm = p.pos.copy(), p.pos.copy()
            xp[a, k] += h
            xm[a, k] -= h
            grad = (o.energy(xp, p.vel) - o.energy(xm, p.vel)) / (2 * h)
            assert -grad == pytest.approx(p.mass[a] * acc[a, k], rel=1e-7, abs=1e-10)


# ------------------------------------------------------------------ full EIH theory (mpmath)
def _eih_system(lam, seed=1):
    """BH (M = 1) + 3 stars of masses lam * O(1), zero-momentum frame: v_1 = -sum m v / M."""
    rng = np.random.default_rng(seed)
    x = rng.uniform(-2.0, 2.0, (3, 3))
    v = 0.3 * rng.standard_normal((3, 3))
    ms = lam * np.array([0.7, 1.0, 1.3])
    mass = np.concatenate([[1.0], ms])
    pos = np.vstack([np.zeros(3), x])
    vel = np.vstack([-(ms[:, None] * v).sum(0) / 1.0, v])
    return mass, pos, vel


def _to_list(a):
    return [[mpf(float(t)) for t in row] for row in a]


def _eih_residuals(lam, c, kind):
    mass, pos, vel = _eih_system(lam)
    o = Oracle(mass, 1.0, c, 0.0, kind=kind)
    a_hot = o.accel(pos, vel)
    a_eih = np.array([[float(t) for t in row] for row in eih.eih_acc(list(mass), _to_list(pos), _to_list(vel), 1.0, c)])
    d = np.abs(a_hot - a_eih)
    return d[0].max(), d[1:].max()


@pytest.mark.parametrize("kind", KINDS)
def test_accel_vs_full_eih_residual_scaling(kind):
    """Hot-path equations (Eqs. 2.1+2.2, 2.4+[a_i]_BH without the Cross terms) are the complete 1PN
    equations at leading order in the star mass: |a_1 - a_1^EIH| = O(lam^2 / c^2), |a_i - a_i^EIH| =
    O(lam / c^2).  The Newtonian parts carry no 1/c^2, so a wrong Newtonian term breaks the c-scaling;
    a wrong coefficient/sign/index in [a_1]_BH or [a_i]_BH breaks the lam-scaling (residual O(lam), O(1))."""
    r = {(lam, c): _eih_residuals(lam, c, kind) for lam in (1e-2, 1e-3, 1e-4) for c in (10.0, 100.0)}
    for c in (10.0, 100.0):
        # lam-scaling: a_1 residual ~ lam^2, a_i residual ~ lam
        assert r[(1e-2, c)][0] / r[(1e-3, c)][0] == pytest.approx(100.0, rel=0.1)
        assert r[(1e-3, c)][0] / r[(1e-4, c)][0] == pytest.approx(100.0, rel=0.1)
        assert r[(1e-2, c)][1] / r[(1e-3, c)][1] == pytest.approx(10.0, rel=0.1)
        assert r[(1e-3, c)][1] / r[(1e-4, c)][1] == pytest.approx(10.0, rel=0.1)
    for lam in (1e-2, 1e-3):
        # c-scaling: everything that is left is a 1PN term
        assert r[(lam, 10.0)][0] / r[(lam, 100.0)][0] == pytest.approx(100.0, rel=0.05)
        assert r[(lam, 10.0)][1] / r[(lam, 100.0)][1] == pytest.approx(100.0, rel=0.05)
    # the dropped Cross terms are small, O(0.1) coefficients: not O(1) mistakes
    assert r[(1e-3, 10.0)][0] < 0.2 * 1e-6 and r[(1e-3, 10.0)][1] < 0.5 * 1e-3


@pytest.mark.parametrize("kind", KINDS)
def test_energy_vs_full_eih_residual_scaling(kind):
    """Eq. 2.7 keeps every EIH energy term up to second order in the star masses: E - E^EIH = O(lam^3)
    (PAPER.md:94), with i = j INCLUDED in the last sum (reading R5; excluding it leaves O(lam^2))."""
    res = {}
    for lam in (1e-1, 1e-2, 1e-3):
        mass, pos, vel = _eih_system(lam, seed=2)
        E = Oracle(mass, 1.0, 10.0, 0.0, kind=kind).energy(pos, vel, terms=True)
        E_eih = eih.eih_energy(list(mass), _to_list(pos), _to_list(vel), 1.0, 10.0)
        # compare in mpmath from the oracle's separately returned terms to avoid fp64 cancellation
        t = E[1]
        E_or = sum(mpf(t[k]) for k in ("T1", "T2", "T3", "T4")) + sum(mpf(t[k]) for k in ("P1", "P2", "P3", "P4", "P5", "P6", "P7")) / 100
        res[lam] = abs(float(E_or - E_eih))
    # dropped: 3/8 M v_1^4 (O(lam^4)) and the star-star-star triple sum (O(lam^3))
    assert res[1e-1] / res[1e-2] == pytest.approx(1e3, rel=0.25)
    assert res[1e-2] / res[1e-3] > 300  # fp64 rounding of the terms (1e-16 * lam) starts to show below 1e-3
    assert res[1e-2] < 1e-2 * (1e-2) ** 3 * 100


def test_eih_reference_conserves_its_own_energy():
    """Pin of the pin: d/dt E_EIH along the EIH flow is O(c^-4) (the 1PN theory conserves its energy)."""
    rng = np.random.default_rng(7)
    m = [1.0, 0.3, 0.2, 0.1]
    x = _to_list(rng.uniform(-2, 2, (4, 3)))
    v = _to_list(0.3 * rng.standard_normal((4, 3)))
    out = []
    for c in (10.0, 100.0, 1000.0):
        a = eih.eih_acc(m, x, v, 1.0, c)
        h = mpf(10) ** -20
        xp = [[x[i][k] + h * v[i][k] for k in range(3)] for i in range(4)]
        xm = [[x[i][k] - h * v[i][k] for k in range(3)] for i in range(4)]
        vp = [[v[i][k] + h * a[i][k] for k in range(3)] for i in range(4)]
        vm = [[v[i][k] - h * a[i][k] for k in range(3)] for i in range(4)]
        dE = (eih.eih_energy(m, xp, vp, 1.0, c) - eih.eih_energy(m, xm, vm, 1.0, c)) / (2 * h)
        out.append(float(dE) * c**4)
    assert out[0] == pytest.approx(out[1], rel=0.05) and out[1] == pytest.approx(out[2], rel=0.01)


# ------------------------------------------------------------------ periastron advance (closed form)
def _kepler_ic(a, e, GM, m_ratio):
    rp = a * (1 - e)
    vp = math.sqrt(GM * (1 + e) / (a * (1 - e)))
    mass = np.array([GM, GM * m_ratio])
    pos = np.array([[0.0, 0, 0], [rp, 0, 0]])
    vel = np.array([[0.0, 0, 0], [0, vp, 0]])
    return mass, pos, vel


def _periastron_angle_after_one_orbit(o, pos, vel, period, steps_per_orbit=20000):
    dt = period / steps_per_orbit
    rv = lambda x, v: float(np.dot(x[1] - x[0], v[1] - v[0]))
    # go past apoastron, then look for the -/+ sign change of r.v (periastron)
    pos, vel = o.step(pos, vel, dt, steps_per_orbit // 2 + steps_per_orbit // 4)
    for _ in range(steps_per_orbit):
        p2, v2 = o.step(pos, vel, dt, 1)
        if rv(pos, vel) < 0 <= rv(p2, v2):
            break
        pos, vel = p2, v2
    else:
        raise AssertionError("no periastron found")
    lo, hi = 0.0, dt
    for _ in range(60):
        mid = 0.5 * (lo + hi)
        pm, vm = o.step(pos, vel, mid, 1)
        if rv(pm, vm) < 0:
            lo = mid
        else:
            hi = mid
    pm, vm = o.step(pos, vel, 0.5 * (lo + hi), 1)
    d = pm[1] - pm[0]
    return math.atan2(d[1], d[0])


@pytest.mark.parametrize("kind", KINDS)
@pytest.mark.parametrize("e,c,tol", [(0.5, 100.0, 1e-3), (0.5, 1000.0, 1e-3), (0.9, 100.0, 5e-3)])
def test_periastron_advance_test_particle(kind, e, c, tol):
    """BH + one star with m/M = 1e-9: advance per orbit = 6 pi G M / (c^2 a (1 - e^2)) (north_star)."""
    a, GM = 1.0, 1.0
    mass, pos, vel = _kepler_ic(a, e, GM, 1e-9)
    o = Oracle(mass, 1.0, c, 0.0, kind=kind)
    period = 2 * math.pi * math.sqrt(a**3 / GM)
    steps = 20000 if e < 0.8 else 80000
    dphi = _periastron_angle_after_one_orbit(o, pos, vel, period, steps)
    expected = 6 * math.pi * GM / (c * c * a * (1 - e * e))
    assert dphi == pytest.approx(expected, rel=tol)


# ------------------------------------------------------------------ integrator
@pytest.mark.parametrize("kind", KINDS)
def test_rk4_fourth_order_convergence(kind):
    """Classical RK4 (reading R13): on a Newtonian circular orbit the error after a fixed time drops by
    2^4 when dt is halved; also pins that the BH (body 0) is integrated too (finite mass ratio)."""
    M, m = 1.0, 0.25
    mu = M + m
    r = 1.0
    w = math.sqrt(mu / r**3)
    mass = np.array([M, m])
    pos = np.array([[-m / mu * r, 0, 0], [M / mu * r, 0, 0]])
    vel = np.array([[0, -m / mu * r * w, 0], [0, M / mu * r * w, 0]])
    o = Oracle(mass, 1.0, math.inf, 0.0, kind=kind)
    T = 1.0

    def err(nsteps):
        p, v = o.step(pos, vel, T / nsteps, nsteps)
        ex = np.array([[-m / mu * r * math.cos(w * T), -m / mu * r * math.sin(w * T), 0],
                       [M / mu * r * math.cos(w * T), M / mu * r * math.sin(w * T), 0]])
        return np.abs(p - ex).max()

    e1, e2, e3 = err(50), err(100), err(200)
    assert e1 / e2 == pytest.approx(16.0, rel=0.08)
    assert e2 / e3 == pytest.approx(16.0, rel=0.08)


@pytest.mark.parametrize("kind", KINDS)
def test_rk4_one_step_matches_tableau_on_linear_problem(kind):
    """With c = inf and a single far star of negligible mass the BH moves uniformly: x_1(t) = x_1 + v_1 t exactly,
    which checks that positions are advanced with the stage velocities (k_x = v) and weights sum to 1."""
    mass = np.array([1.0, 1e-30])
    pos = np.array([[0.0, 0, 0], [1e6, 0, 0]])
    vel = np.array([[0.1, -0.2, 0.3], [0, 0, 0]])
    o = Oracle(mass, 1.0, math.inf, 0.0, kind=kind)
    p, v = o.step(pos, vel, 0.5, 3)
    np.testing.assert_allclose(p[0], [0.15, -0.3, 0.45], rtol=1e-14)
    np.testing.assert_allclose(v[0], vel[0], rtol=1e-14)


# ------------------------------------------------------------------ 1PN energy conservation
@pytest.mark.parametrize("kind", KINDS)
def test_two_body_1pn_energy_conservation(kind):
    """BH + star, m/M = 1e-9, a = 1, e = 0.5: Eq. 2.7 is conserved by Eqs. 2.1-2.5 up to O(c^-4):
    the relative excursion over an orbit scales as c^-4 and shows no secular drift (reading R8).
    A wrong coefficient in P1, P2 or P3 leaves an O(c^-2) excursion instead."""
    a, e, GM = 1.0, 0.5, 1.0
    period = 2 * math.pi
    amp = {}
    for c in (100.0, 1000.0):
        mass, pos, vel = _kepler_ic(a, e, GM, 1e-9)
        o = Oracle(mass, 1.0, c, 0.0, kind=kind)
        E0 = o.energy(pos, vel)
        dev = []
        n_chunks, steps = 64, 250
        for _ in range(2 * n_chunks):  # two orbits
            pos, vel = o.step(pos, vel, period / (n_chunks * steps), steps)
            dev.append((o.energy(pos, vel) - E0) / abs(E0))
        dev = np.array(dev)
        amp[c] = np.abs(dev).max()
        # no secular drift: (nearly) back at periastron after one and two orbits (the 1PN radial period differs
        # from 2 pi by O(c^-2), hence "nearly"), and the second orbit repeats the first
        assert abs(dev[n_chunks - 1]) < 0.05 * amp[c] + 1e-13
        assert abs(dev[-1]) < 0.05 * amp[c] + 1e-13
        assert np.abs(dev[n_chunks:]).max() == pytest.approx(np.abs(dev[:n_chunks]).max(), rel=0.02, abs=1e-13)
    assert amp[100.0] == pytest.approx(2.0e-6, rel=0.2)  # SURVEY 8(c)-A8 survey-time measurement
    assert amp[100.0] / amp[1000.0] == pytest.approx(1e4, rel=0.1)


@pytest.mark.parametrize("kind", KINDS)
def test_energy_pair_form_identity(kind):
    """Eq. 2.7's star-star terms regrouped per unordered pair (the form the CUDA kernel uses):
    sum_{i<j} (G m_i m_j / rho)[-1 + (1/c^2)(w_i + w_j - 7/2 v_i.v_j - 1/2 (x_ij.v_i)(x_ij.v_j)/rho^2)],
    w_i = 3/2 v_i^2 + G M / r_1i, equals T3 + (P4 + P6)/c^2 -- written here independently in numpy."""
    p = inputs.random_small(7, seed=9, M=1.0, m_scale=0.05, c=10.0, softening=0.2, bh_moving=True)
    o = Oracle(p.mass, p.G, p.c, p.softening, kind=kind)
    _, t = o.energy(p.pos, p.vel, terms=True)
    m, x, v = p.mass[1:], p.pos[1:], p.vel[1:]
    r1 = np.linalg.norm(x - p.pos[0], axis=1)
    w = 1.5 * (v**2).sum(1) + p.G * p.mass[0] / r1
    tot = 0.0
    for i in range(len(m)):
        for j in range(i + 1, len(m)):
            d = x[i] - x[j]
            rho = math.sqrt(d @ d + p.softening**2)
            tot += p.G * m[i] * m[j] / rho * (-1 + (w[i] + w[j] - 3.5 * (v[i] @ v[j]) - 0.5 * (d @ v[i]) * (d @ v[j]) / rho**2) / p.c**2)
    assert tot == pytest.approx(t["T3"] + (t["P4"] + t["P6"]) / p.c**2, rel=1e-13)


# ------------------------------------------------------------------ API behaviour
@pytest.mark.parametrize("kind", KINDS)
def test_accel_rows_subset_equals_full(kind):
    p = inputs.plummer_bh(200, seed=4)
    o = Oracle(p.mass, p.G, p.c, p.softening, kind=kind)
    full = o.accel(p.pos, p.vel)
    rows = np.array([0, 5, 17, 200, 1])
    np.testing.assert_array_equal(o.accel_rows(p.pos, p.vel, rows), full[rows])


def test_ref_and_fast_builds_agree():
    p = inputs.plummer_bh(300, seed=8)
    a = Oracle(p.mass, p.G, p.c, p.softening, kind="ref").accel(p.pos, p.vel)
    b = Oracle(p.mass, p.G, p.c, p.softening, kind="fast").accel(p.pos, p.vel)
    assert np.max(np.abs(a - b) / np.linalg.norm(a, axis=1, keepdims=True)) < 1e-13


def test_invalid_arguments_rejected():
    with pytest.raises(ValueError):
        Oracle([1.0, -1.0], 1.0, 10.0, 0.0).accel(np.zeros((2, 3)), np.zeros((2, 3)))
    with pytest.raises(ValueError):
        Oracle([1.0, 1.0], 1.0, 10.0, -1.0).accel(np.zeros((2, 3)), np.zeros((2, 3)))
    with pytest.raises(ValueError):
        Oracle([1.0, 1.0], 1.0, 10.0, 0.0).accel(np.zeros((3, 3)), np.zeros((3, 3)))


# ------------------------------------------------------------------ NEXT rows: the Cross terms, Eqs. 2.3 and 2.6
def _eih_residuals_terms(lam, c, kind, terms):
    mass, pos, vel = _eih_system(lam)
    o = Oracle(mass, 1.0, c, 0.0, kind=kind, terms=terms)
    a = o.accel(pos, vel)
    a_eih = np.array([[float(t) for t in row] for row in eih.eih_acc(list(mass), _to_list(pos), _to_list(vel), 1.0, c)])
    d = np.abs(a - a_eih)
    return d[0].max(), d[1:].max()


@pytest.mark.parametrize("kind", KINDS)
def test_cross_terms_vs_full_eih_residual_scaling(kind):
    """With [a_i]_Cross (Eq. 2.6) the star equations agree with the full EIH theory to O(lam^2) and with [a_1]_Cross
    (Eq. 2.3) the massive object's to O(lam^3): the truncation orders the paper states.  Every term of
    Eq. 2.6 is O(lam) and every term of Eq. 2.3 O(lam^2), so a wrong coefficient, sign or index in any of them leaves a
    residual one order lower and breaks the ratios below."""
    from oracle.pn_oracle import CROSS_BH, CROSS_STAR

    c = 10.0
    lams = (1e-1, 1e-2, 1e-3)
    both = {lam: _eih_residuals_terms(lam, c, kind, CROSS_STAR | CROSS_BH) for lam in lams}
    star_only = {lam: _eih_residuals_terms(lam, c, kind, CROSS_STAR) for lam in lams}
    for hi, lo in ((1e-1, 1e-2), (1e-2, 1e-3)):
        assert both[hi][1] / both[lo][1] == pytest.approx(100.0, rel=0.15)       # a_i residual ~ lam^2
        assert both[hi][0] / both[lo][0] == pytest.approx(1000.0, rel=0.15)      # a_1 residual ~ lam^3
        assert star_only[hi][0] / star_only[lo][0] == pytest.approx(100.0, rel=0.15)  # without Eq. 2.3: still lam^2
    # the star equations do not depend on which a_1 equation is used
    assert star_only[1e-2][1] == pytest.approx(both[1e-2][1], rel=1e-9)
    # sizes seen when the reading was fixed: 0.18 lam^2 and 4.2e-4 lam^3 at c = 10
    assert both[1e-2][1] == pytest.approx(0.1767e-4, rel=0.02) and both[1e-2][0] == pytest.approx(4.232e-10, rel=0.02)
    # and both are 1PN terms: residuals scale with 1/c^2
    b100 = _eih_residuals_terms(1e-2, 100.0, kind, CROSS_STAR | CROSS_BH)
    assert both[1e-2][1] / b100[1] == pytest.approx(100.0, rel=0.05)


def test_cross_terms_vanish_in_the_newtonian_limit_and_for_massless_stars():
    from oracle.pn_oracle import CROSS_BH, CROSS_STAR

    p = inputs.random_small(12, seed=3, M=1.0, m_scale=1e-2, c=10.0, softening=1e-2, bh_moving=True)
    hot = Oracle(p.mass, p.G, math.inf, p.softening).accel(p.pos, p.vel)
    full = Oracle(p.mass, p.G, math.inf, p.softening, terms=CROSS_STAR | CROSS_BH).accel(p.pos, p.vel)
    assert np.array_equal(hot, full)  # c = inf: every Cross term carries 1/c^2
    m0 = p.mass.copy()
    m0[1:] = 0.0  # massless tracers: every Cross term carries a star mass
    hot = Oracle(m0, p.G, p.c, p.softening).accel(p.pos, p.vel)
    full = Oracle(m0, p.G, p.c, p.softening, terms=CROSS_STAR | CROSS_BH).accel(p.pos, p.vel)
    assert np.array_equal(hot, full)


def test_cross_terms_two_body_finite_mass_periastron_advance():
    """Two bodies, m/M = 0.01, zero-momentum frame, relative orbit a = 1, e = 0.5: the 1PN advance per orbit is
    6 pi G (M + m) / (c^2 a (1 - e^2)) (total mass).  The hot path misses the O(m/M) part (ratio 0.971); with the
    self terms of Eqs. 2.3 and 2.6 (first lines) the ratio is 0.999."""
    from oracle.pn_oracle import CROSS_BH, CROSS_STAR

    a, e, c, M, m = 1.0, 0.5, 100.0, 1.0, 1e-2
    mu = M + m
    rp, vp = a * (1 - e), math.sqrt(mu * (1 + e) / (a * (1 - e)))
    mass = np.array([M, m])
    pos = np.array([[-rp * m / mu, 0, 0], [rp * M / mu, 0, 0]])
    vel = np.array([[0, -vp * m / mu, 0], [0, vp * M / mu, 0]])
    period = 2 * math.pi * math.sqrt(a**3 / mu)
    expected = 6 * math.pi * mu / (c * c * a * (1 - e * e))
    got = {t: _periastron_angle_after_one_orbit(Oracle(mass, 1.0, c, 0.0, terms=t), pos, vel, period) / expected
           for t in (0, CROSS_STAR | CROSS_BH)}
    assert got[CROSS_STAR | CROSS_BH] == pytest.approx(1.0, abs=2.5e-3)
    assert got[0] == pytest.approx(0.9714, abs=2e-3)


# ------------------------------------------------------------------ NEXT-3: total 1PN momentum, Eq. 2.8 (reading R16)
@pytest.mark.parametrize("kind", KINDS)
def test_momentum_vs_full_eih_residual_scaling(kind):
    """Eq. 2.8 in the reading R16 keeps every EIH momentum term up to second order in the star masses: the residual is
    the dropped (1/2c^2) M v_1^2 v_1 = O(lam^3) (the error order the paper states).  Without the a = #1
    term or without the star-star sum the residual would be O(lam^2)."""
    res = {}
    for lam in (1e-1, 1e-2, 1e-3):
        mass, pos, vel = _eih_system(lam, seed=2)
        P_eih = np.array([float(t) for t in eih.eih_momentum(list(mass), _to_list(pos), _to_list(vel), 1.0, 10.0)])
        P = Oracle(mass, 1.0, 10.0, 0.0, kind=kind).momentum(pos, vel)
        res[lam] = np.abs(P - P_eih).max()
    assert res[1e-1] / res[1e-2] == pytest.approx(1000.0, rel=0.05)
    assert res[1e-2] / res[1e-3] == pytest.approx(1000.0, rel=0.05)
    assert res[1e-2] == pytest.approx(1.5756e-10, rel=0.01)  # 1.58e-4 lam^3 at c = 10, seen when the reading was fixed


def test_eih_reference_conserves_its_own_momentum():
    """Pin of the pin: d/dt P_EIH along the EIH flow is O(c^-4)."""
    m, x, v = _eih_system(0.3, seed=4)
    out = {}
    for c in (10.0, 100.0):
        a = np.array([[float(t) for t in r] for r in eih.eih_acc(list(m), _to_list(x), _to_list(v), 1.0, c)])
        h = 1e-6
        Pp = np.array([float(t) for t in eih.eih_momentum(list(m), _to_list(x + h * v), _to_list(v + h * a), 1.0, c)])
        Pm = np.array([float(t) for t in eih.eih_momentum(list(m), _to_list(x - h * v), _to_list(v - h * a), 1.0, c)])
        out[c] = np.abs((Pp - Pm) / (2 * h)).max()
    assert out[10.0] / out[100.0] == pytest.approx(1e4, rel=0.05)


@pytest.mark.parametrize("kind", KINDS)
def test_momentum_newtonian_limit_and_softening(kind):
    p = inputs.random_small(40, seed=21, M=1.0, m_scale=1e-2, c=10.0, softening=0.05, bh_moving=True)
    P_newton = (p.mass[:, None] * p.vel).sum(0)
    assert Oracle(p.mass, p.G, math.inf, p.softening, kind=kind).momentum(p.pos, p.vel) == pytest.approx(P_newton, rel=1e-14, abs=1e-18)
    # the 1PN part written independently in numpy (softened star-star distances, unsoftened distances to body 0)
    n = p.N
    d = p.pos[:, None, :] - p.pos[None, :, :]
    soft = np.full((n, n), p.softening**2)
    soft[0, :] = soft[:, 0] = 0.0
    r = np.sqrt((d**2).sum(-1) + soft)
    np.fill_diagonal(r, np.inf)
    nv = (d * p.vel[:, None, :]).sum(-1) / r  # (v_a . n_ab)
    pair = (p.G * p.mass[:, None] * p.mass[None, :] / r)[:, :, None] * (p.vel[:, None, :] + (nv / r)[:, :, None] * d)
    v2 = (p.vel**2).sum(1)
    v2[0] = 0.0  # the (1/2c^2) M v_1^2 v_1 term is dropped (O(m^3))
    P = P_newton + (p.mass * v2 / (2 * p.c**2))[:, None].__mul__(p.vel).sum(0) - pair.sum((0, 1)) / (2 * p.c**2)
    assert Oracle(p.mass, p.G, p.c, p.softening, kind=kind).momentum(p.pos, p.vel) == pytest.approx(P, rel=1e-12, abs=1e-16)


def test_cross_terms_two_body_finite_mass_energy_conservation():
    """Two bodies, m/M = 0.01 and 0.03, e = 0.5, c = 100: along the flow with both Cross rows the energy of Eq. 2.7 only
    shows the c^-4 excursion of the test-particle case (2.0e-6, independent of the mass ratio); along the hot path alone
    it moves by O(m/M) of that scale (2.9e-5, 9.1e-5).  Pins the self lines of Eqs. 2.3 and 2.6 against Eq. 2.7."""
    from oracle.pn_oracle import CROSS_BH, CROSS_STAR

    a, e, c, M = 1.0, 0.5, 100.0, 1.0
    out = {}
    for m in (1e-2, 3e-2):
        mu = M + m
        rp, vp = a * (1 - e), math.sqrt(mu * (1 + e) / (a * (1 - e)))
        mass = np.array([M, m])
        pos = np.array([[-rp * m / mu, 0, 0], [rp * M / mu, 0, 0]])
        vel = np.array([[0, -vp * m / mu, 0], [0, vp * M / mu, 0]])
        dt = 2 * math.pi / math.sqrt(mu) / 2000
        for terms in (0, CROSS_STAR | CROSS_BH):
            o = Oracle(mass, 1.0, c, 0.0, terms=terms)
            e0, x, v, worst = o.energy(pos, vel), pos, vel, 0.0
            for _ in range(40):
                x, v = o.step(x, v, dt, 50)
                worst = max(worst, abs(o.energy(x, v) - e0) / abs(e0))
            out[(m, terms)] = worst
    for m in (1e-2, 3e-2):
        assert out[(m, 3)] == pytest.approx(2.0e-6, rel=0.25)
        assert out[(m, 0)] > 10 * out[(m, 3)]
    assert out[(3e-2, 0)] / out[(1e-2, 0)] == pytest.approx(3.0, rel=0.15)


def test_cross_terms_hand_values_two_bodies():
    """By hand, G = 1, c = 10, M = 1 at the origin at rest, one star m = 1e-3 at x = (1, 0, 0) with v = (0, 1, 0)
    (the first golden case, whose hot-path values are a_star = (-0.97, 0, 0), a_1 = (9.7e-4, 0, 0)).
    Eq. 2.6 with one star is its first line only: 5 G^2 m M x_i1 / r^4 - (G m / r^3)[4 v^2 x_i1 - 7 (v.x_i1) v]
      = 5e-3 (1,0,0) - 1e-3 [4 (1,0,0) - 0] = (1e-3, 0, 0);  a_star += 1e-3 / c^2 = 1e-5.
    Eq. 2.3 with one star: 4 G^2 m^2 x_1j / r^4 = 4e-6 (-1,0,0); the (j,k) sums with r_jk are empty; the velocity sum has
    the single term k = j: -(G m^2 / (M r^3)) [4 v^2 x_1j - 3 (v.x_1j) v - 4 (v.x_1j) v] = -1e-6 [4 (-1,0,0)] = (4e-6,0,0):
    the two cancel, a_1 is unchanged."""
    from oracle.pn_oracle import CROSS_BH, CROSS_STAR

    mass = np.array([1.0, 1e-3])
    pos = np.array([[0.0, 0, 0], [1.0, 0, 0]])
    vel = np.array([[0.0, 0, 0], [0.0, 1.0, 0]])
    a = Oracle(mass, 1.0, 10.0, 0.0, terms=CROSS_STAR | CROSS_BH).accel(pos, vel)
    np.testing.assert_allclose(a[1], [-0.97 + 1e-5, 0.0, 0.0], rtol=1e-15, atol=1e-18)
    np.testing.assert_allclose(a[0], [9.7e-4, 0.0, 0.0], rtol=1e-13, atol=1e-18)
    # second star velocity along x: v = (0.5, 0, 0): L0 = 5e-3 (1,0,0) - 1e-3 [4 * 0.25 (1,0,0) - 7 * 0.5 * (0.5,0,0)]
    #   = (5e-3 - 1e-3 + 1.75e-3, 0, 0) = (5.75e-3, 0, 0)
    vel[1] = [0.5, 0.0, 0.0]
    hot = Oracle(mass, 1.0, 10.0, 0.0).accel(pos, vel)
    a = Oracle(mass, 1.0, 10.0, 0.0, terms=CROSS_STAR).accel(pos, vel)
    np.testing.assert_allclose(a[1] - hot[1], [5.75e-5, 0.0, 0.0], rtol=1e-12, atol=1e-18)


def test_cross_terms_and_momentum_hand_values_softened_345():
    """The eps > 0 branch of Eqs. 2.6, 2.3 and 2.8 (reading R9: every star-star distance softened, the r_ij^2 numerators and
    n_ij included): tests/golden/n3_345_softened_cross.txt, worked by hand in exact fractions (rho_AB = 6).  One unsoftened
    occurrence of r_ij in cross_star, cross_bh or oracle_momentum moves a value here by 1e-3 ... 1e-1 of itself."""
    from oracle.pn_oracle import CROSS_BH, CROSS_STAR
    from tests.conftest import load_golden, rel_err_rows

    g = load_golden("n3_345_softened_cross.txt")
    args = (g["mass"], g["G"], g["c"], g["eps"])
    hot = Oracle(*args).accel(g["pos"], g["vel"])
    star = Oracle(*args, terms=CROSS_STAR).accel(g["pos"], g["vel"])
    full = Oracle(*args, terms=CROSS_STAR | CROSS_BH).accel(g["pos"], g["vel"])
    assert rel_err_rows(star, g["acc_cross_star"]).max() <= 1e-14
    assert rel_err_rows(full, g["acc_cross_full"]).max() <= 1e-14
    # the Cross terms by themselves (1e-2 ... 1e-4 of the acceleration): difference to the hot path, times c^2
    c2 = g["c"] ** 2
    np.testing.assert_allclose((star[1:] - hot[1:]) * c2, g["cross_star"], rtol=0, atol=1e-12 * np.abs(g["cross_star"]).max())
    np.testing.assert_allclose((full[0] - hot[0]) * c2, g["cross_bh"], rtol=0, atol=1e-11 * np.abs(g["cross_bh"]).max())
    np.testing.assert_array_equal(star[0], hot[0])
    P = Oracle(*args).momentum(g["pos"], g["vel"])
    np.testing.assert_allclose(P, g["momentum"], rtol=1e-14, atol=0)
    # and the softening matters at the level the pin resolves: eps = 0 changes every one of these values
    full0 = Oracle(g["mass"], g["G"], g["c"], 0.0, terms=CROSS_STAR | CROSS_BH).accel(g["pos"], g["vel"])
    hot0 = Oracle(g["mass"], g["G"], g["c"], 0.0).accel(g["pos"], g["vel"])
    assert np.abs((full0 - hot0) - (full - hot)).max() * c2 > 1e-2 * np.abs(g["cross_star"]).max()
    assert np.abs(Oracle(g["mass"], g["G"], g["c"], 0.0).momentum(g["pos"], g["vel"]) - P).max() > 1e-9


# ------------------------------------------------------------------ symmetries every term must respect
def _rotation(seed):
    rng = np.random.default_rng(seed)
    q, r = np.linalg.qr(rng.standard_normal((3, 3)))
    q *= np.sign(np.diag(r))
    if np.linalg.det(q) < 0:
        q[:, 0] = -q[:, 0]
    return q


@pytest.mark.parametrize("terms", [0, 1, 3])
def test_rotation_covariance_translation_invariance_and_velocity_parity(terms):
    """a(R x + t, R v) = R a(x, v) for a proper rotation R and a shift t; E is invariant, P rotates; every velocity term of
    the limited equations is even in the velocities, so a(x, -v) = a(x, v), E(x, -v) = E(x, v), P(x, -v) = -P(x, v).
    A transposed component, a stray index or an odd velocity power in any line breaks one of these."""
    p = inputs.random_small(9, seed=77, M=1.0, m_scale=2e-2, c=5.0, softening=0.03, bh_moving=True)
    R, t = _rotation(5), np.array([0.3, -1.1, 0.7])
    o = Oracle(p.mass, p.G, p.c, p.softening, terms=terms)
    a = o.accel(p.pos, p.vel)
    xr, vr = p.pos @ R.T + t, p.vel @ R.T
    np.testing.assert_allclose(o.accel(xr, vr), a @ R.T, rtol=0, atol=2e-13 * np.abs(a).max())
    assert o.energy(xr, vr) == pytest.approx(o.energy(p.pos, p.vel), rel=1e-13)
    np.testing.assert_allclose(o.momentum(xr, vr), R @ o.momentum(p.pos, p.vel), rtol=0, atol=1e-15)
    np.testing.assert_allclose(o.accel(p.pos, -p.vel), a, rtol=0, atol=1e-15 * np.abs(a).max())
    assert o.energy(p.pos, -p.vel) == pytest.approx(o.energy(p.pos, p.vel), rel=1e-15)
    np.testing.assert_allclose(o.momentum(p.pos, -p.vel), -o.momentum(p.pos, p.vel), rtol=0, atol=1e-18)
    # the 1PN terms are really exercised: they change the accelerations at the percent level here
    aN = Oracle(p.mass, p.G, math.inf, p.softening).accel(p.pos, p.vel)
    assert np.abs(a - aN).max() > 1e-3 * np.abs(a).max()
