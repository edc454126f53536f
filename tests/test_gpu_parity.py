"""GPU parity: the CUDA path (through the C-ABI, via the thin binding) against the CPU oracle,
element by element on the same seeded inputs.  Tolerances (north_star, R10):
  accelerations  err_i = max_k |a_ik - ref_ik| / ||ref_i||_2 <= 1e-12   (fp64 path)
  trajectories   same measure on positions / velocities after n RK4 steps
  energy drift   |delta_gpu(t) - delta_oracle(t)| <= 1e-10, delta = (E(t) - E(0)) / |E(0)|
"""
import math

import numpy as np
import pytest

from oracle.pn_oracle import Oracle
from paper_1801_07986_b200 import inputs
from tests.conftest import load_golden, rel_err_rows, GOLDEN_CASES

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL_ACC = 1e-12
TOL_DRIFT = 1e-10


def _pn(p, **kw):
    from paper_1801_07986_b200 import PN

    return PN(p.mass, p.G, p.c, p.softening, **kw)


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _gpu_accel(pn, pos, vel):
    return pn.pn_accel(_dev(pos), _dev(vel)).cpu().numpy()


# ------------------------------------------------------------------ hand values straight through the C-ABI
@pytest.mark.parametrize("case", GOLDEN_CASES)
def test_golden_values_on_gpu(case):
    from paper_1801_07986_b200 import PN

    g = load_golden(case)
    with PN(g["mass"], g["G"], g["c"], g["eps"]) as pn:
        acc = _gpu_accel(pn, g["pos"], g["vel"])
        np.testing.assert_allclose(acc, g["acc"], rtol=1e-14, atol=1e-17)
        pn.pn_set_state(_dev(g["pos"]), _dev(g["vel"]))
        assert pn.pn_energy() == pytest.approx(g["energy"], rel=1e-14)
    with PN(g["mass"], g["G"], math.inf, g["eps"]) as pn:
        pn.pn_set_state(_dev(g["pos"]), _dev(g["vel"]))
        assert pn.pn_energy() == pytest.approx(g["energy_newton"], rel=1e-14)


# ------------------------------------------------------------------ accelerations, several tiles + ragged tails
@pytest.mark.parametrize("n_stars", [1, 2, 31, 127, 128, 129, 1023, 3071, 3072, 4099, 12288, 13001])
def test_accel_parity_sizes(n_stars):
    if n_stars <= 2:  # one recentred star sits on the BH, two equal ones cancel a_1 exactly: unequal masses, BH displaced
        p = inputs.random_small(n_stars, seed=101, M=1.0, m_scale=1e-2, c=10.0, softening=1e-3, bh_moving=True)
    else:
        p = inputs.plummer_bh(n_stars, seed=100 + n_stars)
    ref = Oracle(p.mass, p.G, p.c, p.softening).accel(p.pos, p.vel)
    assert np.isfinite(ref).all()
    with _pn(p) as pn:
        acc = _gpu_accel(pn, p.pos, p.vel)
    assert rel_err_rows(acc, ref).max() <= TOL_ACC


@pytest.mark.parametrize("gen", ["cusp", "ball", "random"])
def test_accel_parity_other_distributions(gen):
    if gen == "cusp":
        p = inputs.cusp_bh(5000, seed=2)
    elif gen == "ball":
        p = inputs.uniform_ball_bh(12)
    else:
        p = inputs.random_small(700, seed=5, M=1.0, m_scale=1e-3, c=10.0, softening=0.01, bh_moving=True)
    ref = Oracle(p.mass, p.G, p.c, p.softening).accel(p.pos, p.vel)
    with _pn(p) as pn:
        acc = _gpu_accel(pn, p.pos, p.vel)
    assert rel_err_rows(acc, ref).max() <= TOL_ACC


# both fp64 star-star kernels at every size class: the tiled one (ordered pairs) and the symmetric one (unordered
# pairs applied to both stars) in the forms choose_sym (pn_api.cu) picks by size: the j-split form on 128-star unit tiles
# (below 16000 stars and from 16385 to 35999), one-warp blocks on 128-star tiles (16000 ... 16384), 512-star tiles from
# 36000 stars on (test_gpu_fullsize.py covers those), with one group per tile (m = 1) and several (20000 -> T = 157,
# m = 2, ragged last group)
# "symmetric" on equal-mass stars takes the equal-mass form (variant 4: rho^-3 d accumulated, G m applied at the flush);
# "symmetric_general" switches that off (variant 2), which is also what unequal masses get.
@pytest.mark.parametrize("kernel", ["tiled", "symmetric", "symmetric_general"])
@pytest.mark.parametrize("n_stars", [1, 2, 65, 129, 1023, 3071, 4099, 9000, 13001, 20000])
def test_accel_parity_both_pair_kernels(n_stars, kernel):
    from paper_1801_07986_b200 import binding

    if n_stars <= 2:
        p = inputs.random_small(n_stars, seed=111, M=1.0, m_scale=1e-2, c=10.0, softening=1e-3, bh_moving=True)
    else:
        p = inputs.plummer_bh(n_stars, seed=300 + n_stars)
    ref = Oracle(p.mass, p.G, p.c, p.softening).accel(p.pos, p.vel)
    with _pn(p) as pn:
        pn.pn_set_option(binding.PN_OPT_PAIR_KERNEL, binding.PN_PAIR_TILED if kernel == "tiled" else binding.PN_PAIR_SYMMETRIC)
        if kernel == "symmetric_general":
            pn.pn_set_option(binding.PN_OPT_EQUAL_MASS, 0)
        equal = n_stars != 2  # plummer_bh: equal masses (one star trivially so); random_small(2): unequal
        want = 0 if kernel == "tiled" else (4 if (kernel == "symmetric" and equal) else 2)
        assert pn.pn_get_pair_config()["variant"] == want
        acc = _gpu_accel(pn, p.pos, p.vel)
        again = _gpu_accel(pn, p.pos, p.vel)
    assert rel_err_rows(acc, ref).max() <= TOL_ACC
    assert np.array_equal(acc, again)  # fixed-order partial sums: bit-reproducible


def test_pair_kernels_agree_and_auto_selection():
    from paper_1801_07986_b200 import binding

    for n_stars, want in ((3071, 7), (3072, 4)):  # 7: the one-launch small-system path (N_s < 3072)
        p = inputs.plummer_bh(n_stars, seed=12)
        with _pn(p) as pn:
            assert pn.pn_get_pair_config()["variant"] == want
            acc = {binding.PN_PAIR_AUTO: _gpu_accel(pn, p.pos, p.vel)}
            for k in (binding.PN_PAIR_TILED, binding.PN_PAIR_SYMMETRIC):
                pn.pn_set_option(binding.PN_OPT_PAIR_KERNEL, k)
                assert pn.pn_get_pair_config()["variant"] == (0 if k == binding.PN_PAIR_TILED else 4)
                acc[k] = _gpu_accel(pn, p.pos, p.vel)
            assert rel_err_rows(acc[binding.PN_PAIR_SYMMETRIC], acc[binding.PN_PAIR_TILED]).max() <= 1e-13
            assert rel_err_rows(acc[binding.PN_PAIR_AUTO], acc[binding.PN_PAIR_TILED]).max() <= 1e-13
            with pytest.raises(binding.PNError):
                pn.pn_set_option(binding.PN_OPT_PAIR_KERNEL, 7)


@pytest.mark.parametrize("kernel", ["tiled", "symmetric"])
@pytest.mark.parametrize("n_stars", [300, 4099])
def test_accel_zero_softening_masks_self_pair(n_stars, kernel):
    from paper_1801_07986_b200 import binding

    p = inputs.random_small(n_stars, seed=6, M=1.0, m_scale=1e-3, c=20.0, softening=0.0)
    ref = Oracle(p.mass, p.G, p.c, 0.0).accel(p.pos, p.vel)
    with _pn(p) as pn:
        pn.pn_set_option(binding.PN_OPT_PAIR_KERNEL, binding.PN_PAIR_TILED if kernel == "tiled" else binding.PN_PAIR_SYMMETRIC)
        acc = _gpu_accel(pn, p.pos, p.vel)
    assert np.isfinite(acc).all()
    assert rel_err_rows(acc, ref).max() <= TOL_ACC


def test_accel_zero_softening_equal_mass_form():
    """eps = 0 on equal-mass stars: the self-pair mask inside the equal-mass form of the symmetric kernel."""
    from paper_1801_07986_b200 import binding

    p = inputs.plummer_bh(4099, seed=61, softening=0.0)
    ref = Oracle(p.mass, p.G, p.c, 0.0).accel(p.pos, p.vel)
    with _pn(p) as pn:
        assert pn.pn_get_pair_config()["variant"] == 4
        acc = _gpu_accel(pn, p.pos, p.vel)
    assert np.isfinite(acc).all()
    assert rel_err_rows(acc, ref).max() <= TOL_ACC


def test_accel_newtonian_limit_and_zero_mass_stars():
    p = inputs.plummer_bh(500, seed=7)
    p.mass[5:50] = 0.0  # massless tracers: feel forces, exert none
    ref = Oracle(p.mass, p.G, math.inf, p.softening).accel(p.pos, p.vel)
    from paper_1801_07986_b200 import PN

    with PN(p.mass, p.G, math.inf, p.softening) as pn:
        acc = _gpu_accel(pn, p.pos, p.vel)
    assert rel_err_rows(acc, ref).max() <= TOL_ACC


def test_accel_is_deterministic_and_independent_of_j_split():
    from paper_1801_07986_b200 import binding

    p = inputs.plummer_bh(4099, seed=8)
    ref = Oracle(p.mass, p.G, p.c, p.softening).accel(p.pos, p.vel)
    with _pn(p) as pn:
        a1 = _gpu_accel(pn, p.pos, p.vel)
        a2 = _gpu_accel(pn, p.pos, p.vel)
        assert np.array_equal(a1, a2)  # fixed-order reductions: bit-reproducible
        pn.pn_set_option(binding.PN_OPT_PAIR_KERNEL, binding.PN_PAIR_TILED)  # the j-split belongs to the tiled kernel
        for s in (1, 3, 64):
            pn.pn_set_option(binding.PN_OPT_J_SPLIT, s)
            assert rel_err_rows(_gpu_accel(pn, p.pos, p.vel), ref).max() <= TOL_ACC


def test_accel_host_entry_point_matches_device_entry_point():
    p = inputs.plummer_bh(2000, seed=9)
    with _pn(p) as pn:
        a_dev = _gpu_accel(pn, p.pos, p.vel)
        a_host = pn.pn_accel_host(p.pos, p.vel)
    assert np.array_equal(a_dev, a_host)


def test_accel_does_not_disturb_integrator_state():
    p = inputs.plummer_bh(600, seed=10)
    q = inputs.plummer_bh(600, seed=11)
    with _pn(p) as pn:
        pn.pn_set_state(_dev(p.pos), _dev(p.vel))
        e0 = pn.pn_energy()
        _gpu_accel(pn, q.pos, q.vel)
        assert pn.pn_energy() == e0
        x, v = pn.pn_get_state()
        assert np.array_equal(x.cpu().numpy(), p.pos) and np.array_equal(v.cpu().numpy(), p.vel)


# ------------------------------------------------------------------ energy
@pytest.mark.parametrize("n_stars,eps", [(1, 0.0), (2, 0.0), (129, 1e-3), (1023, 1e-3), (4099, 0.0)])
def test_energy_parity(n_stars, eps):
    p = inputs.random_small(n_stars, seed=20 + n_stars, M=1.0, m_scale=1.0 / n_stars, c=10.0, softening=eps, bh_moving=True)
    ref = Oracle(p.mass, p.G, p.c, eps).energy(p.pos, p.vel)
    with _pn(p) as pn:
        pn.pn_set_state(_dev(p.pos), _dev(p.vel))
        e = pn.pn_energy()
    assert e == pytest.approx(ref, rel=1e-13)


# ------------------------------------------------------------------ config 1: 100 RK4 steps, every step checked
def test_config1_trajectory_accel_and_energy_drift():
    p = inputs.config(1)
    o = Oracle(p.mass, p.G, p.c, p.softening)
    with _pn(p) as pn:
        pn.pn_set_state(_dev(p.pos), _dev(p.vel))
        e0_gpu = pn.pn_energy()
        e0_ref = o.energy(p.pos, p.vel)
        assert e0_gpu == pytest.approx(e0_ref, rel=1e-13)
        xr, vr = p.pos, p.vel
        worst_acc = worst_traj = worst_drift = 0.0
        for step in range(p.nsteps):
            pn.pn_step(p.dt, 1)
            xr, vr = o.step(xr, vr, p.dt, 1)
            xg, vg = pn.pn_get_state()
            xg, vg = xg.cpu().numpy(), vg.cpu().numpy()
            # trajectory: GPU state vs oracle trajectory
            worst_traj = max(worst_traj, rel_err_rows(xg, xr).max(), rel_err_rows(vg, vr).max())
            # accelerations at the SAME (GPU) state
            acc = pn.pn_accel(_dev(xg), _dev(vg)).cpu().numpy()
            worst_acc = max(worst_acc, rel_err_rows(acc, o.accel(xg, vg)).max())
            # energy drift
            d_gpu = (pn.pn_energy() - e0_gpu) / abs(e0_gpu)
            d_ref = (o.energy(xr, vr) - e0_ref) / abs(e0_ref)
            worst_drift = max(worst_drift, abs(d_gpu - d_ref))
        assert worst_acc <= TOL_ACC
        assert worst_traj <= 1e-11
        assert worst_drift <= TOL_DRIFT


def test_config3_like_cusp_trajectory_and_energy_drift():
    """Config 3's recipe (Bahcall-Wolf cusp, mass ratio 1e4, c = 316, eps = 1e-4, dt = 1e-5, 20 steps) at a size the
    oracle integrates in seconds: trajectory and drift parity where the dynamics is stiff (inner orbital period 2e-4, so
    the energy drifts by percents within 20 steps: the drift must be the oracle's, not merely small)."""
    p = inputs.cusp_bh(4095, seed=2)
    o = Oracle(p.mass, p.G, p.c, p.softening)
    with _pn(p) as pn:
        pn.pn_set_state(_dev(p.pos), _dev(p.vel))
        e0_gpu, e0_ref = pn.pn_energy(), o.energy(p.pos, p.vel)
        assert e0_gpu == pytest.approx(e0_ref, rel=1e-13)
        xr, vr = p.pos, p.vel
        worst_traj = worst_drift = 0.0
        drift_ref = 0.0
        for _ in range(4):
            pn.pn_step(p.dt, 5)
            xr, vr = o.step(xr, vr, p.dt, 5)
            xg, vg = pn.pn_get_state()
            worst_traj = max(worst_traj, rel_err_rows(xg.cpu().numpy(), xr).max(), rel_err_rows(vg.cpu().numpy(), vr).max())
            d_gpu = (pn.pn_energy() - e0_gpu) / abs(e0_gpu)
            drift_ref = (o.energy(xr, vr) - e0_ref) / abs(e0_ref)
            worst_drift = max(worst_drift, abs(d_gpu - drift_ref))
    assert worst_traj <= 1e-10
    assert worst_drift <= TOL_DRIFT
    print(f"cusp 4095: oracle drift after 20 steps {drift_ref:.3e}, worst trajectory error {worst_traj:.2e}")


@pytest.mark.parametrize("kernel", ["auto", "tiled"])
def test_step_graph_and_plain_launches_agree_bitwise(kernel):
    """auto: N_s = 2500 takes the small-system path (one cooperative launch, PN_OPT_USE_GRAPH does not apply);
    tiled: the multi-kernel path, as a 16-step batched graph + 3 single-step graphs against plain launches."""
    from paper_1801_07986_b200 import binding

    p = inputs.plummer_bh(2500, seed=12, dt=1e-3)
    out = []
    for use_graph in (1, 0):
        with _pn(p) as pn:
            if kernel == "tiled":
                pn.pn_set_option(binding.PN_OPT_PAIR_KERNEL, binding.PN_PAIR_TILED)
            pn.pn_set_option(binding.PN_OPT_USE_GRAPH, use_graph)
            pn.pn_set_state(_dev(p.pos), _dev(p.vel))
            pn.pn_step(p.dt, 19)  # 16-step batched graph + 3 single-step graphs
            x, v = pn.pn_get_state_host()
            out.append((x, v))
    assert np.array_equal(out[0][0], out[1][0]) and np.array_equal(out[0][1], out[1][1])
    xr, vr = Oracle(p.mass, p.G, p.c, p.softening).step(p.pos, p.vel, p.dt, 19)
    assert rel_err_rows(out[0][0], xr).max() <= 1e-11 and rel_err_rows(out[0][1], vr).max() <= 1e-11


def test_timed_graph_path_matches_and_counts_pair_launches():
    """PN_OPT_TIME_PAIR keeps pn_step on a CUDA graph (event-record nodes around each pair stage): same state bitwise,
    4 timed launches per step, with graphs and with plain launches."""
    from paper_1801_07986_b200 import binding

    p = inputs.plummer_bh(4099, seed=23)
    ref = None
    for time_pair, use_graph in ((0, 1), (1, 1), (1, 0), (2, 1), (2, 0)):
        with _pn(p) as pn:
            pn.pn_set_option(binding.PN_OPT_USE_GRAPH, use_graph)
            pn.pn_set_option(binding.PN_OPT_TIME_PAIR, time_pair)
            pn.pn_set_state_host(p.pos, p.vel)
            pn.pn_step(p.dt, 3)
            pn.pn_step(p.dt, 2)
            x, v = pn.pn_get_state_host()
            ms, n = pn.pn_get_pair_time()
        if ref is None:
            ref = (x, v)
            assert n == 0
        else:
            assert np.array_equal(x, ref[0]) and np.array_equal(v, ref[1])
            assert n == (20 if time_pair == 1 else 5) and 0.0 < ms < 50.0


def test_step_changes_of_dt_are_honoured():
    p = inputs.plummer_bh(300, seed=13)
    o = Oracle(p.mass, p.G, p.c, p.softening)
    with _pn(p) as pn:
        pn.pn_set_state_host(p.pos, p.vel)
        pn.pn_step(1e-3, 2)
        pn.pn_step(5e-4, 3)
        x, v = pn.pn_get_state_host()
    xr, vr = o.step(p.pos, p.vel, 1e-3, 2)
    xr, vr = o.step(xr, vr, 5e-4, 3)
    assert rel_err_rows(x, xr).max() <= 1e-12 and rel_err_rows(v, vr).max() <= 1e-12


def test_two_body_periastron_orbit_on_gpu_tracks_oracle():
    """Degenerate smallest system N = 2 (one star): the whole path with a single live thread."""
    mass = np.array([1.0, 1e-9])
    pos = np.array([[0.0, 0, 0], [0.5, 0, 0]])
    vel = np.array([[0.0, 0, 0], [0, math.sqrt(3.0), 0]])
    from paper_1801_07986_b200 import PN

    with PN(mass, 1.0, 100.0, 0.0) as pn:
        pn.pn_set_state_host(pos, vel)
        pn.pn_step(2 * math.pi / 4000, 4000)
        x, v = pn.pn_get_state_host()
    xr, vr = Oracle(mass, 1.0, 100.0, 0.0).step(pos, vel, 2 * math.pi / 4000, 4000)
    assert np.abs(x - xr).max() < 1e-10 and np.abs(v - vr).max() < 1e-10


# ------------------------------------------------------------------ errors
def test_state_errors_and_bad_arguments():
    from paper_1801_07986_b200 import binding

    p = inputs.plummer_bh(100, seed=14)
    with _pn(p) as pn:
        with pytest.raises(binding.PNError) as ei:
            pn.pn_step(1e-3, 1)
        assert ei.value.code == binding.PN_ESTATE
        with pytest.raises(binding.PNError):
            pn.pn_energy()
        pn.pn_set_state_host(p.pos, p.vel)
        with pytest.raises(binding.PNError) as ei:
            pn.pn_step(float("nan"), 1)
        assert ei.value.code == binding.PN_EINVAL
        with pytest.raises(binding.PNError):
            pn.pn_step(1e-3, -1)
        with pytest.raises(binding.PNError):
            pn.pn_set_option(99, 0)
        with pytest.raises(TypeError):
            pn.pn_accel(torch.zeros(5, 3, dtype=torch.float64, device="cuda"), _dev(p.vel))

