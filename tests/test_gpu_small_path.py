"""The small-system path (N_s < 3072): one cooperative launch runs a whole pn_step call (every stage of every RK4 step)
or one pn_accel -- pair sums, BH <-> star 1PN terms, the a_1 reduction and the fused RK4 update in small_path_kernel, with one
grid-wide barrier per force evaluation.  Parity against the oracle at every i-stars-per-warp class (IW = 1 ... 6), ragged
sizes, eps = 0, unequal masses and massless tracers; trajectories, bit-reproducibility, agreement with the multi-kernel path.
"""
import numpy as np
import pytest

from oracle.pn_oracle import Oracle
from paper_1801_07986_b200 import inputs
from tests.conftest import rel_err_rows

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL_ACC = 1e-12


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


# IW = ceil(N_s / warps of the grid), 4 warps per SM; the sizes below are the class boundaries on a 148-SM B200 (592 warps)
@pytest.mark.parametrize("n_stars", [2, 3, 31, 33, 255, 592, 593, 1023, 1184, 1185, 1777, 2368, 2369, 2961, 3071])
def test_small_path_accel_parity(n_stars):
    from paper_1801_07986_b200 import PN

    p = inputs.random_small(n_stars, seed=n_stars, M=1.0, m_scale=1e-3, c=20.0, softening=1e-3)  # unequal masses
    if n_stars > 40:
        p.mass[5:40:7] = 0.0  # massless tracers
    ref = Oracle(p.mass, p.G, p.c, p.softening).accel(p.pos, p.vel)
    with PN(p.mass, p.G, p.c, p.softening) as pn:
        cfg = pn.pn_get_pair_config()
        warps = 4 * torch.cuda.get_device_properties(0).multi_processor_count
        assert cfg["variant"] == 7 and cfg["i_per_thread"] == -(-n_stars // warps)
        acc = pn.pn_accel(_dev(p.pos), _dev(p.vel)).cpu().numpy()
        again = pn.pn_accel(_dev(p.pos), _dev(p.vel)).cpu().numpy()
    assert np.isfinite(acc).all()
    assert rel_err_rows(acc, ref).max() <= TOL_ACC
    assert np.array_equal(acc, again)


@pytest.mark.parametrize("n_stars", [300, 1500])
def test_small_path_zero_softening(n_stars):
    from paper_1801_07986_b200 import PN

    p = inputs.random_small(n_stars, seed=6, M=1.0, m_scale=1e-3, c=20.0, softening=0.0)
    ref = Oracle(p.mass, p.G, p.c, p.softening).accel(p.pos, p.vel)
    with PN(p.mass, p.G, p.c, p.softening) as pn:
        acc = pn.pn_accel(_dev(p.pos), _dev(p.vel)).cpu().numpy()
    assert np.isfinite(acc).all()
    assert rel_err_rows(acc, ref).max() <= TOL_ACC


@pytest.mark.parametrize("n_stars,nsteps", [(3, 50), (100, 40), (1023, 24), (2047, 8)])
def test_small_path_trajectory_split_calls_and_other_path(n_stars, nsteps):
    """nsteps in one launch == the same steps in several launches (bitwise); both track the oracle; the multi-kernel path
    (PN_PAIR_TILED) lands on the same trajectory to rounding; pn_energy / pn_get_state see the state the launch left."""
    from paper_1801_07986_b200 import PN, binding

    p = inputs.plummer_bh(n_stars, seed=3, dt=1e-3)
    o = Oracle(p.mass, p.G, p.c, p.softening)
    xr, vr = o.step(p.pos, p.vel, p.dt, nsteps)
    with PN(p.mass, p.G, p.c, p.softening) as pn:
        pn.pn_set_state_host(p.pos, p.vel)
        pn.pn_step(p.dt, nsteps)
        x1, v1 = pn.pn_get_state_host()
        e1 = pn.pn_energy()
        assert pn.pn_get_launch_count() <= 8  # set_state, one launch for all steps, get_state, 3 energy kernels
        pn.pn_set_state_host(p.pos, p.vel)
        for chunk in (1, nsteps // 2, nsteps - 1 - nsteps // 2):
            pn.pn_step(p.dt, chunk)
        x2, v2 = pn.pn_get_state_host()
        pn.pn_set_option(binding.PN_OPT_PAIR_KERNEL, binding.PN_PAIR_TILED)
        pn.pn_set_state_host(p.pos, p.vel)
        pn.pn_step(p.dt, nsteps)
        x3, v3 = pn.pn_get_state_host()
    assert np.array_equal(x1, x2) and np.array_equal(v1, v2)
    assert rel_err_rows(x1, xr).max() <= 1e-11 and rel_err_rows(v1, vr).max() <= 1e-11
    assert rel_err_rows(x3, x1).max() <= 1e-12 and rel_err_rows(v3, v1).max() <= 1e-12
    assert e1 == pytest.approx(o.energy(xr, vr), rel=1e-11)


def test_small_path_accel_between_steps_does_not_disturb_the_state():
    """pn_accel uses the second stage set, which the small-system pn_step also uses as its second position buffer."""
    from paper_1801_07986_b200 import PN

    p = inputs.plummer_bh(700, seed=4, dt=1e-3)
    q = inputs.random_small(700, seed=9, M=0.1, m_scale=1.0 / 700, c=100.0, softening=1e-3)
    with PN(p.mass, p.G, p.c, p.softening) as pn:
        pn.pn_set_state_host(p.pos, p.vel)
        pn.pn_step(p.dt, 6)
        ref = pn.pn_get_state_host()
        pn.pn_set_state_host(p.pos, p.vel)
        pn.pn_step(p.dt, 3)
        pn.pn_accel(_dev(q.pos), _dev(q.vel))
        pn.pn_step(p.dt, 3)
        got = pn.pn_get_state_host()
    assert np.array_equal(ref[0], got[0]) and np.array_equal(ref[1], got[1])


def test_two_small_contexts_on_two_streams():
    """Cooperative launches of two contexts never share the device half and half (each spins at its own grid barrier):
    the library chains them; interleaved stepping on two streams gives each context its sequential result."""
    from paper_1801_07986_b200 import PN

    ps = [inputs.plummer_bh(900, seed=41, dt=1e-3), inputs.plummer_bh(2100, seed=42, dt=1e-3)]
    ref = []
    for p in ps:
        with PN(p.mass, p.G, p.c, p.softening) as pn:
            pn.pn_set_state_host(p.pos, p.vel)
            pn.pn_step(p.dt, 12)
            ref.append(pn.pn_get_state_host())
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    pns = [PN(p.mass, p.G, p.c, p.softening, stream=s) for p, s in zip(ps, streams)]
    try:
        for pn, p in zip(pns, ps):
            pn.pn_set_state_host(p.pos, p.vel)
        for _ in range(4):  # 4 x 3 steps each, enqueued alternately without synchronising in between
            for pn, p in zip(pns, ps):
                pn.pn_step(p.dt, 3)
        got = [pn.pn_get_state_host() for pn in pns]
    finally:
        for pn in pns:
            pn.pn_destroy()
    for (x, v), (xr, vr) in zip(got, ref):
        assert np.array_equal(x, xr) and np.array_equal(v, vr)


def test_small_contexts_of_different_sizes_share_a_kernel():
    """Two contexts whose sizes map to the same kernel instance (IW = 2) but need different amounts of shared memory: the
    second pn_create must not lower the first one's limit."""
    from paper_1801_07986_b200 import PN

    big, small = inputs.plummer_bh(1180, seed=51, dt=1e-3), inputs.plummer_bh(600, seed=52, dt=1e-3)
    with PN(big.mass, big.G, big.c, big.softening) as a, PN(small.mass, small.G, small.c, small.softening) as b:
        assert a.pn_get_pair_config()["i_per_thread"] == b.pn_get_pair_config()["i_per_thread"] == 2
        for pn, p in ((a, big), (b, small), (a, big)):
            acc = pn.pn_accel(_dev(p.pos), _dev(p.vel)).cpu().numpy()
            ref = Oracle(p.mass, p.G, p.c, p.softening).accel(p.pos, p.vel)
            assert rel_err_rows(acc, ref).max() <= TOL_ACC
