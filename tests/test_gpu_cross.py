"""GPU parity of the NEXT rows of the scope table: [a_i]_Cross, Eq. 2.6, and [a_1]_Cross, Eq. 2.3
(PAPER.md:51-57), switched on with PN_OPT_CROSS_TERMS = PN_CROSS_STAR [| PN_CROSS_BH], against the oracle's literal
evaluation with the same terms.  Same tolerance as the hot path: err_i = max_k |a_ik - ref_ik| / ||ref_i||_2 <= 1e-12."""
import numpy as np
import pytest

from oracle.pn_oracle import CROSS_BH, CROSS_STAR, Oracle
from paper_1801_07986_b200 import inputs
from tests.conftest import rel_err_rows

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL_ACC = 1e-12


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


TERMS = [CROSS_STAR, CROSS_STAR | CROSS_BH]  # the oracle's mask values equal the library's PN_CROSS_* values


def _pn_cross(p, terms=CROSS_STAR):
    from paper_1801_07986_b200 import PN, binding

    assert (binding.PN_CROSS_STAR, binding.PN_CROSS_BH) == (CROSS_STAR, CROSS_BH)
    pn = PN(p.mass, p.G, p.c, p.softening)
    pn.pn_set_option(binding.PN_OPT_CROSS_TERMS, terms)
    return pn


@pytest.mark.parametrize("terms", TERMS)
# from 6144 stars on the Cross terms run in the symmetric kernel (every unordered pair once, variant 8 / 9): 64-star unit
# tiles in up to 128 groups of m tiles (m = 1 up to 8192 stars, 2 up to 16384, 3 at 20000)
@pytest.mark.parametrize("n_stars", [1, 2, 3, 129, 592, 593, 1023, 1185, 1279, 1280, 4099, 6143, 6144, 8200, 13001, 16383, 20000])
def test_cross_accel_parity_sizes(n_stars, terms):
    if n_stars <= 3:
        p = inputs.random_small(n_stars, seed=700 + n_stars, M=1.0, m_scale=1e-2, c=10.0, softening=1e-3, bh_moving=True)
    else:
        p = inputs.plummer_bh(n_stars, seed=700 + n_stars, c=20.0)  # a small c makes the 1PN terms 25 x larger than at c = 100
    ref = Oracle(p.mass, p.G, p.c, p.softening, terms=terms).accel(p.pos, p.vel)
    hot = Oracle(p.mass, p.G, p.c, p.softening).accel(p.pos, p.vel)
    from paper_1801_07986_b200 import binding

    with _pn_cross(p, terms) as pn:
        sym, small = n_stars >= 6144, n_stars <= 1279
        # symmetric kernel: 10 / 11 in its equal-mass form (these Plummer sets), 8 / 9 in the general form; ordered pairs: 5 / 6;
        # up to 1279 stars the small-system path (one cooperative launch per call): 12 / 13
        bhx = bool(terms & CROSS_BH)
        assert pn.pn_get_pair_config()["variant"] == ((13 if bhx else 12) if small else ((11 if bhx else 10) if sym else (6 if bhx else 5)))
        acc = pn.pn_accel(_dev(p.pos), _dev(p.vel)).cpu().numpy()
        again = pn.pn_accel(_dev(p.pos), _dev(p.vel)).cpu().numpy()
        if small:  # the same set through the multi-kernel path (ordered-pair kernel)
            pn.pn_set_option(binding.PN_OPT_PAIR_KERNEL, binding.PN_PAIR_TILED)
            assert pn.pn_get_pair_config()["variant"] == (6 if bhx else 5)
            tiled = pn.pn_accel(_dev(p.pos), _dev(p.vel)).cpu().numpy()
            assert rel_err_rows(tiled, ref).max() <= TOL_ACC
            pn.pn_set_option(binding.PN_OPT_PAIR_KERNEL, binding.PN_PAIR_AUTO)
        if sym:  # the same set through the general-mass form
            pn.pn_set_option(binding.PN_OPT_EQUAL_MASS, 0)
            assert pn.pn_get_pair_config()["variant"] == (9 if terms & CROSS_BH else 8)
            general = pn.pn_accel(_dev(p.pos), _dev(p.vel)).cpu().numpy()
            assert rel_err_rows(general, ref).max() <= TOL_ACC
            assert rel_err_rows(general, acc).max() <= 1e-13
    assert rel_err_rows(acc, ref).max() <= TOL_ACC
    assert np.array_equal(acc, again)  # fixed-order sums
    if n_stars >= 2:  # the Cross term is really there (with one star only the O(m_i) self line is left)
        assert rel_err_rows(hot[1:], ref[1:]).max() > 1e-9
    if terms & CROSS_BH:
        assert rel_err_rows(hot[:1], ref[:1]).max() > 1e-9  # [a_1]_Cross is really there
    else:
        assert np.array_equal(ref[0], hot[0])  # the massive object keeps Eqs. 2.1 + 2.2


@pytest.mark.parametrize("terms", TERMS)
@pytest.mark.parametrize("gen", ["cusp", "unequal_eps0", "tracers", "cusp_sym", "unequal_eps0_sym", "tracers_sym"])
def test_cross_accel_parity_other_inputs(gen, terms):
    """*_sym: sizes at which the symmetric Cross kernel runs (>= 6144 stars), compared on sampled rows + the massive object."""
    if gen == "cusp":
        p = inputs.cusp_bh(3000, seed=5)
    elif gen == "unequal_eps0":
        p = inputs.random_small(500, seed=8, M=1.0, m_scale=1e-3, c=10.0, softening=0.0, bh_moving=True)
    elif gen == "tracers":
        p = inputs.plummer_bh(700, seed=9, c=30.0)
        p.mass[10:200] = 0.0
    elif gen == "cusp_sym":
        p = inputs.cusp_bh(8000, seed=5)
    elif gen == "unequal_eps0_sym":
        p = inputs.random_small(7001, seed=8, M=1.0, m_scale=1e-4, c=10.0, softening=0.0, bh_moving=True)
    else:
        p = inputs.plummer_bh(6500, seed=9, c=30.0)
        p.mass[10:3000:3] = 0.0
    rows = np.arange(p.N) if p.N < 4000 else np.concatenate(
        [[0, 1, p.N - 1], np.sort(np.random.default_rng(3).choice(np.arange(2, p.N - 1), 1500, replace=False))])
    ref = Oracle(p.mass, p.G, p.c, p.softening, terms=terms).accel_rows(p.pos, p.vel, rows)
    with _pn_cross(p, terms) as pn:
        assert (pn.pn_get_pair_config()["variant"] in (8, 9, 10, 11)) == gen.endswith("_sym")
        acc = pn.pn_accel(_dev(p.pos), _dev(p.vel)).cpu().numpy()
    assert np.isfinite(acc).all()
    assert rel_err_rows(acc[rows], ref).max() <= TOL_ACC


@pytest.mark.parametrize("terms", TERMS)
def test_cross_symmetric_and_ordered_kernels_agree_and_track_the_oracle(terms):
    """6500 stars: the symmetric Cross kernel (default from 6144 stars) against the ordered-pair kernel (PN_PAIR_TILED) on
    every row, and three RK4 steps of each against the oracle with the same terms."""
    from paper_1801_07986_b200 import PN, binding

    p = inputs.plummer_bh(6500, seed=21, c=20.0, dt=1e-3)
    xr, vr = Oracle(p.mass, p.G, p.c, p.softening, terms=terms).step(p.pos, p.vel, p.dt, 3)
    acc, traj = {}, {}
    for kernel in (binding.PN_PAIR_AUTO, binding.PN_PAIR_TILED):
        with PN(p.mass, p.G, p.c, p.softening) as pn:
            pn.pn_set_option(binding.PN_OPT_PAIR_KERNEL, kernel)  # before the Cross option: it sizes the Cross buffers
            pn.pn_set_option(binding.PN_OPT_CROSS_TERMS, terms)
            assert (pn.pn_get_pair_config()["variant"] in (8, 9, 10, 11)) == (kernel == binding.PN_PAIR_AUTO)
            acc[kernel] = pn.pn_accel(_dev(p.pos), _dev(p.vel)).cpu().numpy()
            pn.pn_set_state_host(p.pos, p.vel)
            pn.pn_step(p.dt, 3)
            traj[kernel] = pn.pn_get_state_host()
    assert rel_err_rows(acc[binding.PN_PAIR_AUTO], acc[binding.PN_PAIR_TILED]).max() <= 1e-13
    for x, v in traj.values():
        assert max(rel_err_rows(x, xr).max(), rel_err_rows(v, vr).max()) <= 1e-11


def test_cross_switch_off_restores_the_hot_path_bitwise_and_is_deterministic():
    from paper_1801_07986_b200 import PN, binding

    p = inputs.plummer_bh(4099, seed=11, c=20.0)
    with PN(p.mass, p.G, p.c, p.softening) as pn:
        pos, vel = _dev(p.pos), _dev(p.vel)
        a0 = pn.pn_accel(pos, vel).cpu().numpy()
        pn.pn_set_option(binding.PN_OPT_CROSS_TERMS, binding.PN_CROSS_STAR)
        c1 = pn.pn_accel(pos, vel).cpu().numpy()
        c2 = pn.pn_accel(pos, vel).cpu().numpy()
        pn.pn_set_option(binding.PN_OPT_CROSS_TERMS, 0)
        a1 = pn.pn_accel(pos, vel).cpu().numpy()
        with pytest.raises(binding.PNError):
            pn.pn_set_option(binding.PN_OPT_CROSS_TERMS, binding.PN_CROSS_BH)  # Eq. 2.3 needs the sums of Eq. 2.6: not alone
    assert np.array_equal(a0, a1) and np.array_equal(c1, c2) and not np.array_equal(a0, c1)


@pytest.mark.parametrize("kernel", ["auto", "tiled"])
@pytest.mark.parametrize("terms", TERMS)
def test_cross_rk4_trajectory_tracks_oracle(terms, kernel):
    """pn_step with the Cross terms against the oracle's RK4 with the same terms.  auto: 600 stars take the small-system
    path (one cooperative launch for the 20 steps); tiled: the multi-kernel path, as a CUDA graph and as plain launches."""
    from paper_1801_07986_b200 import binding

    p = inputs.plummer_bh(600, seed=13, c=20.0, dt=1e-3)
    xr, vr = Oracle(p.mass, p.G, p.c, p.softening, terms=terms).step(p.pos, p.vel, p.dt, 20)
    xh, vh = Oracle(p.mass, p.G, p.c, p.softening).step(p.pos, p.vel, p.dt, 20)
    out = []
    for use_graph in (1, 0):
        with _pn_cross(p, terms) as pn:
            if kernel == "tiled":
                pn.pn_set_option(binding.PN_OPT_PAIR_KERNEL, binding.PN_PAIR_TILED)
            assert pn.pn_get_pair_config()["variant"] == ((6 if terms & CROSS_BH else 5) if kernel == "tiled" else (13 if terms & CROSS_BH else 12))
            pn.pn_set_option(binding.PN_OPT_USE_GRAPH, use_graph)
            pn.pn_set_state_host(p.pos, p.vel)
            pn.pn_step(p.dt, 20)
            out.append(pn.pn_get_state_host())
    (x, v), (x2, v2) = out
    assert np.array_equal(x, x2) and np.array_equal(v, v2)
    assert max(rel_err_rows(x, xr).max(), rel_err_rows(v, vr).max()) <= 1e-11
    assert rel_err_rows(v, vh).max() > 1e-9  # and it is not the hot-path trajectory


@pytest.mark.parametrize("kernel", ["auto", "tiled", "symmetric"])
def test_cross_hand_values_softened_345_on_gpu(kernel):
    """tests/golden/n3_345_softened_cross.txt (Eqs. 2.6 + 2.3 with rho_AB = 6, worked by hand) straight through the C-ABI:
    the small-system kernel, the ordered-pair kernel and the symmetric kernel each soften every star-star distance."""
    from paper_1801_07986_b200 import PN, binding
    from tests.conftest import load_golden

    g = load_golden("n3_345_softened_cross.txt")
    opt = {"auto": binding.PN_PAIR_AUTO, "tiled": binding.PN_PAIR_TILED, "symmetric": binding.PN_PAIR_SYMMETRIC}[kernel]
    for terms, key in ((CROSS_STAR, "acc_cross_star"), (CROSS_STAR | CROSS_BH, "acc_cross_full")):
        with PN(g["mass"], g["G"], g["c"], g["eps"]) as pn:
            pn.pn_set_option(binding.PN_OPT_CROSS_TERMS, terms)
            pn.pn_set_option(binding.PN_OPT_PAIR_KERNEL, opt)
            acc = pn.pn_accel(_dev(g["pos"]), _dev(g["vel"])).cpu().numpy()
        assert rel_err_rows(acc, g[key]).max() <= 1e-14, (kernel, key)
        # the Cross part by itself is 1e-4 of a_i here: it must be right to 1e-10 of its own size
        hot = load_golden("n3_345_softened.txt")["acc"]
        cr = (acc - hot) * g["c"] ** 2
        np.testing.assert_allclose(cr[1:], g["cross_star"], rtol=0, atol=1e-10 * np.abs(g["cross_star"]).max())
        if terms & CROSS_BH:
            np.testing.assert_allclose(cr[0], g["cross_bh"], rtol=0, atol=1e-9 * np.abs(g["cross_bh"]).max())
