"""BASELINE.json configs 2, 3 and 4 run AS STATED through the CUDA path, against the long-double oracle.

config 2 (configs[1], the metric's config): N = 1+16383 Plummer + BH 0.1, dt = 1e-4, all 50 steps: trajectory and 1PN
    energy after every step against the oracle's 50-step run (tests/golden/config2_digest.npz, 128 rows per step; the
    full run with 2048 rows + the final state in tests/cache/ when present), same script as config 3.

config 3 (configs[2]): N = 1+65535 Bahcall-Wolf cusp, dt = 1e-5, 20 steps, "1PN energy drift tracked": the GPU trajectory
    and E after every step against the oracle's full-size 20-step run (3.4e11 long-double pair visits + 21 O(N^2)
    energies; produced once by tests/make_fullsize_refs.py, which calls only oracle/, and kept in tests/cache/ outside
    git -- SURVEY.md section 7 item 11; a committed subset of the same run, tests/golden/config3_digest.npz, serves when
    the cache file is absent).
config 4 (configs[3]): N = 1+262143 Plummer + BH 0.05, dt = 1e-4, 10 steps in BOTH pair precisions with pn_energy after
    every step: pn_accel at the GPU's state after every step against the oracle on a seeded subset of 4096 i-rows (each
    against all j) + the massive object's row, and the energy of the full initial set against the oracle's
    (tests/golden/config4_energy.txt, same script).
"""
import numpy as np
import pytest

from oracle.pn_oracle import Oracle
from paper_1801_07986_b200 import inputs
from tests.conftest import GOLDEN, rel_err_rows
from tests.make_fullsize_refs import CACHE, ref_key

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL_ACC = 1e-12
TOL_FP32 = 1e-5
TOL_DRIFT = 1e-10
TOL_TRAJ = 1e-10


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def load_traj_reference(p, name):
    """The oracle's run of a config as stated: the full cache if it is there, else the committed subset of the same run."""
    key = ref_key(p)
    for path in (CACHE / f"{name}_traj.npz", GOLDEN / f"{name}_digest.npz"):
        if path.exists():
            z = np.load(path)
            if str(z["key"]) == key:
                return {k: z[k] for k in z.files}, path.name
    pytest.fail(f"no oracle reference for {name} matches oracle/pn_oracle.c and the seeded inputs: "
                f"run `python tests/make_fullsize_refs.py --only {name}` (config 3: about 1.5 h of host time, config 2: 0.5 h)")


def load_config3_reference(p):
    return load_traj_reference(p, "config3")


def _run_as_stated(p, ref, variant):
    """pn_step one step at a time; after every step the sampled rows of (x, v) and the drift against the oracle's."""
    from paper_1801_07986_b200 import PN

    rows, E = ref["rows"], ref["E"]
    assert E.shape == (p.nsteps + 1,) and ref["x_rows"].shape[:2] == (p.nsteps, rows.size)
    with PN(p.mass, p.G, p.c, p.softening) as pn:
        assert pn.pn_get_pair_config()["variant"] == variant  # the kernel bench.py times at this size
        pn.pn_set_state_host(p.pos, p.vel)
        e0 = pn.pn_energy()
        assert e0 == pytest.approx(E[0], rel=1e-13)
        worst_traj = worst_drift = 0.0
        for s in range(p.nsteps):
            pn.pn_step(p.dt, 1)
            x, v = pn.pn_get_state_host()
            worst_traj = max(worst_traj, rel_err_rows(x[rows], ref["x_rows"][s]).max(),
                             rel_err_rows(v[rows], ref["v_rows"][s]).max())
            d_gpu = (pn.pn_energy() - e0) / abs(e0)
            d_ref = (E[s + 1] - E[0]) / abs(E[0])
            worst_drift = max(worst_drift, abs(d_gpu - d_ref))
        if "x_final" in ref:  # the cache holds every row of the final state
            worst_traj = max(worst_traj, rel_err_rows(x, ref["x_final"]).max(), rel_err_rows(v, ref["v_final"]).max())
    return worst_traj, worst_drift, d_ref


def test_config2_full_size_50_steps():
    """The metric's configuration exactly as BASELINE.json states it: 50 RK4 steps at N = 1+16383, every step compared."""
    p = inputs.config(2)
    ref, source = load_traj_reference(p, "config2")
    assert p.nsteps == 50
    worst_traj, worst_drift, d_last = _run_as_stated(p, ref, variant=4)
    print(f"config 2 ({source}): oracle drift after 50 steps {d_last:.3e}, worst trajectory error {worst_traj:.2e}, "
          f"worst drift difference {worst_drift:.2e}")
    assert worst_traj <= TOL_TRAJ
    assert worst_drift <= TOL_DRIFT


def load_config4_energy(p):
    kv = dict(line.split(None, 1) for line in (GOLDEN / "config4_energy.txt").read_text().splitlines()
              if line and not line.startswith("#"))
    if kv["key"].strip() != ref_key(p):
        pytest.fail("tests/golden/config4_energy.txt is stale: run `python tests/make_fullsize_refs.py --only config4`")
    return float.fromhex(kv["energy_hex"].strip())


def test_config3_full_size_20_steps():
    from paper_1801_07986_b200 import PN

    p = inputs.config(3)
    ref, source = load_config3_reference(p)
    rows, E = ref["rows"], ref["E"]
    assert p.nsteps == 20 and E.shape == (21,) and ref["x_rows"].shape[:2] == (20, rows.size)
    with PN(p.mass, p.G, p.c, p.softening) as pn:
        assert pn.pn_get_pair_config()["variant"] == 4  # the kernel bench.py times at this size
        pn.pn_set_state_host(p.pos, p.vel)
        e0 = pn.pn_energy()
        assert e0 == pytest.approx(E[0], rel=1e-13)
        worst_traj = worst_drift = 0.0
        drift = []
        for s in range(p.nsteps):
            pn.pn_step(p.dt, 1)
            x, v = pn.pn_get_state_host()
            worst_traj = max(worst_traj, rel_err_rows(x[rows], ref["x_rows"][s]).max(),
                             rel_err_rows(v[rows], ref["v_rows"][s]).max())
            d_gpu = (pn.pn_energy() - e0) / abs(e0)
            d_ref = (E[s + 1] - E[0]) / abs(E[0])
            drift.append(d_ref)
            worst_drift = max(worst_drift, abs(d_gpu - d_ref))
        if "x_final" in ref:  # the cache holds every row of the final state
            worst_traj = max(worst_traj, rel_err_rows(x, ref["x_final"]).max(), rel_err_rows(v, ref["v_final"]).max())
    print(f"config 3 ({source}): oracle drift after 20 steps {drift[-1]:.3e}, worst trajectory error {worst_traj:.2e}, "
          f"worst drift difference {worst_drift:.2e}")
    assert worst_traj <= TOL_TRAJ
    assert worst_drift <= TOL_DRIFT


def test_config3_energy_full_size_against_long_double():
    """E of the full initial set (4.3e9 ordered pairs) against the long-double oracle's value."""
    from paper_1801_07986_b200 import PN

    p = inputs.config(3)
    ref, _ = load_config3_reference(p)
    with PN(p.mass, p.G, p.c, p.softening) as pn:
        pn.pn_set_state_host(p.pos, p.vel)
        e = pn.pn_energy()
        e_again = pn.pn_energy()
    assert e == e_again
    assert e == pytest.approx(float(ref["E"][0]), rel=1e-13)


def test_config4_10_steps_both_variants_energy_every_step():
    from paper_1801_07986_b200 import PN, binding

    p = inputs.config(4)
    e_ref = load_config4_energy(p)
    rng = np.random.default_rng(4096)
    rows = np.concatenate([[0], np.sort(rng.choice(np.arange(1, p.N), size=4096, replace=False))]).astype(np.int64)
    o = Oracle(p.mass, p.G, p.c, p.softening)
    energies = {}
    for prec, tol in ((binding.PN_FP64, TOL_ACC), (binding.PN_FP32_PAIR, TOL_FP32)):
        with PN(p.mass, p.G, p.c, p.softening) as pn:
            pn.pn_set_option(binding.PN_OPT_PAIR_PRECISION, prec)
            pn.pn_set_state_host(p.pos, p.vel)
            e = [pn.pn_energy()]
            assert e[0] == pytest.approx(e_ref, rel=1e-13)  # pn_energy is fp64 in both variants
            worst = 0.0
            for s in range(p.nsteps):
                pn.pn_step(p.dt, 1)
                e.append(pn.pn_energy())
                xg, vg = pn.pn_get_state()
                acc = pn.pn_accel(xg, vg).cpu().numpy()
                xh, vh = xg.cpu().numpy(), vg.cpu().numpy()
                assert np.isfinite(acc).all()
                worst = max(worst, rel_err_rows(acc[rows], o.accel_rows(xh, vh, rows)).max())
            assert worst <= tol, (prec, worst)
            if prec == binding.PN_FP32_PAIR:
                assert worst > 1e-9  # it really is the fp32-pair path
            energies[prec] = np.array(e)
    e64, e32 = energies[binding.PN_FP64], energies[binding.PN_FP32_PAIR]
    assert p.nsteps == 10 and e64.shape == (11,)
    # the run barely drifts (t = 1e-3 of a crossing time); the fp32-pair run stays on the fp64 run's energy
    assert np.abs((e64 - e64[0]) / e64[0]).max() <= 1e-7
    assert np.abs((e32 - e64) / e64).max() <= 1e-8
