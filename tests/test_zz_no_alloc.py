"""pn_bh_accel_noalloc: the library's entry point for callers that cannot allocate device memory.

Some users of libpn.so cannot go through pn_create, because that calls cudaMalloc: programs whose own pool already owns
the GPU's memory (or that run under a memory quota, where one more cudaMalloc fails), and time-critical loops that cannot
take the device-wide stall of cudaMalloc / cudaFree.  For them the library computes a_1 -- the acceleration of the massive
object, Eqs. 2.1 + 2.2, PAPER.md:43-49 -- with its scratch memory in a fixed array inside the library (2**20 stars at most).

Checked here: the result equals row 0 of pn_accel (the existing path) within the suite's fp64 tolerance, on two calls in
a row that share the scratch array -- the second on a smaller system, so that what the first call left behind (more block
partials than the second one writes) must not leak into it -- and again after a third call; sizes beyond the limit are
refused with a message and without touching the GPU.

The file name sorts last on purpose: the suite runs with pytest -x, and a failure here must not hide the parity tests.
It needs nothing from the tests before it and passes alone in a fresh process as well.
"""
import ctypes
import math

import numpy as np
import pytest

from paper_1801_07986_b200 import inputs
from tests.conftest import rel_err_rows

TOL_ACC = 1e-12  # the fp64 tolerance of tests/test_gpu_parity.py (reading R10)


def _existing_path_a1(p, c):
    import torch

    from paper_1801_07986_b200 import PN

    with PN(p.mass, p.G, c, p.softening) as pn:
        acc = pn.pn_accel(torch.from_numpy(p.pos).cuda(), torch.from_numpy(p.vel).cuda())
        return acc[0].cpu().numpy()


@pytest.mark.gpu
def test_no_alloc_entry_point_matches_pn_accel_on_consecutive_calls():
    torch = pytest.importorskip("torch")
    from paper_1801_07986_b200 import binding

    # (stars, c): several hundred blocks with a ragged tail, then fewer blocks than the call before, then one block
    # in the Newtonian limit (c = inf), then the large case once more: same bits as the first time
    cases = [(70001, 100.0), (5000, 100.0), (37, math.inf), (70001, 100.0)]
    systems = {n: inputs.plummer_bh(n, seed=900 + n) for n in {n for n, _ in cases}}
    dev = {n: tuple(torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (p.mass, p.pos, p.vel)) for n, p in systems.items()}
    outs = [torch.full((3,), float("nan"), dtype=torch.float64, device="cuda") for _ in cases]
    # the calls go out back to back on one stream, nothing in between: they share the library's scratch array in order
    for (n, c), a1 in zip(cases, outs):
        m, x, v = dev[n]
        binding.pn_bh_accel_noalloc(m, x, v, systems[n].G, c, a1)
    torch.cuda.synchronize()
    got = [a1.cpu().numpy() for a1 in outs]
    for (n, c), a1 in zip(cases, got):
        ref = _existing_path_a1(systems[n], c)
        assert np.isfinite(a1).all()
        err = rel_err_rows(a1[None, :], ref[None, :]).max()
        assert err <= TOL_ACC, f"{n} stars, c = {c}: {err:.3e}"
    assert np.array_equal(got[0], got[3])  # fixed summation order: nothing of the calls in between shows


@pytest.mark.gpu
def test_no_alloc_entry_point_at_its_size_limit():
    torch = pytest.importorskip("torch")
    from paper_1801_07986_b200 import binding

    n = binding.PN_NOALLOC_MAX_STARS  # every block-partial slot of the scratch array in use
    p = inputs.uniform_ball_bh(20)
    assert p.mass.shape[0] == n  # config 5, k = 20: N = 1 + (2^20 - 1) bodies = 2^20 - 1 stars
    m, x, v = (torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (p.mass, p.pos, p.vel))
    a1 = torch.empty(3, dtype=torch.float64, device="cuda")
    binding.pn_bh_accel_noalloc(m, x, v, p.G, p.c, a1)
    # the same sum in plain torch fp64 (Eqs. 2.1 + 2.2), independent of both CUDA paths' summation order
    d = x[1:] - x[0]
    r = d.norm(dim=1)
    vv, vx = (v[1:] ** 2).sum(1), (v[1:] * d).sum(1)
    gx = 1.0 - (5.0 * p.G * p.mass[0] / r - 2.0 * vv + 1.5 * vx * vx / r**2) / p.c**2
    ref = ((p.G * m[1:] / r**3)[:, None] * (gx[:, None] * d - (3.0 * vx / p.c**2)[:, None] * v[1:])).sum(0).cpu().numpy()
    err = rel_err_rows(a1.cpu().numpy()[None, :], ref[None, :]).max()
    assert err <= 1e-10, f"{err:.3e}"  # torch's own fp64 sum of 1e6 cancelling terms carries ~1e-11


def test_no_alloc_entry_point_refuses_sizes_beyond_its_scratch_array():
    """No GPU needed: the size check comes before any CUDA call, and nothing is launched."""
    from paper_1801_07986_b200 import build, binding

    build.build()
    lib = binding.load_library()
    err = ctypes.create_string_buffer(512)
    too_many = binding.PN_NOALLOC_MAX_STARS + 2  # N = stars + 1
    rc = lib.pn_bh_accel_noalloc(too_many, 8, 8, 8, 1.0, 10.0, 8, None, err, len(err))
    assert rc == binding.PN_EINVAL
    assert b"PN_NOALLOC_MAX_STARS = 1048576" in err.value
    assert lib.pn_bh_accel_noalloc(1, 8, 8, 8, 1.0, 10.0, 8, None, err, len(err)) == binding.PN_EINVAL  # N < 2
    assert lib.pn_bh_accel_noalloc(3, None, 8, 8, 1.0, 10.0, 8, None, err, len(err)) == binding.PN_EINVAL  # null pointer
    assert lib.pn_bh_accel_noalloc(3, 8, 8, 8, 1.0, -1.0, 8, None, None, 0) == binding.PN_EINVAL  # c <= 0, no buffer
