"""Combinatorics behind the symmetric pair kernels (paper_1801_07986_b200/csrc/pn_pair_fp64.cuh, pn_pair_cross.cuh, pn_energy.cuh), checked on the CPU.

The kernels let the j-side sums of a 32-star sub-group travel through the lanes of a warp in Gray-code order: at step r lane l
works on j-star l ^ g(r), g(r) = r ^ (r >> 1), and after the step the sums move with a butterfly shuffle (lane l receives from
lane l ^ mask).  These tests replay exactly the index and mask formulas the kernels use (16-step halves in
sym_unit_tile_gray / sym32_unit_tile_gray, chunks of CSTEPS steps in pair_cross_sym_kernel) and assert what the kernels rely on:
every lane meets every j-star exactly once, the sums always sit in the lane that works on their star, and after step 31 they are
back in their home lane.  Also the work-item decodings (triangular block index, upper-triangular tile-pair list)."""
import math

import pytest


def gray(r):
    return r ^ (r >> 1)


def walk(chunk):
    """(j offset, shuffle mask after the step) for the 32 steps, from the kernels' formulas for chunks of `chunk` steps."""
    steps = []
    for c in range(32 // chunk):
        r0, r1, r2 = chunk * c, chunk * c + chunk - 1, (chunk * c + chunk) & 31
        off = gray(r0)                      # base = jb + (lane ^ g(r0))
        last_mask = gray(r1) ^ gray(r2)     # into the next chunk or, after step 31, home
        for q in range(chunk):
            mask = ((q + 1) & -(q + 1)) if q + 1 < chunk else last_mask
            steps.append((off ^ gray(q), mask))
    return steps


@pytest.mark.parametrize("chunk", [4, 8, 16])
def test_gray_walk_meets_every_star_once_and_returns_home(chunk):
    steps = walk(chunk)
    assert len(steps) == 32
    # closed forms the kernels hard-code: halves start at 0 and 24; quarters at 0, 12, 24, 20; last masks 16 / (8, 16, 8, 16)
    if chunk == 16:
        assert [steps[0][0], steps[16][0]] == [0, 24] and [steps[15][1], steps[31][1]] == [16, 16]
    if chunk == 8:
        assert [steps[8 * c][0] for c in range(4)] == [0, 12, 24, 20]
        assert [steps[8 * c + 7][1] for c in range(4)] == [8, 16, 8, 16]
    owner = list(range(32))  # owner[lane] = j-star whose sums sit in that lane; lane l starts with star l ^ g(0) = l
    met = [set() for _ in range(32)]
    for off, mask in steps:
        for lane in range(32):
            j = lane ^ off
            assert owner[lane] == j          # the sums are where their star is being worked on
            assert j not in met[lane]
            met[lane].add(j)
        assert mask in (1, 2, 4, 8, 16)      # single-bit butterfly, an immediate in the unrolled body
        owner = [owner[lane ^ mask] for lane in range(32)]
    assert all(m == set(range(32)) for m in met)
    assert owner == list(range(32))          # home again: lane l stores the sums of star jb + l


def test_triangular_block_decode():
    """sym_decode_block: id = B (B + 1) / 2 + A with A <= B, float sqrt first guess + integer correction."""
    def decode(i):
        b = int((math.sqrt(8.0 * i + 1.0) - 1.0) * 0.5)
        while (b + 1) * (b + 2) // 2 <= i:
            b += 1
        while b * (b + 1) // 2 > i:
            b -= 1
        return i - b * (b + 1) // 2, b

    seen = set()
    for g in (1, 2, 7, 128):
        for i in range(g * (g + 1) // 2):
            a, b = decode(i)
            assert 0 <= a <= b < g
            seen.add((g, a, b))
        assert len({(a, b) for (gg, a, b) in seen if gg == g}) == g * (g + 1) // 2


@pytest.mark.parametrize("n_tiles", [1, 2, 3, 8, 129, 8192])
def test_upper_triangular_tile_pair_list(n_tiles):
    """tri_decode + the row-by-row walk of energy_pair_kernel / momentum_pair_kernel: equal runs cover every (it <= jt) once."""
    def off(q):
        return q * n_tiles - q * (q - 1) // 2

    def decode(p):
        b = 2.0 * n_tiles + 1.0
        r = int((b - math.sqrt(b * b - 8.0 * p)) * 0.5)
        r = max(0, min(r, n_tiles - 1))
        while r > 0 and off(r) > p:
            r -= 1
        while r + 1 < n_tiles and off(r + 1) <= p:
            r += 1
        return r, r + (p - off(r))

    n_pairs = n_tiles * (n_tiles + 1) // 2
    per_block = max(1, -(-n_pairs // (148 * 7)))
    probes = range(n_pairs) if n_pairs <= 10000 else list(range(0, n_pairs, 9973)) + [n_pairs - 1]
    for p in probes:
        it, jt = decode(p)
        assert 0 <= it <= jt < n_tiles and off(it) + (jt - it) == p
    if n_pairs <= 10000:  # replay the kernel's walk block by block
        seen = []
        for b in range(-(-n_pairs // per_block)):
            p0, p1 = b * per_block, min(n_pairs, (b + 1) * per_block)
            it, jt = decode(p0)
            for _ in range(p0, p1):
                seen.append((it, jt))
                jt += 1
                if jt == n_tiles:
                    it, jt = it + 1, it + 1
        assert seen == [(i, j) for i in range(n_tiles) for j in range(i, n_tiles)]
