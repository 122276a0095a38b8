"""Pins of the Morton-order oracle (oracle/morton_oracle.py): hand-computed codes, a per-element pure-Python
interleave, the defining properties of a Z-order curve, and exact-arithmetic quantisation."""
from fractions import Fraction

import numpy as np

from oracle import morton_oracle as M


def py_interleave(qx, qy, qz):
    code = 0
    for k in range(21):
        code |= ((qx >> k) & 1) << (3 * k + 2)
        code |= ((qy >> k) & 1) << (3 * k + 1)
        code |= ((qz >> k) & 1) << (3 * k)
    return code


def test_hand_computed_codes():
    q = np.array([[0, 0, 0], [1, 0, 0], [0, 1, 0], [0, 0, 1], [1, 1, 1], [2, 0, 0], [3, 5, 6],
                  [2 ** 21 - 1, 2 ** 21 - 1, 2 ** 21 - 1]], dtype=np.uint64)
    got = M.interleave(q)
    # (3, 5, 6) = x 011, y 101, z 110 -> bit triples (x y z) from the top: 011, 101, 110 -> 0b011101110
    want = [0, 4, 2, 1, 7, 32, 0b011101110, 2 ** 63 - 1]
    assert [int(c) for c in got] == want


def test_interleave_matches_pure_python_on_random_integers():
    rng = np.random.default_rng(0)
    q = rng.integers(0, 2 ** 21, (500, 3), dtype=np.uint64)
    got = M.interleave(q)
    for i in range(500):
        assert int(got[i]) == py_interleave(int(q[i, 0]), int(q[i, 1]), int(q[i, 2]))


def test_z_order_properties():
    rng = np.random.default_rng(1)
    q = rng.integers(0, 2 ** 21 - 1, (200, 3), dtype=np.uint64)
    c = M.interleave(q)
    for axis in range(3):                       # monotone along every axis
        q2 = q.copy(); q2[:, axis] += np.uint64(1)
        assert np.all(M.interleave(q2) > c)
    # all points of an aligned 2^k cube share the code's high bits: codes of the 8 children of a cell are contiguous
    base = np.array([[6, 10, 12]], dtype=np.uint64)            # even coordinates: an aligned 2-cube
    kids = np.array([[dx, dy, dz] for dx in (0, 1) for dy in (0, 1) for dz in (0, 1)], dtype=np.uint64) + base
    ck = np.sort(M.interleave(kids))
    assert np.array_equal(ck, ck[0] + np.arange(8, dtype=np.uint64)) and int(ck[0]) % 8 == 0


def test_quantisation_against_exact_rational_arithmetic():
    rng = np.random.default_rng(2)
    means = rng.uniform(-7.0, 13.0, (300, 3)).astype(np.float32)
    lo, hi = M.bounds(means)
    sc = M.scales(lo, hi)
    q = M.quantise(means, lo, hi)
    assert q.min() == 0 and q.max() == 2 ** 21 - 1             # the box corners map to the first and the last cell
    for i in range(300):
        for a in range(3):
            d = np.float32(means[i, a]) - np.float32(lo[a])     # fp32 difference, as specified (one rounding)
            t = np.float32(d) * np.float32(sc[a])               # fp32 product (one rounding)
            exact = Fraction(float(t))                          # the rounded product, floored exactly
            want = min(max(exact.numerator // exact.denominator, 0), 2 ** 21 - 1)
            assert int(q[i, a]) == want
    # within half a cell of the real-valued position
    real = (means.astype(np.float64) - lo.astype(np.float64)) / (hi.astype(np.float64) - lo.astype(np.float64)) * 2 ** 21
    assert np.abs(np.clip(np.floor(real), 0, 2 ** 21 - 1) - q.astype(np.float64)).max() <= 1


def test_degenerate_axis_and_order_is_stable():
    means = np.zeros((6, 3), np.float32)
    means[:, 0] = [3, 1, 2, 1, 3, 2]                           # y and z degenerate (hi == lo): scale 1, q = 0
    perm = M.morton_order(means)
    assert perm.tolist() == [1, 3, 2, 5, 0, 4]                 # ties keep ascending index
    assert M.scales(*M.bounds(means)).tolist()[1:] == [1.0, 1.0]


def test_order_groups_spatial_neighbours():
    """After the sort, consecutive Gaussians are much closer in space than in a random order."""
    rng = np.random.default_rng(3)
    means = rng.uniform(0, 1, (20000, 3)).astype(np.float32)
    perm = M.morton_order(means)
    d_sorted = np.linalg.norm(np.diff(means[perm], axis=0), axis=1).mean()
    d_random = np.linalg.norm(np.diff(means, axis=0), axis=1).mean()
    assert d_sorted < 0.15 * d_random
