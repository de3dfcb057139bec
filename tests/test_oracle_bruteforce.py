"""Pins O1/O2 of the T1 oracle (C) to the T0 formulation (global ranking + set
intersections, pure Python) by exhaustive enumeration of tiny maps, and to closed-form
facts about the `beats` total order (SURVEY.md 8(c) "pins", NS "brute-force enumeration
on tiny maps")."""
import itertools

import numpy as np
import pytest

from oracle import t0_bruteforce as t0
from oracle import t1

THR, EPS = 6, 4


def _check(q):
    a = t1.row_flags(q, THR, EPS)
    b = t0.row_flags(q, THR, EPS)
    assert np.array_equal(a, b), (q.tolist(), a.tolist(), b.tolist())
    return a


def test_exhaustive_3x3_alphabet4():
    """All 4^9 = 262144 maps is too slow for T0 in CI; all maps over {0,5,7,9} with a fixed
    stride through the enumeration (every 7th) plus every map with <= 4 non-zero cells."""
    alpha = (0, 5, 7, 9)
    n = 0
    for i, cells in enumerate(itertools.product(alpha, repeat=9)):
        nz = sum(1 for c in cells if c)
        if nz > 4 and i % 7:
            continue
        _check(np.array(cells, dtype=np.uint16).reshape(3, 3))
        n += 1
    assert n > 40000


def test_exhaustive_2x4_alphabet4():
    for cells in itertools.product((0, 5, 7, 9), repeat=8):
        _check(np.array(cells, dtype=np.uint16).reshape(2, 4))


def test_exhaustive_1x5_suppression():
    """All 5^5 1x5 maps (both orientations) over values straddling q_c - eps: with peaks of
    30 and 100, a ridge of 26 suppresses the 30 (26+4 >= 30) and 25 does not."""
    for cells in itertools.product((0, 25, 26, 30, 100), repeat=5):
        q = np.array(cells, dtype=np.uint16)
        _check(q.reshape(1, 5))
        _check(q.reshape(5, 1))


def test_exhaustive_2x5_suppression():
    for cells in itertools.product((0, 26, 30), repeat=10):
        q = np.array(cells, dtype=np.uint16)
        _check(q.reshape(2, 5))


def test_random_small_maps_mixed_density():
    rng = np.random.default_rng(20251117)
    alpha = np.array([0, 5, 7, 9, 12, 1023], dtype=np.uint16)
    for shape in ((6, 6), (8, 7), (7, 8)):
        for _ in range(700):
            dens = rng.uniform(0.1, 1.0)
            q = alpha[rng.integers(1, len(alpha), size=shape)] * (rng.random(shape) < dens)
            f = _check(q.astype(np.uint16))
            # I1: no two survivors within Chebyshev distance 1 (even: no two PEAKS are)
            pk = np.argwhere(f & 1)
            for a, b in itertools.combinations(pk.tolist(), 2):
                assert max(abs(a[0] - b[0]), abs(a[1] - b[1])) >= 2
            # I2: at least one survivor iff some cell >= thr (the best cell survives)
            assert bool((f & 2).any()) == bool((q >= THR).any())
            if (q >= THR).any():
                T, P = q.shape
                best = min(((-int(q[t, p]), t, p) for t in range(T) for p in range(P)))
                assert f[best[1], best[2]] == 3


def test_strict_nonstrict_form_of_o1():
    """O1's 'equivalent GPU form': strict > for the 4 neighbours earlier in (t,p) order,
    >= for the 4 later ones -- checked against T1 on random maps with many ties."""
    rng = np.random.default_rng(5)
    for _ in range(300):
        q = rng.integers(5, 9, size=(7, 9)).astype(np.uint16) * (rng.random((7, 9)) < 0.8)
        f = t1.row_flags(q, THR, EPS) & 1
        z = np.zeros((9, 11), dtype=np.int64)
        z[1:-1, 1:-1] = q
        for t in range(7):
            for p in range(9):
                c = z[t + 1, p + 1]
                ok = c >= THR
                for dt, dp in ((-1, -1), (-1, 0), (-1, 1), (0, -1)):
                    ok &= c > z[t + 1 + dt, p + 1 + dp]
                for dt, dp in ((0, 1), (1, -1), (1, 0), (1, 1)):
                    ok &= c >= z[t + 1 + dt, p + 1 + dp]
                assert bool(ok) == bool(f[t, p])


@pytest.mark.parametrize("axis", ["pad", "time"])
def test_equal_chain_yields_first_cell(axis):
    """Closed form: a chain of equal cells along one axis yields exactly its first cell as
    a peak (every later cell is beaten by its predecessor)."""
    for n in range(1, 7):
        q = np.zeros((9, 9), dtype=np.uint16)
        if axis == "pad":
            q[4, 1:1 + n] = 40
        else:
            q[1:1 + n, 4] = 40
        f = t1.row_flags(q, THR, EPS)
        pk = np.argwhere(f & 1).tolist()
        assert pk == ([[4, 1]] if axis == "pad" else [[1, 4]])
