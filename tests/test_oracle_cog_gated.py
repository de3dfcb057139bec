"""Pins of reading Q10' (R7): outer-ring gating of the 5x5 CoG.
An outer-ring cell counts only if the inner cell between it and the peak holds charge.  Hand
vectors with sums worked out by hand and finalised by exact rational arithmetic (exact_f32),
T0 (pure Python definition) against T1 (C) on random maps, and the identity with the ungated
reading whenever the inner ring is full."""
import numpy as np

from exact_f32 import finalize_exact
from oracle import t0_bruteforce as t0
from oracle import t1

P, T = 40, 120


def _run(cells, gated):
    d = t1.make_digits([(0, 0, p, t, q) for (p, t, q) in cells])
    cl, st, n = t1.clusterize(d, 1, 1, T, [P], 6, 4, cog_gated=gated)
    assert st == 0 and n == len(cl)
    return cl


def _bits(x):
    return int(np.array(x, dtype=np.float32).view(np.uint32))


def _expect(c, Q, Sp, St, Spp, Stt, p_c, t_c):
    e = finalize_exact(Q, Sp, St, Spp, Stt, p_c, t_c)
    assert int(c["q_tot"]) == Q and (int(c["pad_peak"]), int(c["time_peak"])) == (p_c, t_c)
    assert [_bits(c[k]) for k in ("pad_mean", "time_mean", "sigma_pad", "sigma_time")] == e


def test_isolated_outer_cell_is_cut_off():
    # A = 100 at (10,50), B = 30 at (12,50), nothing between them: both are peaks, B survives O2
    # (no common neighbour reaches 30 - 4).  Ungated each window holds both: Q = 130.
    cells = [(10, 50, 100), (12, 50, 30)]
    u = _run(cells, False)
    assert [int(c["q_tot"]) for c in u] == [130, 130]
    _expect(u[0], 130, +60, 0, 120, 0, 10, 50)      # Sp = 30 * (+2), Spp = 30 * 4
    _expect(u[1], 130, -200, 0, 400, 0, 12, 50)     # Sp = 100 * (-2)
    # Gated: (11,50) is empty, so neither window takes the other's charge.
    g = _run(cells, True)
    _expect(g[0], 100, 0, 0, 0, 0, 10, 50)
    _expect(g[1], 30, 0, 0, 0, 0, 12, 50)


def test_bridge_cell_opens_the_gate():
    # same, with 5 ADC (below thr_peak, not a peak) on the bridge cell (11,50): the gate is open,
    # A's window is 100 + 5 + 30.  B is now suppressed?  common neighbour (11,50): 5 + 4 >= 30 is false -> no.
    cells = [(10, 50, 100), (11, 50, 5), (12, 50, 30)]
    g = _run(cells, True)
    assert len(g) == 2
    _expect(g[0], 135, 5 + 60, 0, 5 + 120, 0, 10, 50)
    _expect(g[1], 135, -5 - 200, 0, 5 + 400, 0, 12, 50)
    assert g.tobytes() == _run(cells, False).tobytes()


def test_diagonal_and_knight_use_the_diagonal_inner_cell():
    # peak 100 at (10,50); outer cells: diagonal (12,52) = 8, knight (12,51) = 9, knight (9,52) = 7.
    # Inner cells: (11,51) for the first two, (9,51)?? no: clamp(dp=-1, dt=2) -> (9,51).
    base = [(10, 50, 100), (12, 52, 4), (12, 51, 5), (9, 52, 3)]       # outer cells below thr: no extra peaks
    g = _run(base, True)
    assert len(g) == 1
    _expect(g[0], 100, 0, 0, 0, 0, 10, 50)                              # all three gates closed
    g = _run(base + [(11, 51, 3)], True)                                 # opens (12,52) and (12,51), not (9,52)
    # cells in: 100 (0,0); 3 (dp 1, dt 1); 4 (2,2); 5 (2,1)
    _expect(g[0], 112, 3 + 8 + 10, 3 + 8 + 5, 3 + 16 + 20, 3 + 16 + 5, 10, 50)
    g = _run(base + [(9, 51, 3)], True)                                  # opens (9,52) only
    _expect(g[0], 106, -3 - 3, 3 + 6, 3 + 3, 3 + 12, 10, 50)


def test_gate_at_the_map_edge():
    # peak at pad 1: the outer column dp = -2 is outside the map (weight 0 by Q8), dp = +2 is gated as usual
    g = _run([(1, 50, 60), (3, 50, 4)], True)
    _expect(g[0], 60, 0, 0, 0, 0, 1, 50)
    assert int(g[0]["flags"]) & 1
    g = _run([(1, 50, 60), (2, 50, 3), (3, 50, 4)], True)
    _expect(g[0], 67, 3 + 8, 0, 3 + 16, 0, 1, 50)


def test_identity_when_inner_ring_is_full():
    # Appendix A2 (symmetric cross, every inner cell > 0): gating changes nothing
    cells = [(30, 80, 100)] + [(30 + dp, 80 + dt, 50) for dp, dt in ((1, 0), (-1, 0), (0, 1), (0, -1))] + \
        [(30 + dp, 80 + dt, 25) for dp in (-1, 1) for dt in (-1, 1)] + \
        [(30 + dp, 80 + dt, 10) for dp, dt in ((2, 0), (-2, 0), (0, 2), (0, -2))]
    assert _run(cells, True).tobytes() == _run(cells, False).tobytes()


def test_t0_equals_t1_gated_random_maps():
    rng = np.random.default_rng(2511)
    alpha = np.array([0, 3, 5, 7, 9, 12, 40, 1023])
    for shape in ((7, 8), (9, 9)):
        for _ in range(300):
            Tm, Pm = shape
            q = alpha[rng.integers(1, len(alpha), size=shape)] * (rng.random(shape) < rng.uniform(0.15, 0.9))
            rows = [(0, 0, p, t, int(q[t, p])) for t in range(Tm) for p in range(Pm) if q[t, p]]
            d = t1.make_digits(rows)
            a, st, n = t1.clusterize(d, 1, 1, Tm, [Pm], 6, 4, cog_gated=True)
            b, bad = t0.clusterize(rows, 1, 1, Tm, [Pm], 6, 4, cog_gated=True)
            assert n == len(b)
            for x, y in zip(a, b):
                for k in ("q_tot", "q_max", "time_peak", "pad_peak", "flags"):
                    assert int(x[k]) == int(y[k]), k
                for k in ("pad_mean", "time_mean", "sigma_pad", "sigma_time"):
                    assert _bits(x[k]) == _bits(y[k]), k
            # gating only ever removes charge, and never from the 3x3 core
            u, _, _ = t1.clusterize(d, 1, 1, Tm, [Pm], 6, 4)
            assert len(u) == n and (a["q_tot"] <= u["q_tot"]).all() and (a["q_max"] == u["q_max"]).all()
