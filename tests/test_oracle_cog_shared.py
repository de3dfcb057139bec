"""Pins of reading Q10'' (R8, second half): charge sharing between
clusters whose 5x5 windows overlap.  Partners of a survivor c = the survivors at Chebyshev distance
exactly 2; a cell of c's window that a partner's window also holds is split with the integer weights
w_p(x) = (q_p >> 2 cheb(p, x)) + 1, c taking floor(q_x w_c / sum w); peak cells are never split (a
cluster keeps its own in full and takes nothing of a partner's).  Hand vectors with every share
and sum worked out by hand (the artefact of SURVEY.md Appendix A7 "axis, one ADC lower" is the
first), finalised by exact rational arithmetic (exact_f32); T0 (sets and dicts) against T1 (C) on
random maps; the identity with Q10 when no survivor has a partner; and what the rule promises:
two partners alone share a cell without losing more than one ADC count of it."""
import numpy as np

from exact_f32 import finalize_exact
from oracle import t0_bruteforce as t0
from oracle import t1

P, T = 40, 120


def _run(cells, shared=True):
    d = t1.make_digits([(0, 0, p, t, q) for (p, t, q) in cells])
    cl, st, n = t1.clusterize(d, 1, 1, T, [P], 6, 4, cog_shared=shared)
    assert st == 0 and n == len(cl)
    return cl


def _bits(x):
    return int(np.array(x, dtype=np.float32).view(np.uint32))


def _expect(c, Q, Sp, St, Spp, Stt, p_c, t_c):
    e = finalize_exact(Q, Sp, St, Spp, Stt, p_c, t_c)
    assert int(c["q_tot"]) == Q and (int(c["pad_peak"]), int(c["time_peak"])) == (p_c, t_c)
    assert [_bits(c[k]) for k in ("pad_mean", "time_mean", "sigma_pad", "sigma_time")] == e


def test_appendix_a7_axis_one_adc_lower():
    # A = 100 at (10,50), bridge 25 at (11,50), B = 30 at (12,50): both survive O2 (25 + 4 < 30) and under
    # Q10 both windows hold the same three cells: q_tot 155 twice, B's mean sits on A.
    cells = [(10, 50, 100), (11, 50, 25), (12, 50, 30)]
    u = _run(cells, shared=False)
    assert [int(c["q_tot"]) for c in u] == [155, 155]
    # Q10'': the peak cells stay whole; the bridge is at distance 1 from both: w_A = (100 >> 2) + 1 = 26,
    # w_B = (30 >> 2) + 1 = 8  ->  A takes 25*26/34 = 19, B takes 25*8/34 = 5 (one count is lost to the floors)
    g = _run(cells)
    assert len(g) == 2
    _expect(g[0], 100 + 19, 19 * 1, 0, 19 * 1, 0, 10, 50)
    _expect(g[1], 30 + 5, 5 * -1, 0, 5 * 1, 0, 12, 50)
    assert abs(float(g[1]["pad_mean"]) - 12.0) < 0.25 < abs(float(u[1]["pad_mean"]) - 12.0)   # the artefact is gone
    assert int(g[0]["q_max"]) == 100 and int(g[1]["q_max"]) == 30                   # q_max is the cell, not the share


def test_diagonal_partners_and_private_cells():
    # A = 80 at (10,50), B = 40 at (12,52) (diagonal, distance 2); the common cell (11,51) holds 18
    # (no ridge: 18 + 4 < 40); private cells: 20 at (9,49) (distance 3 from B: A's alone), 12 at (13,53).
    cells = [(10, 50, 80), (12, 52, 40), (11, 51, 18), (9, 49, 20), (13, 53, 12)]
    g = _run(cells)
    assert len(g) == 2
    # (11,51): d 1 from both: w_A = (80 >> 2) + 1 = 21, w_B = (40 >> 2) + 1 = 11 -> A 18*21/32 = 11, B 18*11/32 = 6
    _expect(g[0], 80 + 11 + 20, 11 - 20, 11 - 20, 11 + 20, 11 + 20, 10, 50)
    _expect(g[1], 40 + 6 + 12, -6 + 12, -6 + 12, 6 + 12, 6 + 12, 12, 52)


def test_three_survivors_in_a_row_share_pairwise_with_ring_partners_only():
    # 60 at pads 10, 12, 14 of one time bin, bridges of 20 at pads 11 and 13 (no ridge: 20 + 4 < 60): all
    # three survive.  The middle one has two partners, the outer ones one each: 10 and 14 are at distance 4
    # and NOT partners of each other.  w = (60 >> 2) + 1 = 16 at distance 1, (60 >> 4) + 1 = 4 at distance 2.
    cells = [(10, 50, 60), (11, 50, 20), (12, 50, 60), (13, 50, 20), (14, 50, 60)]
    g = _run(cells)
    assert len(g) == 3
    # pad 10's view: bridge 11 split with pad 12 only: 20*16/32 = 10; cell 12 is a partner's peak: 0;
    #   (bridge 13 and cell 14 are outside its window)
    _expect(g[0], 60 + 10, 10, 0, 10, 0, 10, 50)
    # pad 12's view: bridge 11 against pad 10 (d 1) -- pad 14 does not reach it (d 3): 20*16/32 = 10; same for 13
    _expect(g[1], 60 + 10 + 10, 0, 0, 20, 0, 12, 50)
    _expect(g[2], 60 + 10, -10, 0, 10, 0, 14, 50)
    # a cell in THREE windows: 5 (below thr_peak: no peak) at (12,48), two bins before the middle peak, d 2 from all
    g = _run(cells + [(12, 48, 5)])
    assert len(g) == 3
    #   from pad 10: partners {12}: 5*4/(4+4) = 2;  from pad 12: partners {10, 14}: 5*4/12 = 1;  from pad 14: 2
    _expect(g[0], 60 + 10 + 2, 10 + 2 * 2, 2 * -2, 10 + 2 * 4, 2 * 4, 10, 50)
    _expect(g[1], 60 + 20 + 1, 0, 1 * -2, 20, 1 * 4, 12, 50)
    _expect(g[2], 60 + 10 + 2, -10 + 2 * -2, 2 * -2, 10 + 2 * 4, 2 * 4, 14, 50)


def test_identity_without_partners_and_at_edges():
    # isolated clusters (no survivor within distance 2 of another): Q10'' == Q10 byte for byte
    cells = [(5, 10, 50), (6, 10, 20), (5, 11, 9), (20, 60, 200), (21, 61, 40), (19, 59, 7), (0, 0, 33), (39, 119, 44)]
    assert _run(cells).tobytes() == _run(cells, shared=False).tobytes()
    # partners across the clipped window at the pad edge
    g = _run([(0, 50, 100), (2, 50, 30)])
    assert len(g) == 2 and int(g[0]["flags"]) & 1
    _expect(g[0], 100, 0, 0, 0, 0, 0, 50)
    _expect(g[1], 30, 0, 0, 0, 0, 2, 50)


def test_two_partners_lose_at_most_one_count_per_shared_cell():
    rng = np.random.default_rng(7)
    for _ in range(200):
        qa, qb, qm = int(rng.integers(30, 1024)), int(rng.integers(30, 1024)), int(rng.integers(0, 20))
        cells = [(10, 50, qa), (12, 50, qb)] + ([(11, 50, qm)] if qm else [])
        g = _run(cells)
        if len(g) != 2:
            continue   # the smaller one was suppressed by the ridge
        tot = qa + qb + qm
        assert tot - 1 <= int(g[0]["q_tot"]) + int(g[1]["q_tot"]) <= tot
        assert int(g[0]["q_tot"]) >= qa and int(g[1]["q_tot"]) >= qb      # the peak cells stay whole


def test_t0_equals_t1_shared_random_maps():
    rng = np.random.default_rng(2512)
    alpha = np.array([0, 3, 5, 7, 9, 12, 40, 200, 1023])
    n_with_partners = 0
    for shape in ((7, 8), (9, 9), (6, 11)):
        for _ in range(300):
            Tm, Pm = shape
            q = alpha[rng.integers(1, len(alpha), size=shape)] * (rng.random(shape) < rng.uniform(0.1, 0.6))
            rows = [(0, 0, p, t, int(q[t, p])) for t in range(Tm) for p in range(Pm) if q[t, p]]
            d = t1.make_digits(rows)
            a, st, n = t1.clusterize(d, 1, 1, Tm, [Pm], 6, 4, cog_shared=True)
            b, bad = t0.clusterize(rows, 1, 1, Tm, [Pm], 6, 4, cog_shared=True)
            assert n == len(b)
            for x, y in zip(a, b):
                for k in ("q_tot", "q_max", "time_peak", "pad_peak", "flags"):
                    assert int(x[k]) == int(y[k]), k
                for k in ("pad_mean", "time_mean", "sigma_pad", "sigma_time"):
                    assert _bits(x[k]) == _bits(y[k]), k
            # sharing only ever removes charge from a window, never the peak cell's identity or the cluster set
            u, _, _ = t1.clusterize(d, 1, 1, Tm, [Pm], 6, 4)
            assert len(u) == n and (a["q_tot"] <= u["q_tot"]).all() and (a["q_max"] == u["q_max"]).all()
            n_with_partners += int((a["q_tot"] < u["q_tot"]).sum())
    assert n_with_partners > 200      # the random maps do exercise the rule
