"""Pins the oracle (T1 C and T0 Python) to the worked vectors of SURVEY.md
Appendix A (tests/golden/appendix_a.json) and to exact rational arithmetic."""
import json
import os

import numpy as np
import pytest

from exact_f32 import bits_of_float, finalize_exact
from oracle import t0_bruteforce as t0
from oracle import t1

G = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "appendix_a.json")))
P, T = G["n_pads"], G["n_time"]
FLOATS = ("pad_mean", "time_mean", "sigma_pad", "sigma_time")
INTS = ("pad_peak", "time_peak", "q_max", "q_tot", "flags")


def _run_t1(case):
    d = t1.make_digits([(0, 0, p, t, q) for (p, t, q) in case["digits"]])
    cl, st, cnt = t1.clusterize(d, 1, 1, T, [P], G["thr_peak"], G["noise_eps"])
    assert st == 0 and cnt == len(cl)
    return cl


@pytest.mark.parametrize("case", G["cases"], ids=[c["name"] for c in G["cases"]])
def test_t1_matches_appendix_a(case):
    cl = _run_t1(case)
    assert len(cl) == len(case["clusters"])
    for got, exp in zip(cl, case["clusters"]):
        for k in INTS:
            if k in exp:
                assert int(got[k]) == exp[k], k
        for k in FLOATS:
            if k in exp:
                assert bits_of_float(float(got[k])) == int(exp[k], 16), (k, float(got[k]))
        assert got["row"] == 0 and got["sector"] == 0 and got["reserved"] == 0


@pytest.mark.parametrize("case", G["cases"], ids=[c["name"] for c in G["cases"]])
def test_t0_matches_appendix_a(case):
    # T0 ranks every cell of the map, so it gets a map just large enough for the vector: the full pad
    # width and the time range up to the last digit + 8 (no cluster of these vectors sits on the far
    # time edge, so the EDGE_TIME flag and the clipped windows are those of the full 14256-bin map).
    T0 = min(T, max(64, max(t for _, t, _ in case["digits"]) + 8))
    cl, bad = t0.clusterize([(0, 0, p, t, q) for p, t, q in case["digits"]], 1, 1, T0, [P],
                            G["thr_peak"], G["noise_eps"])
    assert not bad and len(cl) == len(case["clusters"])
    for got, exp in zip(cl, case["clusters"]):
        for k in INTS:
            if k in exp:
                assert int(got[k]) == exp[k], k
        for k in FLOATS:
            if k in exp:
                assert bits_of_float(float(got[k])) == int(exp[k], 16), k


@pytest.mark.parametrize("case", [c for c in G["cases"] if "o1_peaks" in c],
                         ids=[c["name"] for c in G["cases"] if "o1_peaks" in c])
def test_o1_peak_sets(case):
    q = np.zeros((64, 32), dtype=np.uint16)
    for p, t, c in case["digits"]:
        q[t, p] = c
    for flags in (t1.row_flags(q, G["thr_peak"], G["noise_eps"]), t0.row_flags(q, G["thr_peak"], G["noise_eps"])):
        peaks = sorted((int(p), int(t)) for t, p in zip(*np.nonzero(flags & 1)))
        assert peaks == sorted(tuple(x) for x in case["o1_peaks"])
        surv = sorted((int(p), int(t)) for t, p in zip(*np.nonzero(flags & 2)))
        assert surv == sorted((c["pad_peak"], c["time_peak"]) for c in case["clusters"])


@pytest.mark.parametrize("case", [c for c in G["cases"] if "sums" in c],
                         ids=[c["name"] for c in G["cases"] if "sums" in c])
def test_sums_and_exact_rounding(case):
    """The printed integer sums reproduce the printed float32 patterns under exact
    real arithmetic rounded once per operation -- independent of any float library."""
    s = case["sums"]
    assert s["Vp"] == s["Q"] * s["Spp"] - s["Sp"] ** 2 and s["Vt"] == s["Q"] * s["Stt"] - s["St"] ** 2
    # sums recomputed from the digit list by brute force around the printed peak
    c = case["clusters"][0]
    Q = Sp = St = Spp = Stt = 0
    for p, t, q in case["digits"]:
        dp, dt = p - c["pad_peak"], t - c["time_peak"]
        assert abs(dp) <= 2 and abs(dt) <= 2
        Q += q; Sp += q * dp; St += q * dt; Spp += q * dp * dp; Stt += q * dt * dt
    assert (Q, Sp, St, Spp, Stt) == (s["Q"], s["Sp"], s["St"], s["Spp"], s["Stt"])
    bits = finalize_exact(Q, Sp, St, Spp, Stt, c["pad_peak"], c["time_peak"])
    assert bits == [int(c[k], 16) for k in FLOATS]
    got = t1.finalize(Q, Sp, St, Spp, Stt, c["pad_peak"], c["time_peak"])
    assert [bits_of_float(float(x)) for x in got] == bits


@pytest.mark.parametrize("v", G["finalize_only"], ids=[v["name"] for v in G["finalize_only"]])
def test_finalize_only(v):
    assert v["V"] == v["Q"] * v["Spp"] - v["Sp"] ** 2 and v["V"] >= 1 << 24
    exp = [int(v[k], 16) for k in FLOATS]
    assert finalize_exact(v["Q"], v["Sp"], v["St"], v["Spp"], v["Stt"], v["p_c"], v["t_c"]) == exp
    got = t1.finalize(v["Q"], v["Sp"], v["St"], v["Spp"], v["Stt"], v["p_c"], v["t_c"])
    assert [bits_of_float(float(x)) for x in got] == exp


def test_finalize_exact_random_sums():
    """O4 of T1 == correctly rounded exact arithmetic on random admissible sums
    (catches a fused multiply-add, a double-rounded divide, a wrong operand)."""
    rng = np.random.default_rng(7)
    for _ in range(300):
        q = rng.integers(0, 1024, size=(5, 5))
        q[2, 2] = max(q[2, 2], 1)
        dt, dp = np.meshgrid(np.arange(-2, 3), np.arange(-2, 3), indexing="ij")
        Q, Sp, St = int(q.sum()), int((q * dp).sum()), int((q * dt).sum())
        Spp, Stt = int((q * dp * dp).sum()), int((q * dt * dt).sum())
        p_c, t_c = int(rng.integers(0, 138)), int(rng.integers(0, 14256))
        got = t1.finalize(Q, Sp, St, Spp, Stt, p_c, t_c)
        assert [bits_of_float(float(x)) for x in got] == finalize_exact(Q, Sp, St, Spp, Stt, p_c, t_c)


def test_duplicates_bad_digits_and_clamp():
    """O0 / Q4 / Q5: max wins in either order, out-of-range ignored + flagged, >1023 clamped, 0 ignored."""
    for order in ((7, 9), (9, 7)):
        d = t1.make_digits([(0, 0, 5, 5, order[0]), (0, 0, 5, 5, order[1])])
        cl, st, cnt, m = t1.clusterize(d, 1, 1, 16, [16], return_map=True)
        assert m.reshape(16, 16)[5, 5] == 9 and m.sum() == 9 and cnt == 1 and cl[0]["q_tot"] == 9
    d = t1.make_digits([(0, 0, 5, 5, 2000), (0, 0, 8, 8, 0), (1, 0, 1, 1, 50), (0, 1, 1, 1, 50),
                        (0, 0, 16, 1, 50), (0, 0, 1, 16, 50)])
    cl, st, cnt, m = t1.clusterize(d, 1, 1, 16, [16], return_map=True)
    assert st == t1.STATUS_BAD_DIGITS and cnt == 1
    assert cl[0]["q_max"] == 1023 and cl[0]["flags"] & t1.FLAG_SATURATED and m.sum() == 1023


def test_overflow_reports_true_count():
    d = t1.make_digits([(0, 0, 2, 2, 50), (0, 0, 10, 10, 60), (0, 0, 2, 12, 70)])
    cl, st, cnt = t1.clusterize(d, 1, 1, 16, [16], capacity=2)
    assert cnt == 3 and st & t1.STATUS_OVERFLOW and len(cl) == 2
