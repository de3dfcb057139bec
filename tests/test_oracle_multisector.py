"""Pins the multi-sector / ragged-row bookkeeping of the T1 oracle (oracle/tpcclus_oracle.c,
`oracle_clusterize_ex`: the sector bucketing first/order/fill, `row_off[]` with unequal
`n_pads`, the `dbg_map` sector stride) to T0 (dict maps keyed by (sector,row), no offsets at
all) -- SURVEY.md 8(c) invariant I8 "row/sector independence", O0 and O5.

Every other CPU pin runs one sector with rows of equal width; a slip such as `n_pads[0]` for
`n_pads[d->row]`, a wrong sector stride or a mis-ordered bucket passes all of them and fails
here.  Also: the exhaustive 4^9 enumeration of 3x3 maps through T1 against O1's strict /
non-strict form (the T0 enumeration in test_oracle_bruteforce.py takes a stride)."""
import itertools

import numpy as np
import pytest

from exact_f32 import bits_of_float
from oracle import t0_bruteforce as t0
from oracle import t1

FLOATS = ("pad_mean", "time_mean", "sigma_pad", "sigma_time")
INTS = ("q_tot", "q_max", "time_peak", "pad_peak", "row", "sector", "flags", "reserved")


def _random_frame(rng, S, pads, T, dens, bad=False):
    """Seeded digits on a ragged multi-sector geometry: clustered in time so that peaks, ridges
    and ties occur; unique cells unless `bad` (then duplicates and out-of-range digits too)."""
    rows = []
    for s in range(S):
        for r, P in enumerate(pads):
            n = max(1, int(P * T * dens))
            cells = rng.choice(P * T, size=min(n, P * T), replace=False)
            for c in cells:
                q = int(rng.choice([3, 5, 6, 7, 9, 12, 40, 40, 200, 1023, 1500]))
                rows.append((s, r, int(c % P), int(c // P), q))
    if bad:
        R = len(pads)
        rows += [(S, 0, 0, 0, 50), (0, R, 0, 0, 50), (1, 1, pads[1], 3, 50), (2, 0, pads[0] + 1, 3, 50),
                 (1, 2, 0, T, 50), (0, 3, 1, 1, 0)]
        for k in range(20):   # duplicates of existing cells with another charge (Q5: the maximum wins)
            s, r, p, t, q = rows[int(rng.integers(0, len(rows) - 6))]
            rows.append((s, r, p, t, int(rng.integers(1, 1100))))
    order = rng.permutation(len(rows))
    return [rows[i] for i in order]


def _compare(rows, S, pads, T, thr=6, eps=4, gated=False):
    R = len(pads)
    exp, bad0 = t0.clusterize(rows, S, R, T, pads, thr, eps, cog_gated=gated)
    d = t1.make_digits(rows)
    got, st, cnt, m = t1.clusterize(d, S, R, T, pads, thr, eps, return_map=True, cog_gated=gated)
    assert cnt == len(got) == len(exp)
    assert bool(st & t1.STATUS_BAD_DIGITS) == bad0 and not (st & t1.STATUS_OVERFLOW)
    for g, e in zip(got, exp):   # O5 order and every field, bit for bit
        for k in INTS:
            assert int(g[k]) == int(e[k]), (k, e)
        for k in FLOATS:
            assert bits_of_float(float(g[k])) == bits_of_float(float(e[k])), (k, e)
    # O0: the dense map in [sector][row][time][pad] order against T0's dicts
    maps, _ = t0.build_maps(rows, S, R, T, pads)
    per_sector = T * int(sum(pads))
    assert m.shape == (S * per_sector,)
    ref = np.zeros_like(m)
    off = np.concatenate([[0], np.cumsum([T * p for p in pads])])
    for (s, r), cells in maps.items():
        for (t, p), q in cells.items():
            ref[s * per_sector + off[r] + t * pads[r] + p] = q
    assert np.array_equal(m, ref)
    return got


@pytest.mark.parametrize("seed", range(12))
def test_t0_equals_t1_on_ragged_multisector_frames(seed):
    rng = np.random.default_rng(1000 + seed)
    pads = [[5, 9, 7, 11], [11, 1, 6, 8], [3, 12, 12, 4]][seed % 3]
    T = [13, 9, 17][seed % 3]
    got = _compare(_random_frame(rng, 3, pads, T, dens=[0.25, 0.5, 0.8][(seed // 3) % 3]), 3, pads, T)
    assert len(got) > 0 and len({(int(c["sector"]), int(c["row"])) for c in got}) >= 6


@pytest.mark.parametrize("seed", range(4))
def test_t0_equals_t1_with_bad_digits_duplicates_and_readings(seed):
    rng = np.random.default_rng(2000 + seed)
    pads = [5, 9, 7, 11]
    rows = _random_frame(rng, 3, pads, 12, dens=0.4, bad=True)
    _compare(rows, 3, pads, 12, thr=[6, 1, 9, 6][seed], eps=[4, 0, 1023, 2][seed], gated=bool(seed & 1))


def test_sector_and_row_independence_of_t1():
    """I8 on the ragged geometry: one (sector,row) clusterized alone == its clusters inside the frame,
    and a sector's clusters do not depend on which other sectors are present."""
    rng = np.random.default_rng(7)
    pads = [5, 9, 7, 11]
    rows = _random_frame(rng, 3, pads, 15, dens=0.5)
    d = t1.make_digits(rows)
    full, _, _ = t1.clusterize(d, 3, 4, 15, pads)
    for s in range(3):
        for r in range(4):
            sub = d[(d["sector"] == s) & (d["row"] == r)]
            alone, _, _ = t1.clusterize(sub, 3, 4, 15, pads)
            assert alone.tobytes() == full[(full["sector"] == s) & (full["row"] == r)].tobytes()
    only1, _, _ = t1.clusterize(d[d["sector"] == 1], 3, 4, 15, pads)
    assert only1.tobytes() == full[full["sector"] == 1].tobytes()


def test_exhaustive_3x3_all_262144_maps_strict_nonstrict_form():
    """Every 3x3 map over {0,5,7,9} (4^9) through T1's O1, against the 'equivalent GPU form' of
    SURVEY.md 8(c) O1 evaluated for all maps at once with array shifts: strictly greater than the
    four neighbours earlier in (t,p) order, greater or equal to the four later ones."""
    alpha = np.array([0, 5, 7, 9], dtype=np.uint16)
    idx = np.array(list(itertools.product(range(4), repeat=9)), dtype=np.uint8)
    maps = alpha[idx].reshape(-1, 3, 3)
    z = np.zeros((len(maps), 5, 5), dtype=np.int64)
    z[:, 1:4, 1:4] = maps
    c = z[:, 1:4, 1:4]
    ok = c >= 6
    for dt, dp in ((-1, -1), (-1, 0), (-1, 1), (0, -1)):
        ok &= c > z[:, 1 + dt:4 + dt, 1 + dp:4 + dp]
    for dt, dp in ((0, 1), (1, -1), (1, 0), (1, 1)):
        ok &= c >= z[:, 1 + dt:4 + dt, 1 + dp:4 + dp]
    # one call: the maps stacked along time with two empty rows between them (rows never see each
    # other across an empty gap of 2 for O1; O2 is not compared here)
    tall = np.zeros((len(maps) * 5, 3), dtype=np.uint16)
    tall.reshape(len(maps), 5, 3)[:, :3, :] = maps
    f = t1.row_flags(tall, 6, 4).reshape(len(maps), 5, 3)[:, :3, :] & 1
    assert np.array_equal(f.astype(bool), ok)


def test_sector_parallel_driver_equals_single_call():
    """`t1.clusterize_by_sector` (the all-core baseline of bench.py and the full-frame GPU parity
    tests) is the single-threaded routine applied sector by sector: same bytes, any thread count."""
    from workloads import make_frame
    fr = make_frame(2, sectors=[0, 5, 35], n_time=200)
    d = fr.digits_numpy().view(t1.DIGIT)
    full, st, _ = t1.clusterize(d, fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads)
    assert st == 0 and len(full) > 1000
    for threads in (1, 3):
        tm = {}
        res = t1.clusterize_by_sector(lambda s: d[d["sector"] == s], [0, 5, 35], fr.n_rows, fr.n_time, fr.n_pads,
                                      threads=threads, timing=tm)
        assert np.concatenate([res[s] for s in (0, 5, 35)]).tobytes() == full.tobytes()
        assert tm["cores"] == threads and tm["digits"] == len(d)
