"""Invariants I1..I11 of SURVEY.md 8(c) on the T1 oracle, on CFG[0] and CFG[1] frames and
on hand-built maps (NS: symmetric injected clusters, charge conservation, no two surviving
peaks in a 3x3 window, invariance under digit permutation)."""
import numpy as np
import pytest

from oracle import t1
from workloads import make_frame

KEYS = ("sector", "row", "time_peak", "pad_peak")


@pytest.fixture(scope="module", params=[0, 1])
def frame_and_clusters(request):
    fr = make_frame(request.param, keep_truth=True)
    d = fr.digits_numpy().view(t1.DIGIT)
    cl, st, cnt = t1.clusterize(d, fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads)
    assert st == 0 and cnt == len(cl)
    return fr, d, cl


def _key(cl):
    return (cl["sector"].astype(np.int64) << 32) | (cl["row"].astype(np.int64) << 24) | \
           (cl["time_peak"].astype(np.int64) << 8) | cl["pad_peak"].astype(np.int64)


def test_i1_no_two_clusters_adjacent(frame_and_clusters):
    fr, d, cl = frame_and_clusters
    occ = {}
    for c in cl:
        occ.setdefault((int(c["sector"]), int(c["row"])), set()).add((int(c["time_peak"]), int(c["pad_peak"])))
    for cells in occ.values():
        for (t, p) in cells:
            for dt in (-1, 0, 1):
                for dp in (-1, 0, 1):
                    assert (dt, dp) == (0, 0) or (t + dt, p + dp) not in cells


def test_i2_cluster_iff_cell_above_threshold(frame_and_clusters):
    fr, d, cl = frame_and_clusters
    has = {(int(s), int(r)) for s, r in zip(d["sector"][d["charge"] >= 6], d["row"][d["charge"] >= 6])}
    got = {(int(c["sector"]), int(c["row"])) for c in cl}
    assert has == got


def test_i4_permutation_invariance(frame_and_clusters):
    fr, d, cl = frame_and_clusters
    rng = np.random.default_rng(3)
    for _ in range(3):
        cl2, st, cnt = t1.clusterize(d[rng.permutation(len(d))], fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads)
        assert cl2.tobytes() == cl.tobytes()
    cl3, _, _ = t1.clusterize(np.sort(d.view(np.uint64)).view(t1.DIGIT), fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads)
    assert cl3.tobytes() == cl.tobytes()


def test_i5_i6_i7_i11(frame_and_clusters):
    fr, d, cl = frame_and_clusters
    dig = {(int(x["sector"]), int(x["row"]), int(x["time"]), int(x["pad"])): int(x["charge"]) for x in d}
    for c in cl:   # I5: every cluster sits on an input digit of charge q_max >= thr
        q = dig[(int(c["sector"]), int(c["row"]), int(c["time_peak"]), int(c["pad_peak"]))]
        assert q == int(c["q_max"]) >= 6
    k = _key(cl)
    assert np.all(np.diff(k) > 0)                                   # I6 strictly increasing keys
    assert np.all(np.abs(cl["pad_mean"] - cl["pad_peak"]) <= 2) and np.all(np.abs(cl["time_mean"] - cl["time_peak"]) <= 2)
    for s in ("sigma_pad", "sigma_time"):
        assert np.all(cl[s] >= 0) and np.all(cl[s] <= 2)
    assert np.all(cl["q_max"] <= cl["q_tot"]) and np.all(cl["q_tot"] <= 25575) and np.all(cl["reserved"] == 0)
    assert len(cl) <= int((d["charge"] >= 6).sum())                 # I11


def test_i8_row_independence(frame_and_clusters):
    fr, d, cl = frame_and_clusters
    for r in (0, fr.n_rows // 2, fr.n_rows - 1):
        sub = d[d["row"] == r]
        cr, _, _ = t1.clusterize(sub, fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads)
        assert cr.tobytes() == cl[cl["row"] == r].tobytes()


def test_i9_below_threshold_gives_nothing(frame_and_clusters):
    fr, d, cl = frame_and_clusters
    low = d[d["charge"] < 6]
    cr, st, cnt = t1.clusterize(low, fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads)
    assert cnt == 0 and st == 0
    # and a threshold above every charge
    cr, st, cnt = t1.clusterize(d, fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads, thr_peak=1024)
    assert cnt == 0


def test_i3_charge_conservation_isolated_clusters():
    """Isolated random blobs confined to the 5x5 window of their maximum: q_tot == sum of digits."""
    rng = np.random.default_rng(11)
    rows, sums = [], {}
    for i in range(40):
        t0, p0 = 10 + 12 * (i // 5), 6 + 12 * (i % 5)
        blob = rng.integers(0, 60, size=(5, 5))
        blob[2, 2] = 200 + i                       # unique maximum at the centre
        for dt in range(5):
            for dp in range(5):
                if blob[dt, dp]:
                    rows.append((0, 0, p0 + dp - 2, t0 + dt - 2, int(blob[dt, dp])))
        sums[(t0, p0)] = int(blob.sum())
    d = t1.make_digits(rows)
    # eps = 0 and a high threshold so minor bumps inside a blob do not become clusters of their own
    cl, st, cnt = t1.clusterize(d, 1, 1, 128, [72], thr_peak=200, noise_eps=0)
    assert cnt == 40
    for c in cl:
        assert int(c["q_tot"]) == sums[(int(c["time_peak"]), int(c["pad_peak"]))]


def test_symmetric_injected_clusters_give_integer_cog():
    """NS: exact integer CoG of symmetric injected clusters -- any pattern symmetric under
    (dp,dt)->(-dp,-dt) has mean == peak cell bit-for-bit."""
    rng = np.random.default_rng(12)
    rows = []
    centres = [(20 + 10 * i, 7 + 9 * (i % 6)) for i in range(30)]
    for (t0, p0) in centres:
        h = rng.integers(1, 80, size=(5, 5))
        sym = h + h[::-1, ::-1]
        sym[2, 2] = 500
        for dt in range(5):
            for dp in range(5):
                rows.append((0, 0, p0 + dp - 2, t0 + dt - 2, int(sym[dt, dp])))
    cl, st, cnt = t1.clusterize(t1.make_digits(rows), 1, 1, 400, [64], thr_peak=400, noise_eps=0)
    assert cnt == 30
    for c, (t0, p0) in zip(cl, centres):
        assert float(c["pad_mean"]) == float(p0) and float(c["time_mean"]) == float(t0)
        assert c["sigma_pad"] > 0 and c["sigma_time"] > 0


def test_axis_swap_and_sign_are_detected():
    """A cluster skewed to +pad only / +time only must move only that mean, upward."""
    d = t1.make_digits([(0, 0, 10, 50, 100), (0, 0, 11, 50, 40)])
    c = t1.clusterize(d, 1, 1, 100, [32])[0][0]
    assert c["pad_mean"] > 10 and c["time_mean"] == 50.0 and c["sigma_time"] == 0 and c["sigma_pad"] > 0
    d = t1.make_digits([(0, 0, 10, 50, 100), (0, 0, 10, 49, 40)])
    c = t1.clusterize(d, 1, 1, 100, [32])[0][0]
    assert c["time_mean"] < 50 and c["pad_mean"] == 10.0 and c["sigma_pad"] == 0 and c["sigma_time"] > 0


def test_i10_translation():
    rng = np.random.default_rng(13)
    blob = rng.integers(0, 90, size=(7, 7))
    blob[3, 3] = 300
    def run(t0, p0):
        rows = [(0, 0, p0 + dp - 3, t0 + dt - 3, int(blob[dt, dp])) for dt in range(7) for dp in range(7) if blob[dt, dp]]
        return t1.clusterize(t1.make_digits(rows), 1, 1, 14256, [138])[0]
    a, b = run(100, 20), run(100 + 9000, 20 + 77)
    assert len(a) == len(b) >= 1
    for x, y in zip(a, b):
        assert int(y["time_peak"]) - int(x["time_peak"]) == 9000 and int(y["pad_peak"]) - int(x["pad_peak"]) == 77
        for k in ("q_tot", "q_max", "flags"):
            assert x[k] == y[k]
        assert x["sigma_pad"] == y["sigma_pad"] and x["sigma_time"] == y["sigma_time"]
        assert abs(float(y["pad_mean"]) - float(x["pad_mean"]) - 77) <= 2 ** -16 * 2
        assert abs(float(y["time_mean"]) - float(x["time_mean"]) - 9000) <= 2 ** -10 * 1.01


def test_generator_truth_cfg0():
    """Sanity (not parity): clusters found on CFG[0] sit on the injected centres -- residual
    mean ~ 0 and RMS well below a bin; catches an axis swap or sign error shared by both sides."""
    fr = make_frame(0, keep_truth=True)
    tr = fr.meta["truth"]
    d = fr.digits_numpy().view(t1.DIGIT)
    cl, _, _ = t1.clusterize(d, fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads)
    amp = tr["amp"].numpy()
    sel = amp > 30
    rp, rt = [], []
    for r, p0, t0 in zip(tr["row"].numpy()[sel], tr["p0"].numpy()[sel], tr["t0"].numpy()[sel]):
        if not (3 < p0 < 92 and 3 < t0 < 508):
            continue
        c = cl[cl["row"] == r]
        if len(c) == 0:
            continue
        dist = np.hypot(c["pad_mean"] - p0, c["time_mean"] - t0)
        j = int(np.argmin(dist))
        if dist[j] < 1.5:
            rp.append(float(c["pad_mean"][j]) - p0)
            rt.append(float(c["time_mean"][j]) - t0)
    rp, rt = np.array(rp), np.array(rt)
    assert len(rp) > 0.8 * sel.sum() * 0.85
    assert abs(rp.mean()) < 0.05 and abs(rt.mean()) < 0.05
    assert rp.std() < 0.35 and rt.std() < 0.35
