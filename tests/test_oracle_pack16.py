"""Pins of the packed-record oracle (oracle/pack16.py) against values worked out by hand from
the printed float32 values of SURVEY.md Appendix A -- not by calling the packer's own formula."""
import numpy as np

from oracle import t1
from oracle.pack16 import CLUSTER16, pack16, row_index


def _rec(pad_mean, time_mean, sp, st, q_tot=100, q_max=50, time_peak=0, pad_peak=0, row=0, sector=0, flags=0):
    c = np.zeros(1, dtype=t1.CLUSTER)
    c["pad_mean"], c["time_mean"], c["sigma_pad"], c["sigma_time"] = pad_mean, time_mean, sp, st
    c["q_tot"], c["q_max"], c["time_peak"], c["pad_peak"], c["row"], c["sector"], c["flags"] = \
        q_tot, q_max, time_peak, pad_peak, row, sector, flags
    return c


def test_hand_values_appendix_a():
    # A1: pad 10.0, time 100.0, sigmas 0 -> 2560, 25600, 0, 0
    p = pack16(_rec(10.0, 100.0, 0.0, 0.0, q_tot=50, q_max=50, time_peak=100, pad_peak=10))[0]
    assert (int(p["time_fix_pad_peak"]) & 0xFFFFFF, int(p["time_fix_pad_peak"]) >> 24) == (25600, 10)
    assert (p["pad_fix"], p["time_peak"], p["q_tot"], p["q_max_flags"], p["sigma_pad_fix"], p["sigma_time_fix"]) == \
        (2560, 100, 50, 50, 0, 0)
    # A3: plateaus, means x.5 and sigma exactly 0.5 -> 10.5*256 = 2688, 100.5*256 = 25728, 0.5*16384 = 8192
    p = pack16(_rec(10.5, 100.5, 0.5, 0.5))[0]
    assert (p["pad_fix"], int(p["time_fix_pad_peak"]) & 0xFFFFFF, p["sigma_pad_fix"], p["sigma_time_fix"]) == (2688, 25728, 8192, 8192)
    # A4 (bit patterns printed in the survey): pad_mean 0x41a1631c = 20.17339324951172 -> x256 = 5164.3887 -> 5164
    # time_mean 0x447a0745 = 1000.1135864257812 -> x256 = 256029.078 -> 256029
    # sigma_pad 0x3f456d4e = 0.771199107170105 -> x16384 = 12635.326 -> 12635; sigma_time 0x3f26055d = 0.6485193371772766 -> 10625.34 -> 10625
    f = lambda h: np.array([h], dtype=np.uint32).view(np.float32)[0]
    p = pack16(_rec(f(0x41a1631c), f(0x447a0745), f(0x3f456d4e), f(0x3f26055d)))[0]
    assert (p["pad_fix"], int(p["time_fix_pad_peak"]) & 0xFFFFFF, p["sigma_pad_fix"], p["sigma_time_fix"]) == (5164, 256029, 12635, 10625)
    # A4 at t = 14000: 0x465ac074 = 14000.11328125 -> x256 = 3584029.0 exactly
    p = pack16(_rec(f(0x43022c63), f(0x465ac074), 0.0, 0.0))[0]
    assert int(p["time_fix_pad_peak"]) & 0xFFFFFF == 3584029
    assert p["pad_fix"] == 33324        # 130.1733856201172 * 256 = 33324.387


def test_ties_to_even_clamp_and_flags():
    # 10 + 1/512 and 10 + 3/512 are exact in float32: x256 = 2560.5 -> 2560 (even), 2561.5 -> 2562 (even)
    assert pack16(_rec(10.0 + 1.0 / 512, 0.0, 0.0, 0.0))[0]["pad_fix"] == 2560
    assert pack16(_rec(10.0 + 3.0 / 512, 0.0, 0.0, 0.0))[0]["pad_fix"] == 2562
    # pad_mean 255.999 -> 65535.74 -> 65536 -> clamped to 65535
    assert pack16(_rec(255.999, 0.0, 0.0, 0.0))[0]["pad_fix"] == 65535
    # largest sigma (A5): 1.4142135381698608 * 16384 = 23170.47 -> 23170
    assert pack16(_rec(0.0, 0.0, 1.4142135381698608, 2.0))[0]["sigma_pad_fix"] == 23170
    assert pack16(_rec(0.0, 0.0, 1.0, 2.0))[0]["sigma_time_fix"] == 32768
    p = pack16(_rec(0.0, 0.0, 0.0, 0.0, q_tot=25575, q_max=1023, flags=7, time_peak=14255, pad_peak=137))[0]
    assert p["q_tot"] == 25575 and p["q_max_flags"] == (1023 | (7 << 10)) and p["time_peak"] == 14255
    assert int(p["time_fix_pad_peak"]) >> 24 == 137


def test_row_index_by_hand():
    cl = np.concatenate([_rec(0, 0, 0, 0, sector=0, row=1), _rec(0, 0, 0, 0, sector=0, row=1), _rec(0, 0, 0, 0, sector=1, row=0),
                         _rec(0, 0, 0, 0, sector=1, row=2)])
    assert row_index(cl, 2, 3).tolist() == [0, 0, 2, 2, 3, 3, 4]
    assert row_index(cl[:0], 2, 3).tolist() == [0] * 7


def test_consistency_on_a_frame():
    """On CFG[1]: the packed list keeps order and count, the index brackets exactly the clusters of
    each pad row, and unpacked means stay within half a unit of the float values."""
    from workloads import make_frame
    fr = make_frame(1)
    cl, st, n = t1.clusterize(fr.digits_numpy().view(t1.DIGIT), fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads)
    p = pack16(cl)
    idx = row_index(cl, fr.n_sectors, fr.n_rows)
    assert len(p) == n and idx[-1] == n and p.dtype == CLUSTER16
    for r in range(fr.n_rows):
        seg = cl[int(idx[r]):int(idx[r + 1])]
        assert (seg["row"] == r).all()
    assert np.abs((p["time_fix_pad_peak"] & 0xFFFFFF) / 256.0 - cl["time_mean"]).max() <= 0.5 / 256 + 1e-6
    assert np.abs(p["pad_fix"] / 256.0 - cl["pad_mean"]).max() <= 0.5 / 256 + 1e-6
    assert np.abs(p["sigma_pad_fix"] / 16384.0 - cl["sigma_pad"]).max() <= 0.5 / 16384 + 1e-7
