"""O6 -- packed 16-byte cluster record and per-row index (DESIGN.md
section 3, reading R5).

TEST INFRASTRUCTURE, NOT PRODUCT (see ``oracle/__init__.py``).  The packed record is an
*encoding* of the 32-byte deterministic record, so the oracle is that encoding written out
field by field in plain numpy:

    time_fix        = rn(time_mean  * 256)                      24 bit
    pad_fix         = min(rn(pad_mean * 256), 65535)            16 bit
    sigma_pad_fix   = rn(sigma_pad  * 16384)                    16 bit   (sigma <= 2 -> <= 32768)
    sigma_time_fix  = rn(sigma_time * 16384)                    16 bit

``rn`` converts float32 to integer, round to nearest, ties to even; the multiplication by a
power of two is exact in float32, so every value is a pure function of the record's bits.
Sector and row are dropped from the record; the row index says where each (sector,row) starts
in the list, which is in (sector,row,time_peak,pad_peak) order (O5).

Pins (tests/test_oracle_pack16.py): hand-computed values for the Appendix A vectors A1, A3, A4,
a tie (x.5 -> even), the pad clamp, and the index on a hand-made list.
"""
from __future__ import annotations

import numpy as np

CLUSTER16 = np.dtype([("time_fix_pad_peak", "<u4"), ("pad_fix", "<u2"), ("time_peak", "<u2"), ("q_tot", "<u2"),
                      ("q_max_flags", "<u2"), ("sigma_pad_fix", "<u2"), ("sigma_time_fix", "<u2")])
assert CLUSTER16.itemsize == 16


def _rn(x32: np.ndarray, scale: float) -> np.ndarray:
    """float32 * 2^k (exact), then round to nearest even, as an integer array."""
    y = (x32.astype(np.float32) * np.float32(scale)).astype(np.float32)
    return np.rint(y.astype(np.float64)).astype(np.int64)   # rint: ties to even; float32 -> float64 is exact


def pack16(clusters: np.ndarray) -> np.ndarray:
    """32-byte records (oracle.t1.CLUSTER) -> 16-byte records, same order."""
    out = np.zeros(len(clusters), dtype=CLUSTER16)
    time_fix = _rn(clusters["time_mean"], 256.0)
    pad_fix = np.minimum(_rn(clusters["pad_mean"], 256.0), 65535)
    assert (time_fix >= 0).all() and (time_fix < (1 << 24)).all() and (pad_fix >= 0).all()
    out["time_fix_pad_peak"] = (time_fix | (clusters["pad_peak"].astype(np.int64) << 24)).astype(np.uint32)
    out["pad_fix"] = pad_fix.astype(np.uint16)
    out["time_peak"] = clusters["time_peak"]
    out["q_tot"] = clusters["q_tot"].astype(np.uint16)
    out["q_max_flags"] = (clusters["q_max"].astype(np.uint32) | (clusters["flags"].astype(np.uint32) << 10)).astype(np.uint16)
    out["sigma_pad_fix"] = _rn(clusters["sigma_pad"], 16384.0).astype(np.uint16)
    out["sigma_time_fix"] = _rn(clusters["sigma_time"], 16384.0).astype(np.uint16)
    return out


def row_index(clusters: np.ndarray, n_sectors: int, n_rows: int) -> np.ndarray:
    """index[s * n_rows + r] = number of clusters of all (sector,row) before (s,r); last = total."""
    idx = np.zeros(n_sectors * n_rows + 1, dtype=np.uint64)
    for c in clusters:                      # plain loop: the definition
        idx[int(c["sector"]) * n_rows + int(c["row"]) + 1] += 1
    return np.cumsum(idx).astype(np.uint64)
