"""ctypes front end of the T1 oracle (``tpcclus_oracle.c``).

TEST INFRASTRUCTURE, NOT PRODUCT (see ``oracle/__init__.py``).  The record
dtypes below restate SURVEY.md 8(b); they are typed out here independently of
the CUDA package's binding.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import time

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tpcclus_oracle.c")
_LIB = os.path.join(_HERE, "liboracle_t1.so")

# 8-byte digit, 32-byte cluster (little-endian, natural alignment)
DIGIT = np.dtype(
    [("charge", "<u2"), ("time", "<u2"), ("pad", "u1"), ("row", "u1"), ("sector", "u1"), ("reserved", "u1")]
)
CLUSTER = np.dtype(
    [
        ("pad_mean", "<f4"), ("time_mean", "<f4"), ("sigma_pad", "<f4"), ("sigma_time", "<f4"),
        ("q_tot", "<u4"), ("q_max", "<u2"), ("time_peak", "<u2"),
        ("pad_peak", "u1"), ("row", "u1"), ("sector", "u1"), ("flags", "u1"),
        ("reserved", "<u4"),
    ]
)
assert DIGIT.itemsize == 8 and CLUSTER.itemsize == 32

STATUS_OVERFLOW = 1
STATUS_BAD_DIGITS = 2
FLAG_EDGE_PAD, FLAG_EDGE_TIME, FLAG_SATURATED = 1, 2, 4

# IEEE single precision, no contraction, no fast math.
CFLAGS = ["-O2", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared", "-std=c11"]


def build(force: bool = False) -> str:
    """Compile the C oracle next to its source (gcc). Returns the .so path."""
    if (not force) and os.path.exists(_LIB) and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC):
        return _LIB
    tmp = _LIB + ".tmp%d" % os.getpid()
    subprocess.check_call(["gcc", *CFLAGS, "-o", tmp, _SRC, "-lm"])
    os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.oracle_clusterize.restype = ctypes.c_int64
        _lib.oracle_clusterize.argtypes = [
            ctypes.c_uint32, ctypes.c_uint32, ctypes.c_uint32, ctypes.c_void_p,
            ctypes.c_uint32, ctypes.c_uint32, ctypes.c_void_p, ctypes.c_uint64,
            ctypes.c_void_p, ctypes.c_uint64, ctypes.c_void_p, ctypes.c_void_p,
        ]
        _lib.oracle_clusterize_ex.restype = ctypes.c_int64
        _lib.oracle_clusterize_ex.argtypes = _lib.oracle_clusterize.argtypes + [ctypes.c_int]
        _lib.oracle_finalize.restype = None
        _lib.oracle_finalize.argtypes = [
            ctypes.c_uint32, ctypes.c_int32, ctypes.c_int32, ctypes.c_uint32, ctypes.c_uint32,
            ctypes.c_uint32, ctypes.c_uint32, ctypes.c_void_p,
        ]
        _lib.oracle_row_flags.restype = None
        _lib.oracle_row_flags.argtypes = [
            ctypes.c_uint32, ctypes.c_uint32, ctypes.c_void_p, ctypes.c_uint32, ctypes.c_uint32,
            ctypes.c_void_p,
        ]
        assert _lib.oracle_sizeof_digit() == 8 and _lib.oracle_sizeof_cluster() == 32
    return _lib


def clusterize(digits, n_sectors, n_rows, n_time, n_pads, thr_peak=6, noise_eps=4,
               capacity=None, return_map=False, timing=None, cog_gated=False, cog_shared=False):
    """Run O0..O5.  ``digits``: array of dtype DIGIT (or uint64 / (n,8) uint8 view).

    Returns ``(clusters[DIGIT->CLUSTER array], status)`` (+ the O0 map if
    ``return_map``).  ``timing``, if a dict, receives ``seconds`` spent inside
    the C call only.
    """
    d = np.ascontiguousarray(digits)
    if d.dtype != DIGIT:
        d = d.view(np.uint8).reshape(-1).view(DIGIT)
    n = d.shape[0]
    pads = np.ascontiguousarray(np.asarray(n_pads, dtype=np.uint16))
    assert pads.shape == (n_rows,)
    if capacity is None:
        capacity = max(n, 1)
    out = np.zeros(capacity, dtype=CLUSTER)
    status = ctypes.c_uint32(0)
    dbg = None
    if return_map:
        dbg = np.zeros(int(n_sectors) * int(n_time) * int(pads.astype(np.int64).sum()), dtype=np.uint16)
    t0 = time.perf_counter()
    cnt = lib().oracle_clusterize_ex(
        n_sectors, n_rows, n_time, pads.ctypes.data, thr_peak, noise_eps,
        d.ctypes.data, n, out.ctypes.data, capacity, ctypes.byref(status),
        dbg.ctypes.data if dbg is not None else None, 2 if cog_shared else (1 if cog_gated else 0),
    )
    if timing is not None:
        timing["seconds"] = time.perf_counter() - t0
    if cnt < 0:
        raise MemoryError("oracle_clusterize: allocation failed")
    res = out[: min(cnt, capacity)]
    if return_map:
        return res, status.value, int(cnt), dbg
    return res, status.value, int(cnt)


def finalize(Q, Sp, St, Spp, Stt, p_c, t_c):
    """O4 only: returns float32[4] = pad_mean, time_mean, sigma_pad, sigma_time."""
    out = np.zeros(4, dtype=np.float32)
    lib().oracle_finalize(Q, Sp, St, Spp, Stt, p_c, t_c, out.ctypes.data)
    return out


def row_flags(q, thr_peak=6, noise_eps=4):
    """O1/O2 flags of one [T][P] row map: bit0 peak, bit1 survivor."""
    q = np.ascontiguousarray(q, dtype=np.uint16)
    T, P = q.shape
    f = np.zeros((T, P), dtype=np.uint8)
    lib().oracle_row_flags(T, P, q.ctypes.data, thr_peak, noise_eps, f.ctypes.data)
    return f


def make_digits(rows):
    """Helper for tests: list of (sector,row,pad,time,charge) -> DIGIT array."""
    d = np.zeros(len(rows), dtype=DIGIT)
    for i, (s, r, p, t, q) in enumerate(rows):
        d[i] = (q, t, p, r, s, 0)
    return d


def clusterize_by_sector(digits_of, sectors, n_rows, n_time, n_pads, thr_peak=6, noise_eps=4, threads=None,
                         timing=None, cog_gated=False, cog_shared=False):
    """T1 run sector-parallel ("the same T1 code run sector-parallel ... on all host
    cores"): sectors never interact (O0, invariant I8 -- pinned in tests/test_oracle_multisector.py),
    so each sector is clusterized alone by the unchanged single-threaded C routine as a 1-sector
    geometry and gets its sector number put back.  ctypes releases the GIL, so plain threads do.

    ``digits_of(s)`` returns the DIGIT (or uint64) array of sector ``s`` (any order; the sector
    field is overwritten on a copy).  Returns ``{s: clusters}``; ``timing`` receives ``seconds``
    (wall time of the clusterize calls only), ``cores`` (threads used) and ``digits``."""
    import os
    from concurrent.futures import ThreadPoolExecutor

    sectors = list(sectors)
    if threads is None:
        threads = len(os.sched_getaffinity(0))
    threads = max(1, min(int(threads), len(sectors)))
    lib()   # build / load once, outside the threads
    inputs = {}
    for s in sectors:
        d = np.array(digits_of(s), copy=True)
        if d.dtype != DIGIT:
            d = d.view(np.uint8).reshape(-1).view(DIGIT)
        d["sector"] = 0
        inputs[s] = d

    def one(s):
        d = inputs[s]
        cl, st, cnt = clusterize(d, 1, n_rows, n_time, n_pads, thr_peak, noise_eps,
                                 capacity=max(len(d) // 4, 1024), cog_gated=cog_gated, cog_shared=cog_shared)
        if cnt != len(cl) or st != 0:
            raise RuntimeError("oracle: sector %d: status %d, %d clusters for capacity %d" % (s, st, cnt, len(cl)))
        cl["sector"] = s
        return s, cl

    t0 = time.perf_counter()
    if threads == 1:
        res = dict(one(s) for s in sectors)
    else:
        with ThreadPoolExecutor(max_workers=threads) as ex:
            res = dict(ex.map(one, sectors))
    if timing is not None:
        timing["seconds"] = time.perf_counter() - t0
        timing["cores"] = threads
        timing["digits"] = int(sum(len(d) for d in inputs.values()))
    return res
