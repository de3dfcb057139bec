"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element
on the same seeded digits.  Bar (NS / DESIGN.md): DETERMINISTIC = byte-identical cluster
array (set, order, every field); FAST = identical cluster set after sorting by key,
integer fields exact, float fields within 1e-4 absolute (in fact bit-equal, Q14)."""
import json
import os

import numpy as np
import pytest

from oracle import t1
from workloads import make_frame, n_pads_ramp

pytestmark = pytest.mark.gpu

FLOATS = ("pad_mean", "time_mean", "sigma_pad", "sigma_time")
INTS = ("q_tot", "q_max", "time_peak", "pad_peak", "row", "sector", "flags", "reserved")


@pytest.fixture(scope="module")
def tp(cuda_device):
    import paper_2511_17018_b200 as tp
    tp.lib()   # fails loudly if the extension is missing
    return tp


def _key(cl):
    return (cl["sector"].astype(np.int64) << 32) | (cl["row"].astype(np.int64) << 24) | \
           (cl["time_peak"].astype(np.int64) << 8) | cl["pad_peak"].astype(np.int64)


def _oracle(d_np, S, R, T, pads, thr=6, eps=4):
    cl, st, cnt = t1.clusterize(d_np.view(t1.DIGIT), S, R, T, pads, thr, eps)
    assert cnt == len(cl)
    return cl, st


def _check_fast(got, exp):
    assert len(got) == len(exp)
    g = got[np.argsort(_key(got), kind="stable")]
    assert np.array_equal(_key(g), _key(exp))           # identical cluster set
    for k in INTS:
        assert np.array_equal(g[k], exp[k]), k
    for k in FLOATS:
        assert np.all(np.abs(g[k].astype(np.float64) - exp[k].astype(np.float64)) <= 1e-4), k


def _run_both(tp, digits_t, S, R, T, pads, thr=6, eps=4, rtc=False, max_digits=None):
    import torch
    c = tp.Clusterizer(S, R, T, pads, max_digits or max(1, digits_t.numel()), thr, eps, rtc=rtc)
    det, n_det, st_det = c.run_sync(digits_t, tp.MODE_DETERMINISTIC)
    fast, n_fast, st_fast = c.run_sync(digits_t, tp.MODE_FAST)
    c.close()
    assert n_det == len(det) and n_fast == len(fast) and st_det == st_fast
    return det, fast, st_det


def _digits_tensor(d_np, device):
    import torch
    return torch.from_numpy(np.ascontiguousarray(d_np).view(np.int64).copy()).to(device)


@pytest.mark.parametrize("k", [1, 0])
def test_cfg_small_det_and_fast(tp, cuda_device, k):
    fr = make_frame(k)
    d_np = fr.digits_numpy()
    exp, st = _oracle(d_np, fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads)
    det, fast, st_gpu = _run_both(tp, fr.digits.to(cuda_device), fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads)
    assert st_gpu == st == 0
    assert det.tobytes() == exp.tobytes()               # deterministic mode: bitwise
    _check_fast(fast, exp)
    assert fast[np.argsort(_key(fast))].tobytes() == exp.tobytes()   # Q14: fast values are bit-equal too


@pytest.mark.parametrize("k", [1, 0, 4])
def test_dense_map_step_a1(tp, cuda_device, k):
    """Step a1 (digit -> charge map) in isolation: the tiles the kernels build equal O0's map.
    k = 4: a ragged multi-sector slice of the Pb-Pb-like frame (sectors 0, 7, 35 of 36, all 152 row
    widths, three tiles per row with a ragged last slab)."""
    fr = make_frame(k) if k < 2 else make_frame(k, device=cuda_device, sectors=[0, 7, 35], n_time=300)
    _, _, _, m = t1.clusterize(fr.digits_numpy().view(t1.DIGIT), fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads,
                               return_map=True)
    c = tp.Clusterizer(fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads, fr.n_digits)
    c.run_sync(fr.digits.to(cuda_device), tp.MODE_FAST)
    got = c.dense_map().cpu().numpy().view(np.uint16)
    c.close()
    assert np.array_equal(got, m)


def test_appendix_a_vectors_on_gpu(tp, cuda_device):
    G = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "appendix_a.json")))
    P, T = G["n_pads"], G["n_time"]
    c = tp.Clusterizer(1, 1, T, [P], 64, G["thr_peak"], G["noise_eps"])
    for case in G["cases"]:
        d = t1.make_digits([(0, 0, p, t, q) for (p, t, q) in case["digits"]])
        got, n, st = c.run_sync(_digits_tensor(d, cuda_device), tp.MODE_DETERMINISTIC)
        assert st == 0 and n == len(case["clusters"]), case["name"]
        for g, e in zip(got, case["clusters"]):
            for k2 in ("pad_peak", "time_peak", "q_max", "q_tot", "flags"):
                if k2 in e:
                    assert int(g[k2]) == e[k2], (case["name"], k2)
            for k2 in FLOATS:
                if k2 in e:
                    assert int(np.array(g[k2]).view(np.uint32)) == int(e[k2], 16), (case["name"], k2)
    c.close()


def test_permutation_and_repeat_invariance(tp, cuda_device):
    """I4 / I14 / PAPER.md 47-48: det output is one byte string under any digit order and across runs."""
    import torch
    fr = make_frame(1)
    d = fr.digits.to(cuda_device)
    c = tp.Clusterizer(fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads, fr.n_digits)
    ref = c.run_sync(d, tp.MODE_DETERMINISTIC)[0].tobytes()
    g = torch.Generator(device="cpu").manual_seed(1)
    for i in range(8):
        perm = torch.randperm(d.numel(), generator=g).to(cuda_device)
        assert c.run_sync(d[perm].contiguous(), tp.MODE_DETERMINISTIC)[0].tobytes() == ref
    assert c.run_sync(torch.sort(d)[0], tp.MODE_DETERMINISTIC)[0].tobytes() == ref
    for i in range(5):
        assert c.run_sync(d, tp.MODE_DETERMINISTIC)[0].tobytes() == ref
    c.close()


def test_edge_inputs(tp, cuda_device):
    import torch
    pads = [16] * 4
    c = tp.Clusterizer(2, 4, 300, pads, 64)
    # empty input
    cl, n, st = c.run_sync(torch.zeros(0, dtype=torch.int64, device=cuda_device), tp.MODE_DETERMINISTIC)
    assert n == 0 and st == 0 and len(cl) == 0
    cl, n, st = c.run_sync(torch.zeros(0, dtype=torch.int64, device=cuda_device), tp.MODE_FAST)
    assert n == 0 and st == 0
    # duplicates (Q5: max wins in det mode, either order), clamp, zero charge, out-of-range
    rows = [(0, 0, 5, 5, 7), (0, 0, 5, 5, 9), (1, 3, 15, 299, 2000), (1, 3, 8, 8, 0),
            (2, 0, 1, 1, 50), (0, 4, 1, 1, 50), (0, 0, 16, 1, 50), (0, 0, 1, 300, 50)]
    for order in (rows, rows[::-1]):
        d = t1.make_digits(order)
        exp, st_exp = _oracle(d, 2, 4, 300, pads)
        got, n, st = c.run_sync(_digits_tensor(d, cuda_device), tp.MODE_DETERMINISTIC)
        assert st == st_exp == tp.STATUS_BAD_DIGITS and got.tobytes() == exp.tobytes() and n == 2
        assert got[0]["q_tot"] == 9 and got[1]["q_max"] == 1023 and got[1]["flags"] == 7
    # overflow: true count is returned, first `capacity` clusters in order (det)
    d = t1.make_digits([(0, 0, 2, 2 + 10 * i, 50 + i) for i in range(20)])
    exp, _ = _oracle(d, 2, 4, 300, pads)
    got, n, st = c.run_sync(_digits_tensor(d, cuda_device), tp.MODE_DETERMINISTIC, capacity=7)
    assert n == 20 and st == tp.STATUS_OVERFLOW and got.tobytes() == exp[:7].tobytes()
    got, n, st = c.run_sync(_digits_tensor(d, cuda_device), tp.MODE_FAST, capacity=7)
    assert n == 20 and st == tp.STATUS_OVERFLOW
    c.close()


def test_idempotent_between_different_inputs(tp, cuda_device):
    """Q17: output never depends on an earlier run (stale workspace contents)."""
    a, b = make_frame(1), make_frame(1, seed=99)
    c = tp.Clusterizer(a.n_sectors, a.n_rows, a.n_time, a.n_pads, max(a.n_digits, b.n_digits))
    ra = c.run_sync(a.digits.to(cuda_device), tp.MODE_DETERMINISTIC)[0].tobytes()
    rb = c.run_sync(b.digits.to(cuda_device), tp.MODE_DETERMINISTIC)[0].tobytes()
    assert c.run_sync(a.digits.to(cuda_device), tp.MODE_DETERMINISTIC)[0].tobytes() == ra and ra != rb
    exp, _ = _oracle(b.digits_numpy(), b.n_sectors, b.n_rows, b.n_time, b.n_pads)
    assert rb == exp.tobytes()
    c.close()


def test_thresholds_follow_params(tp, cuda_device):
    """Constant buffers may change between time frames (PAPER.md 79): two handles with different
    thresholds in one process each follow their own parameters."""
    fr = make_frame(1)
    d = fr.digits.to(cuda_device)
    c1 = tp.Clusterizer(fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads, fr.n_digits, thr_peak=6, noise_eps=4)
    c2 = tp.Clusterizer(fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads, fr.n_digits, thr_peak=20, noise_eps=0)
    for c, thr, eps in ((c1, 6, 4), (c2, 20, 0), (c1, 6, 4)):
        exp, _ = _oracle(fr.digits_numpy(), fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads, thr, eps)
        assert c.run_sync(d, tp.MODE_DETERMINISTIC)[0].tobytes() == exp.tobytes()
    c1.close(); c2.close()


def test_rtc_equals_generic(tp, cuda_device):
    """I13 / PAPER.md 91: the run-time-compiled variant changes speed only, never results."""
    fr = make_frame(1)
    exp, _ = _oracle(fr.digits_numpy(), fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads)
    det, fast, st = _run_both(tp, fr.digits.to(cuda_device), fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads, rtc=True)
    assert det.tobytes() == exp.tobytes() and st == 0
    _check_fast(fast, exp)


def test_multi_time_chunk_geometry(tp, cuda_device):
    """n_time > 16256 exercises the coarse time-chunk halo copies of K1 (n_tc = 3), with clusters
    planted across both chunk borders and random digits elsewhere."""
    rng = np.random.default_rng(17)
    T, pads = 40000, [24, 40]
    rows = []
    for tb in (16256, 32512):
        for dt in range(-6, 7):
            for r in (0, 1):
                rows.append((0, r, 10 + (dt % 5), tb + dt, int(rng.integers(3, 200))))
                rows.append((0, r, 3, tb + dt, 60))
    n = 20000
    t = rng.integers(0, T, n); r = rng.integers(0, 2, n); p = rng.integers(0, 24, n); q = rng.integers(1, 120, n)
    seen = {(x[1], x[2], x[3]) for x in rows}
    for i in range(n):
        key = (int(r[i]), int(p[i]), int(t[i]))
        if key not in seen:
            seen.add(key)
            rows.append((0, key[0], key[1], key[2], int(q[i])))
    d = t1.make_digits(rows)
    d = d[rng.permutation(len(d))]
    exp, st_exp = _oracle(d, 1, 2, T, pads)
    det, fast, st = _run_both(tp, _digits_tensor(d, cuda_device), 1, 2, T, pads)
    assert st == st_exp == 0 and det.tobytes() == exp.tobytes()
    _check_fast(fast, exp)


def test_dense_adversarial_tile(tp, cuda_device):
    """Maximum sizes: a fully occupied 138-pad row over 600 time bins with heavy ties (values 5..9),
    plus a checkerboard (the densest possible peak pattern) -- stresses the peak list bound,
    tie-breaking and the rank-by-bitmask emission."""
    rng = np.random.default_rng(23)
    T, P = 600, 138
    q = rng.integers(5, 10, size=(T, P))
    cb = np.zeros((T, P), dtype=np.int64)
    cb[::2, ::2] = 50
    rows = [(0, 0, p, t, int(q[t, p])) for t in range(T) for p in range(P)]
    rows += [(0, 1, p, t, 50) for t in range(0, T, 2) for p in range(0, P, 2)]
    d = t1.make_digits(rows)
    d = d[rng.permutation(len(d))]
    exp, _ = _oracle(d, 1, 2, T, [P, P])
    det, fast, st = _run_both(tp, _digits_tensor(d, cuda_device), 1, 2, T, [P, P])
    assert st == 0 and det.tobytes() == exp.tobytes()
    _check_fast(fast, exp)
    assert (exp["row"] == 1).sum() == (T // 2) * (P // 2)   # every checkerboard cell is its own cluster


def test_skewed_input_one_bin(tp, cuda_device):
    """All digits in one (sector,row): the write-combining stage of K1 overflows every round and
    the bin spans many K5 batches; results must not change."""
    rng = np.random.default_rng(29)
    T, P = 14256, 100
    n = 300000
    cell = rng.choice(T * P, size=n, replace=False)
    rows = np.zeros(n, dtype=t1.DIGIT)
    rows["time"], rows["pad"] = cell // P, cell % P
    rows["row"], rows["sector"] = 3, 1
    rows["charge"] = rng.integers(3, 300, n)
    exp, _ = _oracle(rows, 2, 5, T, [P] * 5)
    det, fast, st = _run_both(tp, _digits_tensor(rows, cuda_device), 2, 5, T, [P] * 5)
    assert st == 0 and det.tobytes() == exp.tobytes()
    _check_fast(fast, exp)


def test_run_host_e2e(tp, cuda_device):
    import torch
    fr = make_frame(0)
    exp, _ = _oracle(fr.digits_numpy(), fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads)
    c = tp.Clusterizer(fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads, fr.n_digits, host_capacity=fr.n_digits)
    dh = fr.digits.pin_memory()
    out = torch.empty((fr.n_digits, 32), dtype=torch.uint8).pin_memory()
    n, st = c.run_host(dh, out, tp.MODE_DETERMINISTIC)
    assert n == len(exp) and st == 0
    assert out[:n].numpy().tobytes() == exp.tobytes()
    n, st = c.run_host(dh, out, tp.MODE_FAST)
    got = out[:n].numpy().view(tp.CLUSTER_DTYPE).reshape(-1)
    _check_fast(got, exp)
    c.close()


def test_full_geometry_sector_slice(tp, cuda_device):
    """CFG[2]/CFG[4] recipe on the full 36x152 ramp geometry, cut to a short time window so the
    oracle finishes in seconds: several tiles per row, ragged last slab (T = 300), all row widths."""
    for k in (2, 4):
        fr = make_frame(k, device=cuda_device, sectors=[0, 7, 35], n_time=300)
        d_np = fr.digits_numpy()
        exp, _ = _oracle(d_np, fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads)
        det, fast, st = _run_both(tp, fr.digits, fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads)
        assert st == 0 and len(exp) > 1000
        assert det.tobytes() == exp.tobytes()
        _check_fast(fast, exp)


@pytest.mark.parametrize("k", [2, 3, 4])
def test_full_frame_complete_parity(tp, cuda_device, k):
    """BASELINE.json's full sizes in the launch configuration bench.py times (whole frame, shuffled,
    one handle): EVERY (sector,row) map of CFG[2], CFG[3] and CFG[4] -- all 5472 of each -- against
    the oracle, byte for byte (NS: "match the oracle bit-exactly ... on all five configs").  Sectors
    never interact (I8, pinned on the CPU in test_oracle_multisector.py), so the unchanged
    single-threaded T1 routine runs sector by sector on the host cores (`t1.clusterize_by_sector`).
    FAST: identical cluster set, every byte (Q14), after sorting by key."""
    import torch
    fr = make_frame(k, device=cuda_device)
    d = fr.digits
    n = fr.n_digits
    c = tp.Clusterizer(fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads, n)
    cap = n // 3 + 1024
    buf = torch.empty((cap, 32), dtype=torch.uint8, device=cuda_device)
    _, nt, st = c.run(d, tp.MODE_DETERMINISTIC, clusters=buf)
    torch.cuda.synchronize()
    n_det = int(nt.item())
    assert int(st.item()) == 0 and 0 < n_det <= cap and not c.det_fallback()
    det = buf[:n_det].clone()
    _, nt, st = c.run(d, tp.MODE_FAST, clusters=buf)
    torch.cuda.synchronize()
    assert int(nt.item()) == n_det and int(st.item()) == 0
    c.close()

    def key_of(t):   # bytes 20..27: q_max u16, time_peak u16, pad_peak u8, row u8, sector u8, flags u8
        w = t[:, 20:28].contiguous().view(torch.int64).reshape(-1)
        tpk, pad, row, sec = (w >> 16) & 0xFFFF, (w >> 32) & 0xFF, (w >> 40) & 0xFF, (w >> 48) & 0xFF
        return (sec << 32) | (row << 24) | (tpk << 8) | pad
    kd = key_of(det)
    assert bool((kd[1:] > kd[:-1]).all())                      # I6: unique keys, ascending
    fast = buf[:n_det]
    order = torch.argsort(key_of(fast))
    assert torch.equal(fast[order], det)                        # fast set == det set, every byte (Q14)
    del fast, order, buf

    # where each sector's clusters start in the ordered output
    bounds = torch.searchsorted(kd, torch.arange(fr.n_sectors + 1, device=cuda_device, dtype=torch.int64) << 32).tolist()
    dsec = (d >> 48) & 0xFF
    n_exp = 0
    group = max(1, min(len(os.sched_getaffinity(0)), 12))       # sectors in flight = host threads (1.5 GB each at T = 14256)
    for s0 in range(0, fr.n_sectors, group):
        secs = list(range(s0, min(s0 + group, fr.n_sectors)))
        host = {s: d[dsec == s].cpu().numpy().view(np.uint64) for s in secs}
        exp = t1.clusterize_by_sector(lambda s: host[s], secs, fr.n_rows, fr.n_time, fr.n_pads, threads=group)
        for s in secs:
            got = det[bounds[s]:bounds[s + 1]].cpu().numpy()
            assert len(exp[s]) > 0
            assert got.tobytes() == exp[s].tobytes(), (k, s)    # every cluster of the sector: order and all 32 bytes
            n_exp += len(exp[s])
        del host, exp
    assert n_exp == n_det


def test_det_fallback_when_run_buffer_is_too_small(tp, cuda_device):
    """DETERMINISTIC normally writes each tile's clusters as a run into a temporary buffer of
    max_digits / 8 clusters and orders the runs afterwards (K7-K9); a frame with more clusters
    than that (here: every digit is its own cluster) must take the chained-scan fallback and
    still be byte-identical to the oracle.  The usual frames must not take it."""
    T, P, R = 3000, 138, 4
    rows = np.zeros((R, T // 2, P // 2), dtype=t1.DIGIT)
    rows["time"] = (2 * np.arange(T // 2, dtype=np.uint16))[None, :, None]
    rows["pad"] = (2 * np.arange(P // 2, dtype=np.uint8))[None, None, :]
    rows["row"] = np.arange(R, dtype=np.uint8)[:, None, None]
    rows["charge"] = 50
    d = rows.reshape(-1)
    d = d[np.random.default_rng(31).permutation(len(d))]
    exp, _ = _oracle(d, 1, R, T, [P] * R)
    assert len(exp) == len(d)
    c = tp.Clusterizer(1, R, T, [P] * R, len(d))
    det, n, st = c.run_sync(_digits_tensor(d, cuda_device), tp.MODE_DETERMINISTIC)
    assert c.det_fallback() and st == 0 and n == len(exp)
    assert det.tobytes() == exp.tobytes()
    fast, n, st = c.run_sync(_digits_tensor(d, cuda_device), tp.MODE_FAST)
    _check_fast(fast, exp)
    c.close()
    # the same through the sparse-frame kernel (emitter warp): tiles of 32 isolated digits -- ranked inside one warp, their
    # runs cut from the CTA's block of the temporary buffer -- in so many tiles that the blocks run past the buffer's end
    T, P, R = 16000, 64, 40
    rows = np.zeros((R, T // 16, P // 16), dtype=t1.DIGIT)
    rows["time"] = (16 * np.arange(T // 16, dtype=np.uint16) + 5)[None, :, None]
    rows["pad"] = (16 * np.arange(P // 16, dtype=np.uint8) + 3)[None, None, :]
    rows["row"] = np.arange(R, dtype=np.uint8)[:, None, None]
    rows["charge"] = 50
    d = rows.reshape(-1)
    d = d[np.random.default_rng(37).permutation(len(d))]
    exp, _ = _oracle(d, 1, R, T, [P] * R)
    assert len(exp) == len(d) == 160000
    c = tp.Clusterizer(1, R, T, [P] * R, len(d))
    det, n, st = c.run_sync(_digits_tensor(d, cuda_device), tp.MODE_DETERMINISTIC)
    assert c.det_fallback() and st == 0 and n == len(exp)
    assert det.tobytes() == exp.tobytes()
    c.close()
    fr = make_frame(0)
    c = tp.Clusterizer(fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads, fr.n_digits)
    c.run_sync(fr.digits.to(cuda_device), tp.MODE_DETERMINISTIC)
    assert not c.det_fallback()
    c.close()


def test_order_and_build_invariance_at_scale(tp, cuda_device):
    """I4 / I13 / I14 on a full-geometry frame (CFG[2], 1.1e8 digits): the deterministic output is
    one byte string whatever the digit order (globally shuffled, readout-like, cell order),
    whichever build (generic __constant__ / NVRTC literals) and however often it is run."""
    import torch
    ref = None
    for order, rtc in (("shuffled", False), ("readout", False), ("cell", False), ("shuffled", True), ("shuffled", False)):
        fr = make_frame(2, device=cuda_device, order=order)
        c = tp.Clusterizer(fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads, fr.n_digits, rtc=rtc)
        buf = torch.empty((fr.n_digits // 3, 32), dtype=torch.uint8, device=cuda_device)
        _, nt, st = c.run(fr.digits, tp.MODE_DETERMINISTIC, clusters=buf)
        torch.cuda.synchronize()
        n = int(nt.item())
        assert int(st.item()) == 0 and not c.det_fallback()
        out = buf[:n].clone()
        c.close()
        del buf, fr
        if ref is None:
            ref = out
        else:
            assert out.shape == ref.shape and torch.equal(out, ref), (order, rtc)


def _rtc_child(cache_dir, q):
    import paper_2511_17018_b200 as tp
    import torch
    tp.tpcclus_set_rtc_cache_dir(cache_dir)
    fr = make_frame(1)
    c = tp.Clusterizer(fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads, fr.n_digits, rtc=True)
    det = c.run_sync(fr.digits.to("cuda:0"), tp.MODE_DETERMINISTIC)[0].tobytes()
    q.put((c.rtc_cache_hit, c.rtc_build_ms, det))
    c.close()


def test_rtc_cubin_cache(tp, cuda_device, tmp_path):
    """PAPER.md 97: processes of one node share a run-time compilation through a file lock.  Two
    processes started together on an empty cache: exactly one compiles, the other waits and loads;
    a third handle hits the cache outright; a different parameter set is a different key; results
    never change."""
    import multiprocessing as mp
    fr = make_frame(1)
    exp, _ = _oracle(fr.digits_numpy(), fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads)
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_rtc_child, args=(str(tmp_path), q)) for _ in range(2)]
    for p in ps:
        p.start()
    res = [q.get(timeout=300) for _ in ps]
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert sorted(r[0] for r in res) == [False, True]            # one compiled, one loaded
    assert all(r[2] == exp.tobytes() for r in res)
    assert len(list(tmp_path.glob("tpcclus_*.cubin"))) == 6      # one binary per compilation unit
    tp.tpcclus_set_rtc_cache_dir(str(tmp_path))
    try:
        c = tp.Clusterizer(fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads, fr.n_digits, rtc=True)
        assert c.rtc_cache_hit and c.rtc_build_ms < max(r[1] for r in res)
        assert c.run_sync(fr.digits.to(cuda_device), tp.MODE_DETERMINISTIC)[0].tobytes() == exp.tobytes()
        c.close()
        c = tp.Clusterizer(fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads, fr.n_digits, thr_peak=9, rtc=True)
        assert not c.rtc_cache_hit                                # thresholds are baked in: another key
        c.close()
        assert len(list(tmp_path.glob("tpcclus_*.cubin"))) == 12
    finally:
        tp.tpcclus_set_rtc_cache_dir(None)


def test_packed_output_and_row_index(tp, cuda_device):
    """the packed 16-byte records and the per-row index, byte for byte
    against the oracle's encoding of its own deterministic records."""
    import torch
    from oracle.pack16 import pack16, row_index
    for fr in (make_frame(1), make_frame(0), make_frame(4, device=cuda_device, sectors=[0, 7, 35], n_time=300)):
        exp, _ = _oracle(fr.digits_numpy(), fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads)
        c = tp.Clusterizer(fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads, fr.n_digits)
        cl, ridx, nt, st = c.run_packed(fr.digits.to(cuda_device))
        torch.cuda.synchronize()
        n = int(nt.item())
        assert n == len(exp) and int(st.item()) == 0
        assert cl[:n].cpu().numpy().tobytes() == pack16(exp).tobytes()
        assert ridx.cpu().numpy().astype(np.uint64).tolist() == row_index(exp, fr.n_sectors, fr.n_rows).tolist()
        # overflow: the first `capacity` stay in order, the index still describes the whole list
        cap = n // 2
        cl2, ridx2, nt, st = c.run_packed(fr.digits.to(cuda_device), capacity=cap)
        torch.cuda.synchronize()
        assert int(nt.item()) == n and int(st.item()) == tp.STATUS_OVERFLOW
        assert cl2.cpu().numpy().tobytes() == pack16(exp[:cap]).tobytes() and torch.equal(ridx2, ridx)
        # the 32-byte path of the same handle is unaffected
        assert c.run_sync(fr.digits.to(cuda_device), tp.MODE_DETERMINISTIC)[0].tobytes() == exp.tobytes()
        c.close()
    # more clusters than the run buffer holds: said loudly, nothing written
    T, P, R = 3000, 138, 4
    rows = np.zeros((R, T // 2, P // 2), dtype=t1.DIGIT)
    rows["time"] = (2 * np.arange(T // 2, dtype=np.uint16))[None, :, None]
    rows["pad"] = (2 * np.arange(P // 2, dtype=np.uint8))[None, None, :]
    rows["row"] = np.arange(R, dtype=np.uint8)[:, None, None]
    rows["charge"] = 50
    d = rows.reshape(-1)
    c = tp.Clusterizer(1, R, T, [P] * R, len(d))
    _, _, nt, st = c.run_packed(_digits_tensor(d, cuda_device))
    torch.cuda.synchronize()
    assert int(nt.item()) == len(d) and int(st.item()) == tp.STATUS_NO_PACKED
    c.close()


def test_cog_gated_reading(tp, cuda_device):
    """Reading Q10' (TPCCLUS_COG_GATED): outer-ring gating of the CoG window,
    byte for byte against the oracle in the same reading -- deterministic, fast, generic and RTC."""
    frames = [make_frame(1), make_frame(0), make_frame(4, device=cuda_device, sectors=[3, 20], n_time=300)]
    for fr in frames:
        d_np = fr.digits_numpy()
        exp, st, n = t1.clusterize(d_np.view(t1.DIGIT), fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads, cog_gated=True)
        plain, _ = _oracle(d_np, fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads)
        assert exp.tobytes() != plain.tobytes() and len(exp) == len(plain)      # the reading matters on these frames
        for rtc in (False, True):
            c = tp.Clusterizer(fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads, fr.n_digits, rtc=rtc, cog_gated=True)
            det = c.run_sync(fr.digits.to(cuda_device), tp.MODE_DETERMINISTIC)[0]
            fast = c.run_sync(fr.digits.to(cuda_device), tp.MODE_FAST)[0]
            c.close()
            assert det.tobytes() == exp.tobytes(), (fr.meta["name"], rtc)
            _check_fast(fast, exp)


def test_random_geometries_fuzz(tp, cuda_device):
    """Seeded fuzz over the parameter space the five configs do not span: odd sector/row counts,
    pad rows from 1 to 256 pads, time lengths around the tile and time-chunk borders, thresholds,
    duplicates and out-of-range digits.  Deterministic = byte-identical, fast = same set; status equal."""
    rng = np.random.default_rng(77)
    cases = [(1, 1, 1, [1]), (2, 3, 127, [1, 2, 256]), (3, 2, 128, [255, 7]), (1, 4, 129, [33, 64, 65, 250]),
             (2, 2, 262, [138, 66]), (1, 2, 16255, [20, 9]), (1, 1, 16257, [12]), (1, 1, 16262, [40]),
             (1, 1, 65536, [5]), (2, 1, 40000, [256]), (7, 5, 300, [17, 30, 1, 99, 140])]
    for (S, R, T, pads) in cases:
        for thr, eps, dens in ((6, 4, 0.25), (1, 0, 0.6), (40, 1023, 0.08)):
            cells = int(sum(pads)) * T * S
            n = max(1, min(int(cells * dens), 60000))
            d = np.zeros(n, dtype=t1.DIGIT)
            d["sector"] = rng.integers(0, S, n)
            d["row"] = rng.integers(0, R, n)
            d["pad"] = rng.integers(0, 256, n) % np.asarray(pads)[d["row"]]
            # cluster the digits in time so that peaks, ridges and ties actually occur
            d["time"] = (rng.integers(0, max(T // 8, 1), n) * 8 + rng.integers(0, 8, n)) % T
            d["charge"] = np.where(rng.random(n) < 0.3, rng.integers(1, 12, n), rng.integers(1, 1100, n))
            k = max(1, n // 50)                       # a few bad ones: pad, time, row, sector out of range; zero charge
            bad = rng.integers(0, n, k)
            d["pad"][bad[: k // 4]] = 255 if max(pads) < 256 else d["pad"][bad[: k // 4]]
            d["charge"][bad[k // 4: k // 2]] = 0
            if T < 65535:
                d["time"][bad[k // 2: 3 * k // 4]] = T   # (T = 65536 cannot be exceeded in 16 bits)
            d["row"][bad[3 * k // 4:]] = R
            exp, st_exp = _oracle(d, S, R, T, pads, thr, eps)
            det, _, st = _run_both(tp, _digits_tensor(d, cuda_device), S, R, T, pads, thr, eps)
            assert st == st_exp, (S, R, T, pads, thr, eps, st, st_exp)
            assert det.tobytes() == exp.tobytes(), (S, R, T, pads, thr, eps)    # duplicates: the maximum wins (Q5)
            # FAST promises the same set for duplicate-free input only (Q5): one digit per cell, the largest
            order = np.lexsort((-d["charge"].astype(np.int64), d["pad"], d["time"], d["row"], d["sector"]))
            ds = d[order]
            first = np.ones(len(ds), dtype=bool)
            first[1:] = (ds["pad"][1:] != ds["pad"][:-1]) | (ds["time"][1:] != ds["time"][:-1]) | \
                (ds["row"][1:] != ds["row"][:-1]) | (ds["sector"][1:] != ds["sector"][:-1])
            du = ds[first][rng.permutation(int(first.sum()))]
            exp_u, _ = _oracle(du, S, R, T, pads, thr, eps)
            assert exp_u.tobytes() == exp.tobytes()                               # the oracle agrees: max per cell
            _, fast, _ = _run_both(tp, _digits_tensor(du, cuda_device), S, R, T, pads, thr, eps)
            _check_fast(fast, exp)


def test_handle_reuse_sizes_and_geometries(tp, cuda_device):
    """One handle fed frames of very different sizes (large, small, empty, large again), capacity 1,
    and two generic handles of different geometry alternating on one stream (R6: one __constant__
    block, re-uploaded per run): every run equals the oracle, nothing leaks from run to run."""
    import torch
    big, small = make_frame(0), make_frame(0, seed=5, n_time=64)
    c = tp.Clusterizer(big.n_sectors, big.n_rows, big.n_time, big.n_pads, big.n_digits)
    sub = big.digits_numpy().view(t1.DIGIT)
    sub = sub[(sub["time"] < 40) & (sub["row"] < 3)]
    empty = torch.zeros(0, dtype=torch.int64, device=cuda_device)
    for d_np in (big.digits_numpy(), sub, None, big.digits_numpy()):
        if d_np is None:
            for mode in (tp.MODE_DETERMINISTIC, tp.MODE_FAST):
                cl, n, st = c.run_sync(empty, mode)
                assert n == 0 and st == 0 and len(cl) == 0
            continue
        exp, _ = _oracle(d_np, big.n_sectors, big.n_rows, big.n_time, big.n_pads)
        dt = _digits_tensor(np.ascontiguousarray(d_np).view(np.uint64), cuda_device)
        assert c.run_sync(dt, tp.MODE_DETERMINISTIC)[0].tobytes() == exp.tobytes()
        _check_fast(c.run_sync(dt, tp.MODE_FAST)[0], exp)
        # capacity 1: the count is still the true one, the overflow is flagged
        for mode in (tp.MODE_DETERMINISTIC, tp.MODE_FAST):
            cl, n, st = c.run_sync(dt, mode, capacity=1)
            assert n == len(exp) and (st == tp.STATUS_OVERFLOW) == (len(exp) > 1)
            if mode == tp.MODE_DETERMINISTIC:
                assert cl.tobytes() == exp[:1].tobytes()
    # a second handle with another geometry, alternating with the first on the same stream
    c2 = tp.Clusterizer(small.n_sectors, small.n_rows, small.n_time, small.n_pads, small.n_digits, thr_peak=9)
    exp_b, _ = _oracle(big.digits_numpy(), big.n_sectors, big.n_rows, big.n_time, big.n_pads)
    exp_s, _ = _oracle(small.digits_numpy(), small.n_sectors, small.n_rows, small.n_time, small.n_pads, 9, 4)
    db, ds = big.digits.to(cuda_device), small.digits.to(cuda_device)
    for _ in range(3):
        rb = c.run(db, tp.MODE_DETERMINISTIC)
        rs = c2.run(ds, tp.MODE_DETERMINISTIC)      # enqueued right behind, no sync in between
        torch.cuda.synchronize()
        assert rb[0][:int(rb[1].item())].cpu().numpy().tobytes() == exp_b.tobytes()
        assert rs[0][:int(rs[1].item())].cpu().numpy().tobytes() == exp_s.tobytes()
    c.close(); c2.close()


def test_sparse_dense_tile_alternation(tp, cuda_device):
    """K6 takes a tile with <= 256 staged records through the one-record-per-thread path, which
    undoes its own map writes instead of sweeping the map; larger tiles take the 16-byte-piece
    path, tiles above the staging capacity several rounds.  One CTA handles consecutive slabs of
    a bin, so every kind of tile here is followed by every other kind: record counts 0, 1 and
    every value around the 256 boundary, a few thousand, and > 4096 (multi-round), with
    duplicates on one cell (Q5), pads out of range (Q4) and records on the slab border rows that
    two tiles share.  A cell left behind by an undo or a missed sweep shows up as a phantom
    cluster or a wrong sum in the next tile."""
    rng = np.random.default_rng(83)
    P, n_slabs = 64, 330
    T = 128 * n_slabs            # 42240 bins = 3 coarse time-chunks
    counts = [0, 1, 2, 31, 32, 33, 64, 65, 128, 300, 1000, 3000, 4090, 4100, 5000] + list(range(236, 280))
    rows = []
    for r in (0, 1):
        order = rng.permutation(n_slabs)
        for i, sl in enumerate(order):
            n = counts[(i + 7 * r) % len(counts)]
            lo = 0 if i % 3 == 0 else 6          # every third slab also uses the border rows
            hi = 128 if i % 3 == 0 else 122
            cells = rng.choice((hi - lo) * P, size=n, replace=False)
            t = sl * 128 + lo + cells // P
            p = cells % P
            q = rng.integers(1, 400, n)
            rows += [(0, r, int(p[k]), int(t[k]), int(q[k])) for k in range(n)]
            if n and i % 4 == 0:   # duplicates of one cell with other charges, an out-of-range pad
                for k in range(min(n, 5)):
                    rows.append((0, r, int(p[k]), int(t[k]), int(rng.integers(1, 1023))))
                rows.append((0, r, P + 3, int(t[0]), 77))
    d = t1.make_digits(rows)
    exp, st_exp = _oracle(d, 1, 2, T, [P, P])
    assert st_exp != 0                       # the out-of-range pads are flagged
    # FAST promises the same set for duplicate-free input only (Q5): one digit per cell, the largest
    ds = d[np.lexsort((-d["charge"].astype(np.int64), d["pad"], d["time"], d["row"]))]
    first = np.ones(len(ds), dtype=bool)
    first[1:] = (ds["pad"][1:] != ds["pad"][:-1]) | (ds["time"][1:] != ds["time"][:-1]) | (ds["row"][1:] != ds["row"][:-1])
    du = ds[first]
    exp_u, _ = _oracle(du, 1, 2, T, [P, P])
    assert exp_u.tobytes() == exp.tobytes()
    for _ in range(2):
        dd = d[rng.permutation(len(d))]
        det, _, st = _run_both(tp, _digits_tensor(dd, cuda_device), 1, 2, T, [P, P])
        assert st == st_exp and det.tobytes() == exp.tobytes()
        dd = du[rng.permutation(len(du))]
        det, fast, st = _run_both(tp, _digits_tensor(dd, cuda_device), 1, 2, T, [P, P])
        assert st == st_exp and det.tobytes() == exp.tobytes()
        _check_fast(fast, exp)


def test_sparse_tiles_through_the_emitter_ring(tp, cuda_device):
    """FAST on a sparse frame: the clusters of a tile with <= 256 records leave through a 64-entry ring
    in shared memory to a warp of their own (k_cluster_tiles_fast_e).  Tiles of single-digit clusters on
    a 3 x 3 lattice -- up to 240 of them, every digit a surviving peak -- overrun the ring, so warps also
    take the fall-back (they emit themselves), the tags of the ring wrap many times, and tiles of 0, 1
    and a few clusters follow in between.  The set must be the oracle's, the count exact under
    overflow of the output, for the readings Q10 and Q10'.  The deterministic mode has the warp as well: there a
    tile with at most 32 peaks (the kinds with 1, 3 and 30 clusters) is ranked inside one warp and its run is cut
    from the block of the temporary buffer the CTA holds; the 30-cluster tiles overrun the ring in that mode too.
    Byte-equal to the oracle."""
    rng = np.random.default_rng(97)
    P, n_slabs = 100, 60
    T = 128 * n_slabs
    rows = []
    for r in (0, 1, 2):
        for sl in range(n_slabs):
            kind = (sl + r) % 7
            n = [240, 0, 3, 120, 30, 32, 33][kind] if sl else 1   # (32 / 33: either side of the one-warp limit of the deterministic path)
            lat = [(t, p) for t in range(1, 127, 3) for p in range(1, P - 1, 3)]   # 42 x 33 sites, pairwise distance >= 3
            for k in rng.choice(len(lat), size=n, replace=False):
                t, p = lat[k]
                rows.append((0, r, p, sl * 128 + t, int(rng.integers(6, 1023))))
                if kind == 2:   # a real 3 x 3 cluster around it
                    for dt, dp in ((0, 1), (1, 0), (-1, 0), (0, -1)):
                        rows.append((0, r, p + dp, sl * 128 + t + dt, 3))
    d = t1.make_digits(rows)
    d = d[rng.permutation(len(d))]
    pads = [P, P, P]
    assert len(d) < 512 * 3 * n_slabs        # the host picks the emitter kernel below this density
    for gated in (False, True):
        cl, st_exp, cnt = t1.clusterize(d.view(t1.DIGIT), 1, 3, T, pads, 6, 4, cog_gated=gated)
        c = tp.Clusterizer(1, 3, T, pads, len(d), 6, 4, cog_gated=gated)
        dt_ = _digits_tensor(d, cuda_device)
        for _ in range(3):
            fast, n, st = c.run_sync(dt_, tp.MODE_FAST)
            assert n == cnt == len(fast) and st == st_exp
            _check_fast(fast, cl)
        det, n, st = c.run_sync(dt_, tp.MODE_DETERMINISTIC)
        assert det.tobytes() == cl.tobytes()
        got, n, st = c.run_sync(dt_, tp.MODE_FAST, capacity=100)
        assert n == cnt and (st & tp.STATUS_OVERFLOW) and len(got) == 100
        keys = set(_key(cl).tolist())
        assert all(k in keys for k in _key(got).tolist()) and len(set(_key(got).tolist())) == 100
        c.close()


def test_more_bins_than_k1_has_stages_for(tp, cuda_device):
    """R1: K1 holds write-combining stages for 5503 coarse bins; a geometry with more is binned in several passes
    over the input, pass p staging the bins [p k, (p + 1) k).  (a) 40 x 152 maps (6080 bins, 2 passes); (b) 20 x 140
    maps over 16300 time bins = two coarse time-chunks (5600 bins, 2 passes), with clusters across the chunk border
    at t = 16256 whose halo copies go to a bin of the OTHER pass.  Both against the oracle, DET byte for byte and
    FAST as a set, generic and RTC build."""
    rng = np.random.default_rng(131)
    cases = []
    S, R, T, P = 40, 152, 300, 24
    n = 400_000
    rows = np.stack([rng.integers(0, S, n), rng.integers(0, R, n), rng.integers(0, P, n), rng.integers(0, T, n),
                     rng.integers(1, 200, n)], axis=1)
    cases.append((S, R, T, [P] * R, t1.make_digits([tuple(int(v) for v in r) for r in rows])))
    S, R, T, P = 20, 140, 16300, 12
    n = 300_000
    t = np.where(rng.random(n) < 0.5, rng.integers(16256 - 8, 16256 + 8, n), rng.integers(0, T, n))
    rows = np.stack([rng.integers(0, S, n), rng.integers(0, R, n), rng.integers(0, P, n), t, rng.integers(1, 200, n)], axis=1)
    cases.append((S, R, T, [P] * R, t1.make_digits([tuple(int(v) for v in r) for r in rows])))
    for S, R, T, pads, d in cases:
        # one digit per cell (FAST promises the oracle's set for duplicate-free input only, Q5)
        key = (d["sector"].astype(np.int64) << 40) | (d["row"].astype(np.int64) << 32) | (d["time"].astype(np.int64) << 8) | d["pad"]
        d = d[np.unique(key, return_index=True)[1]]
        d = d[rng.permutation(len(d))]
        exp, st_exp = _oracle(d, S, R, T, pads)
        assert len(exp) > 1000
        for rtc in (False, True):
            c = tp.Clusterizer(S, R, T, pads, len(d), 6, 4, rtc=rtc)
            assert c.launches_per_run(tp.MODE_FAST) == 8          # K1 twice
            dt_ = _digits_tensor(d, cuda_device)
            det, n_det, st = c.run_sync(dt_, tp.MODE_DETERMINISTIC)
            assert st == st_exp and det.tobytes() == exp.tobytes()
            fast, n_fast, st = c.run_sync(dt_, tp.MODE_FAST)
            assert st == st_exp
            _check_fast(fast, exp)
            c.close()


def test_run_under_cuda_graph_capture(tp, cuda_device):
    """tpcclus_run only enqueues kernel launches on the caller's stream -- no allocation, no synchronisation, no
    host-side read of device results -- so a caller can capture it into a CUDA graph and replay it (the launch-bound
    small frames gain a fifth).  Replays with new digits in the same input buffer must give that frame's clusters."""
    import torch
    fa, fb = make_frame(0), make_frame(0, seed=4242)
    n_max = max(fa.n_digits, fb.n_digits)
    # graph arguments are frozen: the capture takes the larger digit count, the shorter frame is padded with
    # all-zero digits (charge 0 at sector 0, row 0, pad 0, time 0: in range, ignored, Q4)
    buf = torch.zeros(n_max, dtype=torch.int64, device=cuda_device)
    c = tp.Clusterizer(fa.n_sectors, fa.n_rows, fa.n_time, fa.n_pads, n_max)
    out = torch.empty((n_max, 32), dtype=torch.uint8, device=cuda_device)
    for mode in (tp.MODE_DETERMINISTIC, tp.MODE_FAST):
        buf.zero_()
        buf[:fa.n_digits] = fa.digits.to(cuda_device)
        c.run(buf, mode, clusters=out)          # warm-up outside the capture (module loading is lazy)
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            _, n_t, st_t = c.run(buf, mode, clusters=out)
        for fr in (fa, fb, fa):
            buf.zero_()
            buf[:fr.n_digits] = fr.digits.to(cuda_device)
            out.zero_()
            g.replay()
            torch.cuda.synchronize()
            exp, st_exp = _oracle(fr.digits_numpy(), fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads)
            n = int(n_t.item())
            got = out[:n].cpu().numpy().view(tp.CLUSTER_DTYPE).reshape(-1)
            assert n == len(exp) and int(st_t.item()) == st_exp
            if mode == tp.MODE_DETERMINISTIC:
                assert got.tobytes() == exp.tobytes()
            else:
                _check_fast(got, exp)
        del g
    c.close()


def test_two_handles_two_streams_concurrently(tp, cuda_device):
    """Modules and constant blocks are per handle (R6, PAPER.md 81-85): two generic handles of
    different geometry AND thresholds run at the same time on two streams, many times over, and each
    follows its own parameters.  (With one process-wide __constant__ block, as in round 1, the second
    upload could land while the first handle's kernels were running.)"""
    import torch
    a = make_frame(0)                                  # 152 rows x 96 pads x 512
    b = make_frame(2, device=cuda_device, sectors=[0, 1], n_time=700)   # ragged full geometry, another pitch and bin count
    ca = tp.Clusterizer(a.n_sectors, a.n_rows, a.n_time, a.n_pads, a.n_digits, thr_peak=6, noise_eps=4)
    cb = tp.Clusterizer(b.n_sectors, b.n_rows, b.n_time, b.n_pads, b.n_digits, thr_peak=11, noise_eps=1)
    assert ca.constant_buffers == len(ca.loaded_units()) == 6 and "tiles_dump" not in ca.loaded_units()
    exp_a, _ = _oracle(a.digits_numpy(), a.n_sectors, a.n_rows, a.n_time, a.n_pads, 6, 4)
    exp_b, _ = _oracle(b.digits_numpy(), b.n_sectors, b.n_rows, b.n_time, b.n_pads, 11, 1)
    da, db = a.digits.to(cuda_device), b.digits.to(cuda_device)
    sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
    torch.cuda.synchronize()
    outs = []
    for i in range(6):
        with torch.cuda.stream(sa):
            ra = ca.run(da, tp.MODE_DETERMINISTIC if i % 2 else tp.MODE_FAST, stream=sa)
            ra = (ra[0].clone(), ra[1].clone(), ra[2].clone())
        with torch.cuda.stream(sb):
            rb = cb.run(db, tp.MODE_DETERMINISTIC, stream=sb)
            rb = (rb[0].clone(), rb[1].clone(), rb[2].clone())
        outs.append((i, ra, rb))
    torch.cuda.synchronize()
    for i, ra, rb in outs:
        assert int(ra[2].item()) == 0 and int(rb[2].item()) == 0
        ga = ra[0][:int(ra[1].item())].cpu().numpy().view(tp.CLUSTER_DTYPE).reshape(-1)
        gb = rb[0][:int(rb[1].item())].cpu().numpy().view(tp.CLUSTER_DTYPE).reshape(-1)
        assert gb.tobytes() == exp_b.tobytes()
        if i % 2:
            assert ga.tobytes() == exp_a.tobytes()
        else:
            _check_fast(ga, exp_a)
    ca.close(); cb.close()


def test_update_params_rewrites_every_constant_block(tp, cuda_device):
    """PAPER.md 79, 85: constant buffers may change between time frames and the framework rewrites all
    registered copies.  One handle, thresholds changed between runs on one stream without any host
    synchronisation: each run sees the values that were current when it was enqueued -- in every
    unit (K5/K6 read thr/eps, the dump unit is loaded later and must come up with the current values)."""
    import torch
    fr = make_frame(1)
    d = fr.digits.to(cuda_device)
    c = tp.Clusterizer(fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads, fr.n_digits)
    seq = [(6, 4), (20, 0), (3, 9), (6, 4)]
    res = []
    for thr, eps in seq:
        c.update_params(thr, eps)
        cl, n, st = c.run(d, tp.MODE_DETERMINISTIC)
        res.append((cl.clone(), n.clone(), st.clone()))
    torch.cuda.synchronize()
    for (thr, eps), (cl, n, st) in zip(seq, res):
        exp, _ = _oracle(fr.digits_numpy(), fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads, thr, eps)
        assert int(st.item()) == 0 and cl[:int(n.item())].cpu().numpy().tobytes() == exp.tobytes(), (thr, eps)
    assert res[0][0][:int(res[0][1].item())].cpu().numpy().tobytes() != res[1][0][:int(res[1][1].item())].cpu().numpy().tobytes()
    n0 = c.constant_buffers
    c.dense_map()                                    # brings the debug unit in: one more registered block
    assert c.constant_buffers == n0 + 1 and "tiles_dump" in c.loaded_units()
    with pytest.raises(tp.TpcclusError):
        c.update_params(0, 4)
    c.close()
    r = tp.Clusterizer(fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads, fr.n_digits, rtc=True)
    assert r.constant_buffers == 0                   # literals instead of constant memory (PAPER.md 89-91)
    with pytest.raises(tp.TpcclusError):
        r.update_params(7, 4)
    r.close()


def test_internal_status_bit_and_zero_charge_bad_pad(tp, cuda_device):
    """TPCCLUS_STATUS_INTERNAL (bit 31) is raised when a derived workspace capacity is exceeded -- it
    cannot be by construction, so the test hook shrinks the capacities: K1's slice, then K5's blob.
    And O0 tests a digit's range before its charge: a zero-charge digit with pad >= n_pads[row] is
    flagged BAD_DIGITS like the oracle does (it never reaches K5, where pads are checked otherwise)."""
    fr = make_frame(0)
    d = fr.digits.to(cuda_device)
    c = tp.Clusterizer(fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads, fr.n_digits)
    exp, _ = _oracle(fr.digits_numpy(), fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads)
    assert c.run_sync(d, tp.MODE_DETERMINISTIC)[2] == 0
    c.debug_shrink(slice_cap=2)
    assert c.run_sync(d, tp.MODE_DETERMINISTIC)[2] & tp.STATUS_INTERNAL
    c.debug_shrink(blob_cap=1024)
    assert c.run_sync(d, tp.MODE_FAST)[2] & tp.STATUS_INTERNAL
    c.debug_shrink()
    det, n, st = c.run_sync(d, tp.MODE_DETERMINISTIC)
    assert st == 0 and det.tobytes() == exp.tobytes()
    c.close()
    pads = [16, 9, 12]
    for rows in ([(0, 1, 9, 5, 0)], [(0, 1, 200, 5, 0), (0, 0, 3, 3, 40)], [(0, 1, 8, 5, 0), (0, 0, 3, 3, 40)]):
        dd = t1.make_digits(rows)
        e, st_e = _oracle(dd, 1, 3, 64, pads)
        c = tp.Clusterizer(1, 3, 64, pads, 16)
        for mode in (tp.MODE_DETERMINISTIC, tp.MODE_FAST):
            got, n, st = c.run_sync(_digits_tensor(dd, cuda_device), mode)
            assert st == st_e and n == len(e) and got.tobytes() == e.tobytes(), (rows, mode)
        c.close()
    assert st_e == 0          # the last case: pad 8 of a 9-pad row is in range
    # a zero-charge digit on a cell that also holds a real digit is no duplicate: it is ignored (Q4) in both
    # modes and both orders, in a sparse tile (one record per thread) and in a crowded one
    rng = np.random.default_rng(5)
    for n_fill in (0, 900):
        cells = rng.choice(100 * 12, size=n_fill, replace=False) + 12 * 20
        rows = [(0, 2, int(c % 12), int(c // 12), int(rng.integers(3, 90))) for c in cells if (int(c % 12), int(c // 12)) != (5, 5)]
        for pair in ([(0, 2, 5, 5, 0), (0, 2, 5, 5, 40)], [(0, 2, 5, 5, 40), (0, 2, 5, 5, 0)]):
            dd = t1.make_digits(pair + rows + [(0, 2, 7, 9, 0)])
            e, st_e = _oracle(dd, 1, 3, 128, pads)
            c = tp.Clusterizer(1, 3, 128, pads, len(dd))
            for mode in (tp.MODE_FAST, tp.MODE_DETERMINISTIC, tp.MODE_FAST):
                got, n, st = c.run_sync(_digits_tensor(dd, cuda_device), mode)
                assert st == st_e == 0 and n == len(e)
                assert got[np.argsort(_key(got))].tobytes() == e.tobytes(), (n_fill, mode)
            c.close()


def test_rtc_cache_survives_a_damaged_file(tp, cuda_device, tmp_path):
    """A truncated or foreign file in the shared cache directory is not loaded: the header (magic,
    length, checksum) does not match, the file is replaced by a fresh compile, results are unchanged."""
    fr = make_frame(1)
    exp, _ = _oracle(fr.digits_numpy(), fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads)
    tp.tpcclus_set_rtc_cache_dir(str(tmp_path))
    try:
        c = tp.Clusterizer(fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads, fr.n_digits, rtc=True)
        assert not c.rtc_cache_hit
        c.close()
        files = sorted(tmp_path.glob("tpcclus_*.cubin"))
        assert len(files) == 6                        # one cached binary per compilation unit
        files[0].write_bytes(files[0].read_bytes()[:1000])            # cut short
        files[1].write_bytes(b"\x7fELF" + b"\0" * 4096)                # not ours
        raw = bytearray(files[2].read_bytes()); raw[-1] ^= 0xFF
        files[2].write_bytes(bytes(raw))                                # one byte flipped
        c = tp.Clusterizer(fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads, fr.n_digits, rtc=True)
        assert not c.rtc_cache_hit                    # three units were compiled again
        assert c.run_sync(fr.digits.to(cuda_device), tp.MODE_DETERMINISTIC)[0].tobytes() == exp.tobytes()
        c.close()
        c = tp.Clusterizer(fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads, fr.n_digits, rtc=True)
        assert c.rtc_cache_hit
        c.close()
    finally:
        tp.tpcclus_set_rtc_cache_dir(None)


def test_cog_shared_reading(tp, cuda_device):
    """Reading Q10'' (TPCCLUS_COG_SHARED, second half; R8): charge sharing
    between clusters whose windows overlap, byte for byte against the oracle in the same reading --
    deterministic, fast, generic and RTC.  A handle of this reading runs units compiled with a time
    halo of 5 (partition, tiles, debug map): the a1 map, a frame longer than one coarse time-chunk
    (halo copies across the chunk border) and the densest peak pattern go through them too."""
    frames = [make_frame(1), make_frame(0), make_frame(4, device=cuda_device, sectors=[3, 20], n_time=300)]
    for fr in frames:
        d_np = fr.digits_numpy()
        exp, st, n = t1.clusterize(d_np.view(t1.DIGIT), fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads, cog_shared=True)
        plain, _ = _oracle(d_np, fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads)
        assert len(exp) == len(plain)
        if fr.meta["config"] != 0:
            assert exp.tobytes() != plain.tobytes()      # the reading matters on the crowded frames
        for rtc in (False, True):
            c = tp.Clusterizer(fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads, fr.n_digits, rtc=rtc, cog_shared=True)
            det = c.run_sync(fr.digits.to(cuda_device), tp.MODE_DETERMINISTIC)[0]
            fast = c.run_sync(fr.digits.to(cuda_device), tp.MODE_FAST)[0]
            if not rtc:
                assert set(c.loaded_units()) == {"part_coarse_h5", "dir", "part_fine_h5", "tiles_fast_s", "tiles_det_s", "order"}
                _, _, _, m = t1.clusterize(d_np.view(t1.DIGIT), fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads, return_map=True)
                assert np.array_equal(c.dense_map().cpu().numpy().view(np.uint16), m)      # step a1 through the halo-5 units
            c.close()
            assert det.tobytes() == exp.tobytes(), (fr.meta["name"], rtc)
            _check_fast(fast, exp)
    with pytest.raises(tp.TpcclusError):
        tp.Clusterizer(1, 16, 256, [64] * 16, 1000, cog_gated=True, cog_shared=True)
    # three coarse time-chunks, clusters planted on both chunk borders with partners two bins apart
    rng = np.random.default_rng(19)
    T, pads = 40000, [24, 40]
    rows = []
    for tb in (16256, 32512):
        for dt in range(-8, 9, 2):
            for r in (0, 1):
                rows.append((0, r, 10, tb + dt, int(rng.integers(30, 200))))
                rows.append((0, r, 12, tb + dt, int(rng.integers(30, 200))))
                rows.append((0, r, 11, tb + dt, int(rng.integers(3, 9))))
    seen = {(x[1], x[2], x[3]) for x in rows}
    for _ in range(20000):
        key = (int(rng.integers(0, 2)), int(rng.integers(0, 24)), int(rng.integers(0, T)))
        if key not in seen:
            seen.add(key)
            rows.append((0, key[0], key[1], key[2], int(rng.integers(1, 120))))
    d = t1.make_digits(rows)
    d = d[rng.permutation(len(d))]
    exp, st_exp, _ = t1.clusterize(d, 1, 2, T, pads, cog_shared=True)
    c = tp.Clusterizer(1, 2, T, pads, len(d), cog_shared=True)
    det, n, st = c.run_sync(_digits_tensor(d, cuda_device), tp.MODE_DETERMINISTIC)
    fast = c.run_sync(_digits_tensor(d, cuda_device), tp.MODE_FAST)[0]
    c.close()
    assert st == st_exp == 0 and det.tobytes() == exp.tobytes()
    _check_fast(fast, exp)
    # checkerboard of equal charges: every cell a survivor with up to 8 partners; and heavy ties
    T, P = 300, 138
    rows = [(0, 0, p, t, 50) for t in range(0, T, 2) for p in range(0, P, 2)]
    q = rng.integers(5, 10, size=(T, P))
    rows += [(0, 1, p, t, int(q[t, p])) for t in range(T) for p in range(P)]
    d = t1.make_digits(rows)
    d = d[rng.permutation(len(d))]
    exp, _, _ = t1.clusterize(d, 1, 2, T, [P, P], cog_shared=True)
    c = tp.Clusterizer(1, 2, T, [P, P], len(d), cog_shared=True)
    det = c.run_sync(_digits_tensor(d, cuda_device), tp.MODE_DETERMINISTIC)[0]
    fast = c.run_sync(_digits_tensor(d, cuda_device), tp.MODE_FAST)[0]
    c.close()
    assert det.tobytes() == exp.tobytes()
    _check_fast(fast, exp)


def test_host_pipeline_two_frames_in_flight(tp, cuda_device):
    """tpcclus_host_submit / tpcclus_host_wait: a stream of different frames through the two-deep host
    pipeline, results in submission order and equal to the oracle; a third submit without a wait is
    refused; the serial entry of the same handle still works afterwards."""
    import torch
    frames = [make_frame(0), make_frame(0, seed=7, n_time=200), make_frame(1), make_frame(0, seed=9), make_frame(1, seed=3)]
    big = frames[0]
    nmax = max(f.n_digits for f in frames)
    cap = nmax
    c = tp.Clusterizer(big.n_sectors, big.n_rows, big.n_time, big.n_pads, nmax, host_capacity=cap, host_pipelined=True)
    exps = []
    for f in frames:   # every frame on the geometry of the handle (CFG[1] frames use its first rows / pads / bins)
        d = f.digits_numpy().view(t1.DIGIT)
        e, st = _oracle(d, big.n_sectors, big.n_rows, big.n_time, big.n_pads)
        exps.append((e, st))
    hd = [f.digits.pin_memory() for f in frames]
    hc = [torch.empty((cap, 32), dtype=torch.uint8).pin_memory() for _ in range(2)]
    got = []
    for mode in (tp.MODE_DETERMINISTIC, tp.MODE_FAST):
        c.host_submit(hd[0], hc[0], mode)
        for i in range(1, len(frames)):
            c.host_submit(hd[i], hc[i & 1], mode)
            if i == 1:
                with pytest.raises(tp.TpcclusError):
                    c.host_submit(hd[2], hc[0], mode)          # two are in flight already
            n, st = c.host_wait()
            got.append((mode, i - 1, n, st, hc[(i - 1) & 1][:n].numpy().copy().view(tp.CLUSTER_DTYPE).reshape(-1)))
        n, st = c.host_wait()
        got.append((mode, len(frames) - 1, n, st, hc[(len(frames) - 1) & 1][:n].numpy().copy().view(tp.CLUSTER_DTYPE).reshape(-1)))
        with pytest.raises(tp.TpcclusError):
            c.host_wait()                                      # nothing in flight
    for mode, i, n, st, cl in got:
        e, st_e = exps[i]
        assert n == len(e) and st == st_e, (mode, i)
        if mode == tp.MODE_DETERMINISTIC:
            assert cl.tobytes() == e.tobytes(), i
        else:
            _check_fast(cl, e)
    n, st = c.run_host(hd[0], hc[0], tp.MODE_DETERMINISTIC)
    assert hc[0][:n].numpy().tobytes() == exps[0][0].tobytes()
    c.close()
