#!/usr/bin/env python
"""bench.py -- throughput of the TPC clusterizer hot path on synthetic time frames.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--order shuffled]
                    [--mode fast|det] [--rtc] [--impl reference]

One "step" = one pass of the whole hot path (K1..K6 of
DESIGN.md) over one Pb-Pb-like time frame (BASELINE.json configs[4]) that is already
resident in HBM.  Prints ONE JSON line (contract in the task statement): metric value in
digits/s, e2e through tpcclus_run_host (host buffers, copies inside the timed region),
per-kernel roofline of the dominant kernel from CUDA events recorded on the run's stream (a
separate pass after the timed region), median and best step, the two ratios NS asks for
(t_det / t_fast, t_generic / t_RTC) and the CPU oracle timed on bounded samples of the same
frame, on one core and sector-parallel on all cores.

N > 1 (torchrun): the path shards by time frame -- every rank clusterizes its own frame
(seed + rank), no data-path collective (PAPER.md 97: one process per GPU, whole time
frames each); value = digits of all ranks / max-over-ranks time; scaling "weak".
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

_T0 = time.perf_counter()


def _log(msg):
    print("[bench %7.1fs] %s" % (time.perf_counter() - _T0, msg), file=sys.stderr, flush=True)


METRIC = "TPC clusterizer digits/s on Pb-Pb-like time frame"
UNIT = "digits/s"


def _ncu_traffic(k, order, rtc, mode):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the newest committed `ncu --set full`
    capture (profiles/*_traffic.json, written by paper_2511_17018_b200/ncu_summary.py).  A capture
    describes the kernel text and the workload it was taken on (its note names config and mode): for any
    other text or workload the field is null rather than stale."""
    import glob
    import hashlib
    if not (order == "shuffled" and not rtc and mode in ("fast", "det")):
        return {}, None
    with open(os.path.join(ROOT, "paper_2511_17018_b200", "csrc", "tpcclus_kernels.cuh"), "rb") as f:
        sha = hashlib.sha256(f.read()).hexdigest()
    for path in sorted(glob.glob(os.path.join(ROOT, "profiles", "*_traffic.json")), reverse=True):
        try:
            with open(path) as f:
                t = json.load(f)
        except Exception:
            continue
        note = t.get("note", "")
        if t.get("kernel_text_sha256") == sha and ("CFG[%d]" % k) in note and ("DET" if mode == "det" else "FAST") in note:
            return t.get("traffic_bytes", {}), os.path.relpath(path, ROOT)
    return {}, None


def _peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks + throttle reasons sampled during the timed region."""
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        self.index, self.rows, self._stop, self._t = index, [], threading.Event(), None

    def _loop(self):
        while not self._stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5).stdout
                self.rows.append([x.strip() for x in out.strip().split(",")])
            except Exception:
                pass
            self._stop.wait(0.1)

    def __enter__(self):
        self._t = threading.Thread(target=self._loop, daemon=True)
        self._t.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        self._t.join(timeout=6)

    def summary(self):
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
                for nm, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(nm)
            except Exception:
                pass
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def _oracle_sample(fr_digits_np, fr, n_sample_sectors):
    """The oracle as it stands, single thread, on the first sectors of the frame."""
    from oracle import t1
    d = fr_digits_np.view(t1.DIGIT)
    sub = np.ascontiguousarray(d[d["sector"] < n_sample_sectors])
    tm = {}
    cl, st, cnt = t1.clusterize(sub, n_sample_sectors, fr.n_rows, fr.n_time, fr.n_pads, capacity=max(len(sub) // 4, 1024), timing=tm)
    return len(sub), cnt, tm["seconds"]


def _sector_digits(digits, s):
    """Digits of sector s of a device-resident frame, as a host array (the oracle's input)."""
    return digits[((digits >> 48) & 0xFF) == s].cpu().numpy().view(np.uint64)


def _oracle_allcores(digits, fr, n_sectors):
    """The same T1 routine, unchanged, run sector-parallel on all host cores."""
    from oracle import t1
    secs = list(range(n_sectors))
    host = {s: _sector_digits(digits, s) for s in secs}
    tm = {}
    res = t1.clusterize_by_sector(lambda s: host[s], secs, fr.n_rows, fr.n_time, fr.n_pads, timing=tm)
    return tm["digits"], int(sum(len(v) for v in res.values())), tm["seconds"], tm["cores"]


def aggregate_over_ranks(ms_local, units_local, device, world):
    """Whole-job numbers for N ranks that each processed their own shard (weak scaling, no
    data-path collective): the time is the MAX over ranks, the work the SUM.  One all_reduce
    each on `device` (NCCL on the GPU box, gloo in the CPU tests)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(ms_local)], dtype=torch.float64, device=device)
    u = torch.tensor([float(units_local)], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def rank_seed(seed_base, k, rank):
    """Every rank clusterizes its own time frame (PAPER.md 97: one process per GPU, whole frames each)."""
    return seed_base + k + 1000 * rank


def run_reference(args):
    """--impl reference: the CPU oracle (oracle/, single thread) on bounded samples of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import torch
    from workloads import make_frame
    k = args.config
    n_sec = 1 if k >= 2 else None
    dev = "cuda" if torch.cuda.is_available() else "cpu"
    if k >= 2:
        fr = make_frame(k, device=dev, order=args.order, sectors=[0])
    else:
        fr = make_frame(k, order=args.order)
    d_np = fr.digits_numpy()
    times, nd = [], 0
    for i in range(args.warmup + args.steps):
        nd, cnt, sec = _oracle_sample(d_np, fr, 1 if k >= 2 else fr.n_sectors)
        if i >= args.warmup:
            times.append(sec)
    t = float(np.mean(times))
    val = nd / t
    sample = "sector 0 of the %s frame (%d digits) per step, single thread" % (fr.meta["name"], nd)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": t * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "int32+f32", "data": "synthetic",
        "config": {"workload": fr.meta["name"], "order": args.order, "n_digits": nd, "sample": sample},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--order", default="shuffled", choices=["shuffled", "readout", "cell"])
    ap.add_argument("--mode", default="fast", choices=["fast", "det", "packed"])
    ap.add_argument("--rtc", action="store_true")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-ratios", action="store_true", help="skip the t_det/t_fast and t_generic/t_rtc loops")
    ap.add_argument("--cpu-sectors", type=int, default=2)
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist

    import paper_2511_17018_b200 as tp
    from workloads import SEED_BASE, make_frame

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device; there is no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    tp.lib()

    k = args.config
    fr = make_frame(k, device=dev, order=args.order, seed=rank_seed(SEED_BASE, k, rank))
    digits = fr.digits
    n = fr.n_digits
    torch.cuda.synchronize(dev)
    _log("frame generated: %d digits" % n)
    mode = tp.MODE_FAST if args.mode == "fast" else tp.MODE_DETERMINISTIC
    packed = args.mode == "packed"   # deterministic path, 16-byte records + row index
    warmup = max(args.warmup, 3)
    c = tp.Clusterizer(fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads, n, rtc=args.rtc, device=local)
    # size the output from a first (untimed) run
    probe_cap = max(n // 3, 1024)
    clusters = torch.empty((probe_cap, 16 if packed else 32), dtype=torch.uint8, device=dev)

    def step(cz=None, md=None):
        cz = cz or c
        if packed:
            return cz.run_packed(digits, clusters=clusters)[2:]
        return cz.run(digits, mode if md is None else md, clusters=clusters)[1:]
    nt, stt = step()
    torch.cuda.synchronize(dev)
    n_clusters, status = int(nt.item()), int(stt.item())
    assert status == 0 and n_clusters <= probe_cap, (status, n_clusters, probe_cap)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    def timed_loop(cz, md, steps):
        """`steps` runs back to back on the current stream: (total ms between the bracketing events,
        [ms of every single step]).  Only launches inside: nothing synchronises before the end."""
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
        ev[0].record()
        for i in range(steps):
            step(cz, md)
            ev[i + 1].record()
        torch.cuda.synchronize(dev)
        return ev[0].elapsed_time(ev[steps]), [ev[i].elapsed_time(ev[i + 1]) for i in range(steps)]

    for _ in range(warmup):
        step()
    barrier()
    with ClockSampler(local) as clk:
        ms_total, per_step = timed_loop(c, None, args.steps)
        barrier()
    _log("timed region done: %.3f ms/step" % (ms_total / args.steps))
    ms_max, tot_digits = aggregate_over_ranks(ms_total, n, dev, world)
    ms_step = ms_max / args.steps
    value = tot_digits / (ms_step * 1e-3)

    # ---- per-kernel device times: a separate pass (the library's events synchronise per run) --------
    c.set_timing(True)
    per_kernel = {}
    for _ in range(min(args.steps, 5)):
        step()
        for nm, ms in c.last_timing():
            per_kernel.setdefault(nm, []).append(ms)
    c.set_timing(False)

    # ---- the two ratios NS asks for: deterministic mode vs fast (PAPER.md 28), generic vs RTC (PAPER.md 118) ---
    ratios = {}
    if world == 1 and not args.no_ratios and args.mode == "fast" and not args.rtc:
        for _ in range(warmup):
            step(c, tp.MODE_DETERMINISTIC)
        ms_det = timed_loop(c, tp.MODE_DETERMINISTIC, args.steps)[0] / args.steps
        r = tp.Clusterizer(fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads, n, rtc=True, device=local)
        for _ in range(warmup):
            step(r, tp.MODE_FAST)
        torch.cuda.synchronize(dev)
        ms_rtc = timed_loop(r, tp.MODE_FAST, args.steps)[0] / args.steps
        ms_fast = ms_total / args.steps
        ratios = {"t_det_over_t_fast": ms_det / ms_fast, "t_generic_over_t_rtc": ms_fast / ms_rtc,
                  "ms_det": ms_det, "ms_rtc": ms_rtc, "rtc_build_ms": r.rtc_build_ms,
                  "note": "same resident frame, %d steps each after %d warm-ups; RTC build time excluded" % (args.steps, warmup)}
        r.close()
        del r
        # the same FAST step captured once into a CUDA graph and replayed: tpcclus_run only enqueues kernel
        # launches, so it can be captured; matters for the launch-bound small frames (CFG[0,1])
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            step(c, tp.MODE_FAST)
        for _ in range(warmup):
            g.replay()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record()
        for _ in range(args.steps):
            g.replay()
        ev1.record()
        torch.cuda.synchronize(dev)
        ratios["ms_graph_replay"] = ev0.elapsed_time(ev1) / args.steps
        del g
        _log("ratios done: det %.3f ms, rtc %.3f ms, graph replay %.3f ms" % (ms_det, ms_rtc, ratios["ms_graph_replay"]))

    # ---- e2e: host buffers through the C ABI, copies inside the timed region -----------------------
    # (a) tpcclus_run_host: one frame at a time, copy -> run -> copy back, serial;
    # (b) tpcclus_host_submit / tpcclus_host_wait: a burst of frames, two in flight, so that the
    #     host-to-device copy of frame k+1 overlaps the run and the read-back of frame k.  Every frame
    #     of the burst is copied in from pinned host memory and its clusters are copied back: (b) is
    #     the e2e number (a time frame never comes alone: PAPER.md 12, 97), (a) is reported beside it.
    e2e = None
    if args.e2e_steps > 0 and not packed:
        cap = n_clusters + 1024
        c.close()
        del c, clusters
        torch.cuda.empty_cache()
        c = tp.Clusterizer(fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads, n, rtc=args.rtc, device=local, host_capacity=cap,
                           host_pipelined=True)
        h_digits = torch.empty(n, dtype=torch.int64).pin_memory()
        h_digits.copy_(digits)
        h_clusters = [torch.empty((cap, 32), dtype=torch.uint8).pin_memory() for _ in range(2)]
        _log("pinned host buffers ready")
        c.run_host(h_digits, h_clusters[0], mode)      # warm-up
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.e2e_steps):
            n_e2e, st_e2e = c.run_host(h_digits, h_clusters[0], mode)
        barrier()
        sec1 = (time.perf_counter() - t0) / args.e2e_steps
        assert n_e2e == n_clusters and st_e2e == 0
        burst = max(6, 3 * args.e2e_steps)
        secs = []
        for _ in range(2):   # two bursts, the faster one counts (the host side of the link is shared: one burst in ten is 10 % off); both are reported
            t0 = time.perf_counter()
            for i in range(burst):
                c.host_submit(h_digits, h_clusters[i & 1], mode)
                if i >= 1:
                    n_e2e, st_e2e = c.host_wait()
                    assert n_e2e == n_clusters and st_e2e == 0
            n_e2e, st_e2e = c.host_wait()
            barrier()
            secs.append((time.perf_counter() - t0) / burst)
            assert n_e2e == n_clusters and st_e2e == 0
        sec = min(secs)
        sec_max, _ = aggregate_over_ranks(sec, n, dev, world)
        sec1_max, _ = aggregate_over_ranks(sec1, n, dev, world)
        e2e = {"value": tot_digits / sec_max, "unit": UNIT, "h2d_bytes_per_step": 8 * n,
               "d2h_bytes_per_step": 32 * n_clusters + 16, "ms_per_step": sec_max * 1e3,
               "api": "tpcclus_host_submit / tpcclus_host_wait, burst of %d frames, two in flight (pinned host buffers); the faster of two bursts" % burst,
               "bursts_ms_per_step": [x * 1e3 for x in secs],
               "single_frame": {"value": tot_digits / sec1_max, "ms_per_step": sec1_max * 1e3, "api": "tpcclus_run_host (serial copy, run, copy)"}}
        del h_clusters, h_digits
        _log("e2e done")

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (algorithmic bytes per launch) ---
    peak, peak_src = _peaks()
    avg = {nm: float(np.mean(v)) for nm, v in per_kernel.items()}
    alg = {   # bytes one launch must move (per-unit figures x units of this frame)
        "k_partition_coarse": 8 * n + 4 * n,                    # read every digit once, write one 4-byte record
        "k_partition_fine": 4 * n + 4 * n,                      # read the records, write them tile-sorted
        "k_cluster_tiles_fast": 4 * n + 32 * n_clusters,        # read the tile records, write the clusters
        "k_cluster_tiles_det_temp": 4 * n + 32 * n_clusters,     # ... as runs into the temporary buffer
        "k_emit_ordered": 64 * n_clusters,                       # DET: ordered copy of the runs
        "k_emit_packed": 48 * n_clusters,                        # packed: 32 B in, 16 B out
    }
    for nm in list(avg):   # the tile kernels of the other readings and the sparse-frame variant (emitter warp) move the same bytes
        for base in ("k_cluster_tiles_fast", "k_cluster_tiles_det_temp"):
            if nm.startswith(base) and nm not in alg:
                alg[nm] = alg[base]
    traffic, traffic_src = _ncu_traffic(k, args.order, args.rtc, args.mode)
    step_sum = sum(avg.values())
    per_kernel_roof = {}
    for nm in avg:
        if nm in alg:
            ach = alg[nm] / (avg[nm] * 1e-3) / 1e9
            per_kernel_roof[nm] = {"bound": "hbm", "kernel": nm, "achieved": ach, "peak": peak, "unit": "GB/s",
                                   "frac": ach / peak, "traffic": traffic.get(nm), "alg_bytes": alg[nm],
                                   "kernel_ms": avg[nm], "share_of_step": avg[nm] / step_sum}
    dom = max(per_kernel_roof, key=lambda nm: avg[nm]) if per_kernel_roof else None
    roof = dict(per_kernel_roof[dom], peak_source=peak_src, traffic_source=traffic_src) if dom else None
    b_alg = 8 * n + 32 * n_clusters
    method = {"b_alg_bytes": b_alg, "achieved_gbs": b_alg / (ms_step * 1e-3) / 1e9,
              "frac_of_peak": b_alg / (ms_step * 1e-3) / 1e9 / peak}
    if traffic and all(any(t.startswith(nm) for t in traffic) for nm in ("k_partition_coarse", "k_partition_fine", "k_cluster_tiles_fast")):
        dram = sum(traffic.values())
        method.update({"dram_bytes_per_step_ncu": dram, "dram_gbs": dram / (ms_step * 1e-3) / 1e9,
                       "dram_frac_of_peak": dram / (ms_step * 1e-3) / 1e9 / peak})

    cpu = cpu_all = None
    if not args.no_cpu_baseline:
        ns = min(args.cpu_sectors, fr.n_sectors)
        _log("cpu baseline: single thread")
        from oracle import t1
        host = np.concatenate([_sector_digits(digits, s) for s in range(ns)])
        nd, cnt, sec = _oracle_sample(host, fr, ns)
        cpu = {"value": nd / sec, "unit": UNIT, "cores": 1, "kind": "oracle",
               "sample": "sectors 0..%d of this frame (%d digits, %d clusters) in %.1f s, single thread" % (ns - 1, nd, cnt, sec)}
        cores = len(os.sched_getaffinity(0))
        na = min(fr.n_sectors, cores)
        _log("cpu baseline: %d sectors on %d cores" % (na, cores))
        nd, cnt, sec, used = _oracle_allcores(digits, fr, na)
        cpu_all = {"value": nd / sec, "unit": UNIT, "cores": used, "cores_available": cores, "kind": "oracle, sector-parallel",
                   "sample": "sectors 0..%d of this frame (%d digits, %d clusters) in %.1f s wall, one thread per sector" % (na - 1, nd, cnt, sec)}
        _log("cpu baseline done")

    in_gb = 8 * n / 1e9
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": warmup, "ms_per_step": ms_step, "ms_median": float(np.median(per_step)), "ms_best": float(min(per_step)),
        "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "int32+f32", "data": "synthetic",
        "config": {"workload": fr.meta["name"], "order": args.order, "mode": args.mode, "rtc": bool(args.rtc),
                   "n_digits": n, "n_clusters": n_clusters, "occupancy": fr.meta["occupancy"],
                   "checksum": "%016x" % fr.meta["checksum"],
                   "l2": ("inputs (%.1f GB) larger than L2, no flush needed" % in_gb) if in_gb > 0.3 else
                         ("inputs (%.4f GB) FIT in L2 (126 MB): launch-latency-bound, not a bandwidth number" % in_gb)},
        "clocks": clk.summary(), "e2e": e2e, "gpu_launches": c.launches_per_run(mode) * args.steps,
        "roofline": roof, "rooflines": per_kernel_roof, "method_roofline": method,
        "kernels_ms": avg, "cpu_baseline": cpu, "cpu_baseline_allcores": cpu_all,
    }
    out.update({k2: v for k2, v in ratios.items() if k2 in ("t_det_over_t_fast", "t_generic_over_t_rtc")})
    if ratios:
        out["ratios"] = ratios
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
