"""Turns Nsight Compute captures of bench.py into the text summaries kept under profiles/.

    python -m paper_2511_17018_b200.ncu_summary --tag r02a --rep gpurun_out/prof.ncu-rep \
        [--launches gpurun_out/launches.csv] [--note "CFG[4] shuffled FAST generic"]

Writes profiles/<tag>_ncu_full_summary.txt (per kernel: duration, DRAM bytes, occupancy, shared-memory
wavefronts and bank conflicts, instruction counts, the six largest stall reasons), profiles/<tag>_traffic.json
(dram__bytes_read.sum + dram__bytes_write.sum per launch and kernel, with the sha256 of the kernel
text it was measured on: bench.py reports `traffic` from it only while that text is unchanged) and,
with --launches, profiles/<tag>_launches_summary.txt (mean device time and share per kernel from the
`--metrics gpu__time_duration.sum` launch list), with --top-lines N profiles/<tag>_top_lines.txt (the hottest source
lines per kernel from the source page).  Reads reports only; runs no kernel.
"""
from __future__ import annotations

import argparse
import collections
import csv
import hashlib
import json
import os
import subprocess

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
KERNEL_TEXT = os.path.join(ROOT, "paper_2511_17018_b200", "csrc", "tpcclus_kernels.cuh")

WANT = ["gpu__time_duration.sum", "dram__bytes_read.sum", "dram__bytes_write.sum",
        "gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed", "sm__warps_active.avg.pct_of_peak_sustained_active",
        "launch__registers_per_thread", "launch__occupancy_limit_shared_mem", "launch__occupancy_limit_registers",
        "sm__throughput.avg.pct_of_peak_sustained_elapsed", "l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum",
        "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum", "smsp__inst_executed.sum", "lts__t_sector_hit_rate.pct",
        "lts__t_sectors_srcunit_tex_op_read.sum", "lts__t_sectors_srcunit_tex_op_write.sum",
        "sm__cycles_elapsed.max", "smsp__issue_active.avg.pct_of_peak_sustained_active",
        "smsp__thread_inst_executed_per_inst_executed.ratio"]
TO_BYTES = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}


def kernel_text_sha256() -> str:
    with open(KERNEL_TEXT, "rb") as f:
        return hashlib.sha256(f.read()).hexdigest()


def _num(x: str) -> float:
    return float(x.replace(",", ""))


def summarise_rep(rep: str, tag: str, note: str) -> dict:
    raw = subprocess.run(["ncu", "-i", rep, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    rows = list(csv.reader(raw.splitlines()))
    hdr, units, data = rows[0], rows[1], rows[2:]
    stalls = [h for h in hdr if h.startswith("smsp__average_warps_issue_stalled") and h.endswith("_per_issue_active.ratio")]
    ki = hdr.index("Kernel Name")
    out = ["ncu --set full --clock-control none; %s (command in %s_README.md)" % (note, tag)]
    traffic = collections.OrderedDict()
    for x in data:
        out.append("%-70s %s" % ("Kernel Name", x[ki]))
        for w in WANT:
            if w in hdr:
                i = hdr.index(w)
                out.append("%-70s %s %s" % (w, x[i], units[i]))
        st = sorted(((_num(x[hdr.index(s)]), s) for s in stalls if x[hdr.index(s)]), reverse=True)[:6]
        for v, s in st:
            nm = s.replace("smsp__average_warps_issue_stalled_", "").replace("_per_issue_active.ratio", "")
            out.append("  stall %-40s %.3f warps per issue-active cycle" % (nm, v))
        out.append("")
        ir, iw = hdr.index("dram__bytes_read.sum"), hdr.index("dram__bytes_write.sum")
        b = _num(x[ir]) * TO_BYTES[units[ir]] + _num(x[iw]) * TO_BYTES[units[iw]]
        traffic.setdefault(x[ki], []).append(b)
    os.makedirs(os.path.join(ROOT, "profiles"), exist_ok=True)
    with open(os.path.join(ROOT, "profiles", "%s_ncu_full_summary.txt" % tag), "w") as f:
        f.write("\n".join(out) + "\n")
    head = subprocess.run(["git", "-C", ROOT, "rev-parse", "HEAD"], capture_output=True, text=True).stdout.strip()
    tj = {"capture": tag, "note": note, "git_head_at_summary": head, "kernel_text_sha256": kernel_text_sha256(),
          "metric": "dram__bytes_read.sum + dram__bytes_write.sum, bytes per launch (mean over the captured launches)",
          "traffic_bytes": {k: sum(v) / len(v) for k, v in traffic.items()}}
    with open(os.path.join(ROOT, "profiles", "%s_traffic.json" % tag), "w") as f:
        json.dump(tj, f, indent=1)
        f.write("\n")
    return tj


def summarise_launches(path: str, tag: str) -> None:
    rows = [r for r in csv.reader(open(path)) if len(r) > 5]
    h = rows[0]
    k, v = h.index("Kernel Name"), h.index("Metric Value")
    acc = collections.OrderedDict()
    for r in rows[1:]:
        try:
            acc.setdefault(r[k], []).append(_num(r[v]))
        except ValueError:
            pass
    tot = sum(sum(x) / len(x) for x in acc.values())
    with open(os.path.join(ROOT, "profiles", "%s_launches_summary.txt" % tag), "w") as f:
        f.write("kernel, launches, mean gpu__time_duration (ms), share of the summed means\n")
        for n, x in acc.items():
            f.write("%s, %d, %.4f, %.1f %%\n" % (n, len(x), sum(x) / len(x) / 1e6, 100 * sum(x) / len(x) / tot))


def summarise_lines(rep: str, tag: str, top: int) -> None:
    """profiles/<tag>_top_lines.txt: per kernel of the report, the source lines of the kernel text with the most executed
    warp instructions (share of instructions, of stall samples and of shared-memory wavefronts, ideal wavefronts beside
    them).  Needs a capture with --import-source on of a build with -lineinfo; the line numbers are those of the kernel
    text whose sha256 the traffic json of the same tag records."""
    raw = subprocess.run(["ncu", "-i", rep, "--page", "source", "--csv", "--print-source", "cuda,sass"], capture_output=True, text=True, check=True).stdout

    def num(x):
        try:
            return float(x)
        except ValueError:
            return 0.0
    cur, hdr, idx, data = None, None, None, collections.OrderedDict()
    for r in csv.reader(raw.splitlines()):
        if len(r) >= 2 and r[0] == "Function Name":
            cur = r[1]
            continue
        if r and r[0] == "Line No":
            hdr, idx = r, {h: i for i, h in enumerate(r)}
            continue
        if cur is None or hdr is None or len(r) < len(hdr) or r[0] == "":
            continue
        d = data.setdefault(cur, {}).setdefault(int(r[0]), [r[1], 0.0, 0.0, 0.0, 0.0])
        for j, col in ((1, "Instructions Executed"), (2, "# Samples"), (3, "L1 Wavefronts Shared"), (4, "L1 Wavefronts Shared Ideal")):
            if col in idx:   # (a kernel without shared memory has no wavefront columns)
                d[j] += num(r[idx[col]])
    out = ["ncu --page source of %s: the %d source lines with the most executed warp instructions per kernel" % (os.path.basename(rep), top),
           "(line of csrc/tpcclus_kernels.cuh or of a CUDA header, share of the kernel's instructions / stall samples / shared-memory wavefronts (ideal))", ""]
    for k, lines in data.items():
        ti = sum(v[1] for v in lines.values()) or 1.0
        ts = sum(v[2] for v in lines.values()) or 1.0
        tw = sum(v[3] for v in lines.values()) or 1.0
        out.append("== %s: %.3e warp instructions, %.3e shared-memory wavefronts" % (k, ti, tw))
        for ln, v in sorted(lines.items(), key=lambda kv: -kv[1][1])[:top]:
            out.append("%5d  inst %5.1f %%  samples %5.1f %%  wavefronts %5.1f %% (ideal %4.1f %%) | %s" %
                       (ln, 100 * v[1] / ti, 100 * v[2] / ts, 100 * v[3] / tw, 100 * v[4] / tw, v[0].strip()[:110]))
        out.append("")
    with open(os.path.join(ROOT, "profiles", "%s_top_lines.txt" % tag), "w") as f:
        f.write("\n".join(out) + "\n")


SASS_PATTERNS = ["UBLKCP", "UBLKPF", "SYNCS", "FENCE.VIEW.ASYNC", "STG.E.ENL2.256", "LDG.E.NA", "VIMNMX", "ATOMS", "ATOMG", "REDG",
                 "VOTE", "SHFL", "BAR.", "LDS", "STS", "HMMA", "UTC"]


def summarise_sass(tag: str) -> None:
    """Counts of the SASS mnemonics that show what the kernels are made of (bulk copies, mbarriers,
    packed min/max, shared atomics; no tensor-core instruction) per kernel, from the unit binaries the
    build leaves in build/unit_*.cubin (`python -m paper_2511_17018_b200.build`)."""
    import glob
    import re
    out = ["cuobjdump -sass build/unit_<name>.cubin, per kernel: instructions, registers (ptxas), and occurrences of the mnemonics",
           "that matter (UBLKCP/UBLKPF = cp.async.bulk / prefetch, SYNCS = mbarrier, VIMNMX = packed u16x2 max, ENL2.256 = 32-byte store)", ""]
    for cub in sorted(glob.glob(os.path.join(ROOT, "build", "unit_*.cubin"))):
        sass = subprocess.run(["cuobjdump", "-sass", cub], capture_output=True, text=True, check=True).stdout
        res = subprocess.run(["cuobjdump", "-res-usage", cub], capture_output=True, text=True).stdout
        regs = dict(re.findall(r"Function (\w+):\s*\n\s*REG:(\d+)", res))
        out.append("== %s (arch %s)" % (os.path.basename(cub), ",".join(sorted(set(re.findall(r"code for (sm_\w+)", sass))))))
        for fn, body in re.findall(r"Function : (\w+)\n(.*?)(?=\n\s*Function : |\Z)", sass, flags=re.S):
            ins = re.findall(r"^\s+/\*[0-9a-f]{4,}\*/\s+(.*?);", body, flags=re.M)
            counts = []
            for pat in SASS_PATTERNS:
                n = sum(1 for x in ins if pat in x)
                if n:
                    counts.append("%s %d" % (pat, n))
            out.append("  %-34s %5d instructions, %s registers | %s" % (fn, len(ins), regs.get(fn, "?"), ", ".join(counts)))
    with open(os.path.join(ROOT, "profiles", "%s_sass_summary.txt" % tag), "w") as f:
        f.write("\n".join(out) + "\n")


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--tag", required=True)
    ap.add_argument("--rep")
    ap.add_argument("--launches")
    ap.add_argument("--note", default="CFG[4] shuffled FAST generic")
    ap.add_argument("--sass", action="store_true", help="write profiles/<tag>_sass_summary.txt from build/unit_*.cubin")
    ap.add_argument("--top-lines", type=int, default=0, help="also write profiles/<tag>_top_lines.txt: the N hottest source lines per kernel")
    a = ap.parse_args()
    if a.sass:
        summarise_sass(a.tag)
    if a.rep:
        print(json.dumps(summarise_rep(a.rep, a.tag, a.note)["traffic_bytes"]))
    if a.launches:
        summarise_launches(a.launches, a.tag)
    if a.rep and a.top_lines:
        summarise_lines(a.rep, a.tag, a.top_lines)


if __name__ == "__main__":
    main()
