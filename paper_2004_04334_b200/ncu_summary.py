"""Text summaries of an ``ncu --set full`` capture (``.ncu-rep``), for ``profiles/``.

    python -m paper_2004_04334_b200.ncu_summary REPORT.ncu-rep [--label TEXT] [--traffic-json OUT.json] [--source K_CLUSTER_FILE]

Prints a markdown table with one row per profiled launch (time, DRAM bytes, warp instructions, issue rate, shared-memory
wavefronts, the top stall reasons) read with ``ncu -i REPORT --page raw --csv``.  With ``--traffic-json`` it also writes
the per-launch DRAM bytes and warp instructions of the LAST launch of every kernel (``profiles/traffic.json``: what
``bench.py`` quotes as ``roofline.traffic``).  With ``--source FILE`` (a source file name such as ``k_cluster.cuh``) it
adds the share of executed warp instructions and of stall samples per source line of that file from the source page
(needs ``--import-source on`` at capture time and ``-lineinfo`` at build time).  Nothing here runs on the GPU; it only
reads a report that a committed command wrote.
"""
from __future__ import annotations

import argparse
import collections
import csv
import io
import json
import re
import subprocess
import sys


def _ncu(args):
    return subprocess.run(["ncu", *args], capture_output=True, text=True, check=True).stdout


def _num(s):
    s = (s or "").replace(",", "")
    try:
        return float(s)
    except ValueError:
        return 0.0


def short_name(full: str) -> str:
    m = re.search(r"(k_[a-z_]+)(<[^>]*>)?", full)
    return m.group(1) + (m.group(2) or "") if m else full[:40]


def raw_rows(report: str):
    rows = list(csv.reader(io.StringIO(_ncu(["-i", report, "--page", "raw", "--csv"]))))
    hdr = rows[0]
    return [dict(zip(hdr, r)) for r in rows[2:] if len(r) == len(hdr)]


def launch_table(rows):
    out = ["| # | kernel | grid x block | time (us) | dram read (MB) | dram write (MB) | warp-inst (M) | threads/inst | "
           "issue active | warps active % | smem wavefronts (M) | lsu data-pipe % | top stalls |",
           "|---|---|---|---|---|---|---|---|---|---|---|---|---|"]
    for d in rows:
        stall_keys = [k for k in d if "pcsamp_warps_issue_stalled" in k and "not_issued" not in k]
        tot = sum(_num(d[k]) for k in stall_keys) or 1.0
        top = sorted(((_num(d[k]), k.split("stalled_")[1]) for k in stall_keys), reverse=True)[:4]
        t_us = _num(d.get("gpu__time_duration.sum")) * {"ns": 1e-3, "us": 1.0, "ms": 1e3, "s": 1e6}.get(
            _UNITS.get("gpu__time_duration.sum", "us").lower().replace("second", "s").replace("msecond", "ms"), 1.0)
        out.append("| {} | {} | {} x {} | {:.1f} | {:.1f} | {:.1f} | {:.1f} | {:.1f} | {:.2f} | {:.1f} | {:.1f} | {:.1f} | {} |".format(
            d.get("ID"), short_name(d.get("Kernel Name", "")), d.get("Grid Size", ""), d.get("Block Size", ""),
            t_us, _bytes_mb(d, "dram__bytes_read.sum"), _bytes_mb(d, "dram__bytes_write.sum"),
            _num(d.get("smsp__inst_executed.sum")) / 1e6, _num(d.get("smsp__thread_inst_executed_per_inst_executed.ratio")),
            _num(d.get("smsp__issue_active.avg.per_cycle_active")), _num(d.get("sm__warps_active.avg.pct_of_peak_sustained_active")),
            _num(d.get("l1tex__data_pipe_lsu_wavefronts_mem_shared.sum")) / 1e6,
            _num(d.get("l1tex__data_pipe_lsu_wavefronts.avg.pct_of_peak_sustained_elapsed")),
            ", ".join(f"{n} {v / tot * 100:.0f}%" for v, n in top)))
    return "\n".join(out)


_UNITS = {}


def _bytes_mb(d, key):
    """dram__bytes_*.sum in MB whatever unit ncu chose for the column (the unit row is kept in _UNITS)."""
    v = _num(d.get(key))
    u = _UNITS.get(key, "Mbyte").lower()
    return v * {"byte": 1e-6, "kbyte": 1e-3, "mbyte": 1.0, "gbyte": 1e3}.get(u, 1.0)


def traffic_json(rows, source_note):
    last = collections.OrderedDict()
    for d in rows:
        last[short_name(d.get("Kernel Name", "")).split("<")[0]] = d
    return {"source": source_note,
            "kernels": {k: {"dram_bytes_per_launch": int(round((_bytes_mb(d, "dram__bytes_read.sum") + _bytes_mb(d, "dram__bytes_write.sum")) * 1e6)),
                            "warp_inst_per_launch": int(_num(d.get("smsp__inst_executed.sum")))} for k, d in last.items()}}


def source_lines(report: str, file_suffix: str, kernel_regex: str, min_pct: float = 0.3):
    txt = _ncu(["-i", report, "--page", "source", "--csv", "--print-source", "cuda,sass", "-k", f"regex:{kernel_regex}"])
    cur, hdr, seen = None, None, set()
    per_line, total_inst, total_samp = collections.OrderedDict(), 0.0, 0.0
    for r in csv.reader(io.StringIO(txt)):
        if not r:
            continue
        if r[0] == "File Path":
            cur = r[1]
        elif r[0] == "Line No":
            hdr = r
        elif hdr and cur and r[0].isdigit():
            key = (cur, int(r[0]))
            if key in seen:                       # a second launch of the same kernel in the report
                continue
            seen.add(key)
            d = dict(zip(hdr, r))
            inst, samp = _num(d.get("Instructions Executed")), _num(d.get("# Samples"))
            total_inst += inst
            total_samp += samp
            if cur.endswith(file_suffix):
                per_line[int(r[0])] = (r[1], inst, samp)
    out = [f"| line | % of warp instructions | % of stall samples | source ({file_suffix}) |", "|---|---|---|---|"]
    for ln, (src, inst, samp) in per_line.items():
        pi, ps = inst / max(total_inst, 1) * 100, samp / max(total_samp, 1) * 100
        if pi >= min_pct or ps >= min_pct:
            out.append(f"| {ln} | {pi:.2f} | {ps:.2f} | `{src.strip()[:110]}` |")
    return "\n".join(out)


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("report")
    ap.add_argument("--label", default="")
    ap.add_argument("--traffic-json", default=None)
    ap.add_argument("--source", default=None, help="source file name whose lines to list (e.g. k_cluster.cuh)")
    ap.add_argument("--kernel", default="k_cluster", help="kernel regex for --source")
    a = ap.parse_args(argv)
    raw = list(csv.reader(io.StringIO(_ncu(["-i", a.report, "--page", "raw", "--csv"]))))
    hdr, units = raw[0], raw[1]
    _UNITS.update(dict(zip(hdr, units)))
    rows = [dict(zip(hdr, r)) for r in raw[2:] if len(r) == len(hdr)]
    print(f"### {a.label or a.report}\n")
    print(launch_table(rows))
    if a.source:
        print()
        print(source_lines(a.report, a.source, a.kernel))
    if a.traffic_json:
        with open(a.traffic_json, "w") as f:
            json.dump(traffic_json(rows, f"python -m paper_2004_04334_b200.ncu_summary {a.report} ({a.label}): dram__bytes_read.sum + "
                                         "dram__bytes_write.sum and smsp__inst_executed.sum of the last launch of every kernel"), f, indent=1)
            f.write("\n")


if __name__ == "__main__":
    sys.exit(main())
