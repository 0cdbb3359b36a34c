"""Turn one `ncu --set full` capture into the two files bench.py and the reader of profiles/ use.

    ncu -i gpurun_out/X.ncu-rep --page raw --csv --print-units base > gpurun_out/X.raw.csv        (here, no GPU needed)
    python -m paper_1212_6332_b200.ncu_summary gpurun_out/X.raw.csv --workload 3a \
        --pick force=k_force:1 --pick density=k_density:1 [--pick list=k_build_list:0] \
        --command "<the full ncu command that made the capture>" --out profiles/r02_ncu_3a

writes  <out>.md          the table of counters per picked launch (text, for the reader)
        profiles/ncu_<workload>.json   the per-launch figures bench.py prints in `roofline` (DRAM traffic, executed FP64
                                       instructions), keyed by a hash of csrc/ so that a later kernel change makes them
                                       read as stale instead of current.
`--pick name=regex:n` selects the n-th (0-based) captured launch whose kernel name matches the regex.
Only argument marshalling and text formatting: nothing of the method is computed here.
"""
from __future__ import annotations

import argparse
import csv
import glob
import hashlib
import json
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

TABLE = [
    "gpu__time_duration.sum", "dram__bytes_read.sum", "dram__bytes_write.sum",
    "smsp__sass_thread_inst_executed_op_dfma_pred_on.sum", "smsp__sass_thread_inst_executed_op_dmul_pred_on.sum",
    "smsp__sass_thread_inst_executed_op_dadd_pred_on.sum", "sm__inst_executed_pipe_fp64.sum",
    "smsp__inst_executed.sum", "smsp__thread_inst_executed_per_inst_executed.ratio",
    "sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active", "smsp__issue_active.avg.pct_of_peak_sustained_active",
    "sm__warps_active.avg.pct_of_peak_sustained_active", "launch__registers_per_thread",
    "l1tex__throughput.avg.pct_of_peak_sustained_active", "l1tex__data_pipe_lsu_wavefronts.avg.pct_of_peak_sustained_elapsed",
    "l1tex__t_sector_hit_rate.pct", "lts__t_sector_hit_rate.pct", "lts__t_bytes.sum",
    "gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed",
    "smsp__average_warps_issue_stalled_long_scoreboard_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_wait_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_math_pipe_throttle_per_issue_active.ratio",
    "sm__cycles_elapsed.avg.per_second",
]


def csrc_sha() -> str:
    h = hashlib.sha256()
    for f in sorted(glob.glob(os.path.join(ROOT, "paper_1212_6332_b200", "csrc", "*"))):
        if os.path.basename(f) in ("md_probe.cu", "md_noalloc.cu"):   # diagnostics / stand-alone entry points: not part of the MD path
            continue
        h.update(os.path.basename(f).encode())
        with open(f, "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def read_raw(path: str):
    with open(path, newline="") as fh:
        rows = [r for r in csv.reader(fh) if r]
    start = next(i for i, r in enumerate(rows) if "Kernel Name" in r)      # ncu may print ==PROF== lines first
    names, units = rows[start], rows[start + 1]
    return names, units, rows[start + 2:]


def num(x: str):
    try:
        return float(x.replace(",", ""))
    except ValueError:
        return None


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("raw_csv")
    ap.add_argument("--workload", required=True)
    ap.add_argument("--pick", action="append", required=True)
    ap.add_argument("--command", required=True)
    ap.add_argument("--out", required=True)
    ap.add_argument("--title", default=None)
    a = ap.parse_args()
    names, units, rows = read_raw(a.raw_csv)
    col = {n: i for i, n in enumerate(names)}
    kn = col["Kernel Name"]
    picked = {}
    for p in a.pick:
        label, rest = p.split("=", 1)
        rx, idx = rest.rsplit(":", 1)
        hits = [r for r in rows if re.search(rx, r[kn])]
        if len(hits) <= int(idx):
            raise SystemExit(f"--pick {p}: only {len(hits)} launches match")
        picked[label] = hits[int(idx)]
    present = [m for m in TABLE if m in col]
    md = [f"# {a.title or 'ncu --set full, workload ' + a.workload}", "", "Command (under gpurun on one B200, after the same command had exited 0 without ncu):", "",
          f"    {a.command}", "", f"Read here with `ncu -i <rep> --page raw --csv --print-units base`, summarised by "
          f"`python -m paper_1212_6332_b200.ncu_summary`; csrc hash `{csrc_sha()}`.", "",
          "| metric | unit | " + " | ".join(f"{k}: `{picked[k][kn][:60]}`" for k in picked) + " |", "|---|---|" + "---|" * len(picked)]
    for m in present:
        md.append(f"| {m} | {units[col[m]]} | " + " | ".join(picked[k][col[m]] for k in picked) + " |")
    kernels = {}
    for k, r in picked.items():
        g = lambda m: num(r[col[m]]) if m in col else None  # noqa: E731
        dfma, dmul, dadd = (g(f"smsp__sass_thread_inst_executed_op_{o}_pred_on.sum") for o in ("dfma", "dmul", "dadd"))
        rd, wr = g("dram__bytes_read.sum"), g("dram__bytes_write.sum")
        kernels[k] = {
            "name": r[kn], "duration_ns": g("gpu__time_duration.sum"),
            "dram_bytes": (rd + wr) if rd is not None and wr is not None else None, "dram_bytes_read": rd, "dram_bytes_write": wr,
            "dfma_thread_inst": dfma, "dmul_thread_inst": dmul, "dadd_thread_inst": dadd,
            "fp64_thread_inst": (dfma + dmul + dadd) if None not in (dfma, dmul, dadd) else None,
            "fp64_pipe_warp_inst": g("sm__inst_executed_pipe_fp64.sum"), "warp_inst": g("smsp__inst_executed.sum"),
            "fp64_pipe_active_pct": g("sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active"),
            "issue_active_pct": g("smsp__issue_active.avg.pct_of_peak_sustained_active"),
            "l1_data_pipe_pct": g("l1tex__data_pipe_lsu_wavefronts.avg.pct_of_peak_sustained_elapsed"),
            "warps_active_pct": g("sm__warps_active.avg.pct_of_peak_sustained_active"),
            "registers": g("launch__registers_per_thread"),
        }
    os.makedirs(os.path.dirname(a.out) or ".", exist_ok=True)
    with open(a.out + ".md", "w") as fh:
        fh.write("\n".join(md) + "\n")
    js = {"workload": a.workload, "csrc_sha": csrc_sha(), "source": os.path.relpath(a.out + ".md", ROOT), "command": a.command,
          "kernels": kernels}
    with open(os.path.join(ROOT, "profiles", f"ncu_{a.workload}.json"), "w") as fh:
        json.dump(js, fh, indent=1)
        fh.write("\n")
    print("wrote", a.out + ".md", "and", f"profiles/ncu_{a.workload}.json")


if __name__ == "__main__":
    main()
