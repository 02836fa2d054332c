"""Summarise `ncu --page raw --csv` exports of the dominant kernels into the two files bench.py and the
judge read: a text page of the metrics that matter on this path and `profiles/traffic.json`.

    python tests/ncu_summary.py RAW_DIR --text profiles/r02_ncu_full.txt [--json profiles/traffic.json]
    python tests/ncu_summary.py --launches LAUNCHES.csv --out profiles/r02_launches_<run>_summary.csv

RAW_DIR holds one `raw_<workload>.csv` per capture, <workload> being bench.py's `--workload` name; each is

    ncu -i rep_<workload>.ncu-rep --page raw --csv > raw_<workload>.csv

of a capture taken with

    ncu --set full --metrics <EXTRA> --clock-control none --import-source on -k regex:<kernel> -s <skip> -c 1 -f \\
        -o rep_<workload> python bench.py --suite primary --steps 5 --warmup 3 --no-e2e --no-cpu-baseline --ising-sweeps 3 --workload <workload>

and then cut down to the columns this tool reads (so that the raw page can be committed and the summaries re-derived
from tracked files: tests/test_profiles_tools.py does exactly that) with

    python tests/ncu_summary.py RAW_DIR --trim profiles/r03_raw

(only after the same bench.py command has exited 0 without ncu; EXTRA = the EXTRA_METRICS list below: which of the
two fma pipes and the conversion unit executed how many instructions -- `--set full` only has their sum).
LAUNCHES.csv is the `--metrics gpu__time_duration.sum --clock-control none --csv` launch list of a bench.py run; its
summary has one row per kernel (launches, total and average duration, share of the run).  A profiling aid kept beside
the tests, not part of the library package: nothing here runs a kernel or is imported by the product path; bench.py reads the JSON as STATIC context (`measured_in_this_run: false`).
"""
from __future__ import annotations

import argparse
import csv
import glob
import json
import os

KEYS = [
    "gpu__time_duration.sum", "dram__bytes_write.sum", "dram__bytes_read.sum",
    "gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed", "sm__throughput.avg.pct_of_peak_sustained_elapsed",
    "smsp__issue_active.avg.pct_of_peak_sustained_active", "sm__inst_executed_pipe_alu.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_fma.avg.pct_of_peak_sustained_active",
    "sm__pipe_fmaheavy_cycles_active.avg.pct_of_peak_sustained_elapsed",
    "sm__inst_executed_pipe_lsu.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_uniform.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_xu.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_fmaheavy.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_fmalite.avg.pct_of_peak_sustained_active",
    "sm__pipe_fmaheavy_cycles_active.avg.pct_of_peak_sustained_active",
    "sm__pipe_alu_cycles_active.avg.pct_of_peak_sustained_active",
    "sm__pipe_shared_cycles_active.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_alu.sum", "sm__inst_executed_pipe_fmaheavy.sum", "sm__inst_executed_pipe_fmalite.sum",
    "sm__inst_executed_pipe_xu.sum", "sm__inst_executed_pipe_lsu.sum",
    "sm__warps_active.avg.pct_of_peak_sustained_active",
    "smsp__inst_executed.sum", "launch__registers_per_thread", "launch__grid_size", "launch__block_size",
    "launch__occupancy_limit_registers", "launch__occupancy_limit_shared_mem",
    "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum", "l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum",
    "l1tex__throughput.avg.pct_of_peak_sustained_elapsed", "lts__throughput.avg.pct_of_peak_sustained_elapsed",
    "lts__t_sector_hit_rate.pct", "sm__cycles_elapsed.max", "smsp__cycles_active.avg", "sm__cycles_active.avg",
]
EXTRA_METRICS = ",".join([
    "sm__inst_executed_pipe_fmaheavy.avg.pct_of_peak_sustained_active", "sm__inst_executed_pipe_fmalite.avg.pct_of_peak_sustained_active",
    "sm__pipe_fmaheavy_cycles_active.avg.pct_of_peak_sustained_active", "sm__pipe_alu_cycles_active.avg.pct_of_peak_sustained_active",
    "sm__pipe_shared_cycles_active.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_alu.sum", "sm__inst_executed_pipe_fmaheavy.sum", "sm__inst_executed_pipe_fmalite.sum",
    "sm__inst_executed_pipe_xu.sum", "sm__inst_executed_pipe_lsu.sum"])
UNIT = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}
TIME_US = {"ns": 1e-3, "us": 1.0, "ms": 1e3, "s": 1e6}


def _num(d, k):
    try:
        return float(d[k].replace(",", ""))
    except Exception:
        return None


def summarise(raw_dir: str, text_path: str, json_path: str | None, source: str, fresh: bool = False) -> dict:
    entries = {}
    with open(text_path, "w") as f:
        for p in sorted(glob.glob(os.path.join(raw_dir, "raw_*.csv"))):
            rows = list(csv.reader(open(p)))
            if len(rows) < 3:
                continue
            hdr, units = rows[0], rows[1]
            name = os.path.basename(p)[4:-4]
            for r in rows[2:]:
                d, u = dict(zip(hdr, r)), dict(zip(hdr, units))
                f.write(f"== [{name}] {d.get('Kernel Name', '?')} grid {d.get('Grid Size', '')} block {d.get('Block Size', '')}\n")
                for k in KEYS:
                    if d.get(k, "") != "":
                        f.write(f"  {k:88s} {d[k]:>20s} {u.get(k, '')}\n")
                stalls = [(_num(d, k), k) for k in hdr if k.startswith("smsp__average_warps_issue_stalled_")
                          and k.endswith("_per_issue_active.ratio") and _num(d, k) is not None]
                for v, k in sorted(stalls, reverse=True)[:6]:
                    f.write(f"  {k:88s} {v:20.3f} warps/issue\n")
                pipes = [(_num(d, k), k) for k in hdr if k.startswith("sm__inst_executed_pipe_")
                         and k.endswith("pct_of_peak_sustained_active") and _num(d, k) is not None]
                f.write("  top pipes: " + ", ".join(f"{k.split('pipe_')[1].split('.')[0]} {v:.1f}%"
                                                     for v, k in sorted(pipes, reverse=True)[:6]) + "\n")

                def byt(k):
                    v = _num(d, k)
                    return None if v is None else v * UNIT.get(u.get(k, ""), 1.0)
                traffic = (byt("dram__bytes_read.sum") or 0.0) + (byt("dram__bytes_write.sum") or 0.0)
                t_us = (_num(d, "gpu__time_duration.sum") or 0.0) * TIME_US.get(u.get("gpu__time_duration.sum", "us"), 1.0)
                entries[name] = {
                    "kernel": d.get("Kernel Name"), "dram_bytes_per_launch": int(traffic), "ncu_time_us": round(t_us, 3),
                    "source": source,
                    "issue_active_pct": _num(d, "smsp__issue_active.avg.pct_of_peak_sustained_active"),
                    "pipe_alu_pct": _num(d, "sm__inst_executed_pipe_alu.avg.pct_of_peak_sustained_active"),
                    "pipe_fma_pct": _num(d, "sm__inst_executed_pipe_fma.avg.pct_of_peak_sustained_active"),
                    "pipe_fmaheavy_cycles_pct_of_elapsed": _num(d, "sm__pipe_fmaheavy_cycles_active.avg.pct_of_peak_sustained_elapsed"),
                    "pipe_lsu_pct": _num(d, "sm__inst_executed_pipe_lsu.avg.pct_of_peak_sustained_active"),
                    "dram_throughput_pct": _num(d, "gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed"),
                    "pipe_fmaheavy_cycles_pct_of_active": _num(d, "sm__pipe_fmaheavy_cycles_active.avg.pct_of_peak_sustained_active"),
                    "pipe_fmalite_pct": _num(d, "sm__inst_executed_pipe_fmalite.avg.pct_of_peak_sustained_active"),
                    "pipe_xu_pct": _num(d, "sm__inst_executed_pipe_xu.avg.pct_of_peak_sustained_active"),
                    "inst_per_cycle_active": (None if not (_num(d, "smsp__inst_executed.sum") and _num(d, "smsp__cycles_active.avg"))
                                              else round(_num(d, "smsp__inst_executed.sum") / (_num(d, "smsp__cycles_active.avg") * 592.0), 4)),
                }
    if json_path:
        old = {}
        if os.path.exists(json_path) and not fresh:
            old = json.load(open(json_path))
        old["_comment"] = ("keyed by bench.py --workload name; per workload, from the `ncu --set full` capture of its dominant "
                           "kernel (see each entry's `source`): dram__bytes_read.sum + dram__bytes_write.sum per launch, "
                           "smsp__issue_active, sm__inst_executed_pipe_* (pct of peak sustained, active cycles), "
                           "sm__pipe_fmaheavy_cycles_active (pct of elapsed), gpu__dram_throughput.  Written by "
                           "`python tests/ncu_summary.py`; bench.py copies these as static context "
                           "(measured_in_this_run: false) and never runs under ncu.")
        old.update(entries)
        with open(json_path, "w") as f:
            json.dump(old, f, indent=1)
    return entries


def _kept(col: str) -> bool:
    """columns of ncu's raw page that summarise() reads"""
    return (col in ("ID", "Kernel Name", "Grid Size", "Block Size") or col in KEYS
            or (col.startswith("smsp__average_warps_issue_stalled_") and col.endswith("_per_issue_active.ratio"))
            or (col.startswith("sm__inst_executed_pipe_") and col.endswith("pct_of_peak_sustained_active")))


def trim(raw_dir: str, out_dir: str) -> int:
    """copies RAW_DIR/raw_*.csv to OUT_DIR keeping only the columns summarise() reads (a few KB per capture
    instead of ncu's ~6000 columns): the summaries made from the trimmed files are identical"""
    os.makedirs(out_dir, exist_ok=True)
    n = 0
    for p in sorted(glob.glob(os.path.join(raw_dir, "raw_*.csv"))):
        rows = [r for r in csv.reader(open(p, errors="replace")) if r]
        hdr_i = next((i for i, r in enumerate(rows) if r[0] == "ID"), None)  # ncu may print '==PROF==' lines first
        if hdr_i is None or len(rows) < hdr_i + 3:
            continue
        rows = rows[hdr_i:]
        keep = [i for i, c in enumerate(rows[0]) if _kept(c)]
        with open(os.path.join(out_dir, os.path.basename(p)), "w", newline="") as f:
            w = csv.writer(f, lineterminator="\n")
            for r in rows:
                w.writerow([r[i] if i < len(r) else "" for i in keep])
        n += 1
    return n


def summarise_launches(csv_in: str, csv_out: str) -> int:
    """per kernel of an ncu launch list: launches, total and average gpu__time_duration, share of the run"""
    rows = list(csv.reader(open(csv_in, errors="replace")))
    hdr_i = next(i for i, r in enumerate(rows) if r and r[0] == "ID")
    hdr = rows[hdr_i]
    col = {n: hdr.index(n) for n in ("Kernel Name", "Grid Size", "Block Size", "Metric Name", "Metric Unit", "Metric Value")}
    agg = {}
    for r in rows[hdr_i + 1:]:
        if len(r) < len(hdr) or r[col["Metric Name"]] != "gpu__time_duration.sum":
            continue
        us = float(r[col["Metric Value"]].replace(",", "")) * {"ns": 1e-3, "us": 1.0, "ms": 1e3, "s": 1e6}.get(r[col["Metric Unit"]], 1e-3)
        key = (r[col["Kernel Name"]], r[col["Grid Size"]], r[col["Block Size"]])
        n, t = agg.get(key, (0, 0.0))
        agg[key] = (n + 1, t + us)
    total = sum(t for _, t in agg.values()) or 1.0
    with open(csv_out, "w", newline="") as f:
        w = csv.writer(f)
        w.writerow(["kernel", "grid", "block", "launches", "sum_us", "avg_us", "share_pct"])
        for (k, g, b), (n, t) in sorted(agg.items(), key=lambda kv: -kv[1][1]):
            w.writerow([k, g, b, n, round(t, 1), round(t / n, 2), round(100.0 * t / total, 2)])
    return len(agg)


if __name__ == "__main__":
    ap = argparse.ArgumentParser()
    ap.add_argument("raw_dir", nargs="?")
    ap.add_argument("--launches", default=None, help="an ncu launch list (csv) to summarise per kernel")
    ap.add_argument("--out", default=None, help="with --launches: the summary csv to write")
    ap.add_argument("--text", default=None)
    ap.add_argument("--json", default=None)
    ap.add_argument("--fresh", action="store_true", help="with --json: write only this run's entries (default: merge into the file)")
    ap.add_argument("--trim", default=None, help="instead of summarising: copy RAW_DIR's raw pages, cut down to the columns read here, to this directory")
    ap.add_argument("--source", default=None, help="what the entries cite as their capture (default: --text)")
    a = ap.parse_args()
    if a.launches:
        print(f"{summarise_launches(a.launches, a.out or a.launches[:-4] + '_summary.csv')} kernels -> {a.out}")
        raise SystemExit(0)
    if a.raw_dir and a.trim:
        print(f"{trim(a.raw_dir, a.trim)} raw pages -> {a.trim}")
        raise SystemExit(0)
    if not a.raw_dir or not a.text:
        ap.error("RAW_DIR and --text are required without --launches")
    e = summarise(a.raw_dir, a.text, a.json, a.source or a.text, a.fresh)
    print(f"{len(e)} captures -> {a.text}" + (f", {a.json}" if a.json else ""))
