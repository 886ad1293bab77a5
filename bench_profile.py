"""Ties the ncu figures bench.py reports to the CUDA sources they were measured on.

    # 1. on the GPU box, after `python bench.py --steps 2 --warmup 3` has exited 0 without ncu:
    ncu --set full --clock-control none --import-source on -k regex:k_ -o gpurun_out/r02_full -f \
        python bench.py --steps 1 --warmup 3 --no-cpu-baseline --no-e2e
    # 2. here:
    ncu -i gpurun_out/r02_full.ncu-rep --page raw --csv > gpurun_out/r02_full_raw.csv
    python bench_profile.py gpurun_out/r02_full_raw.csv --workload config3_batch16_central

Step 2 writes profiles/r02_ncu_kernels.json: per stage kernel the LAST captured launch's DRAM bytes (read + written),
thread instructions, warp instructions, duration, L2 hit rate, and `source_hash` = sha256 over
paper_1712_09434_b200/csrc/* and include/tpc_tracker.h.  bench.py reports `roofline.traffic` and the `alu` block
only while that hash equals the hash of the sources it runs on; otherwise it prints null (never a stale constant).
"""
from __future__ import annotations

import argparse
import csv
import glob
import hashlib
import json
import os
import sys

ROOT = os.path.dirname(os.path.abspath(__file__))
OUT = os.path.join(ROOT, "profiles", "r02_ncu_kernels.json")

# kernel name (substring) -> stage name of tpc_stage_name()
STAGE_OF = {"k_grid_build": "grid_build", "k_neighbours": "neighbour_finder", "k_clean": "cleaner",
            "k_seeds": "start_hits", "k_trk_chain": "tracklet_chain_fit", "k_trk_up": "tracklet_up_pass",
            "k_trk_refit": "tracklet_refit", "k_trk_finish": "tracklet_down_finish",
            "k_task_offsets": "ownership", "k_resolve": "ownership", "k_select_output": "selector_output",
            "k_order": "tracklet_queue_order", "k_merge": "merger_refit"}

METRICS = {
    "dram_read": "dram__bytes_read.sum", "dram_write": "dram__bytes_write.sum",
    "thread_inst": "smsp__thread_inst_executed.sum", "warp_inst": "smsp__inst_executed.sum",
    "lanes_per_inst": "smsp__thread_inst_executed_per_inst_executed.ratio",
    "duration_ns": "gpu__time_duration.sum", "l2_hit_pct": "lts__t_sector_hit_rate.pct",
    "issue_active_pct": "smsp__issue_active.avg.pct_of_peak_sustained_active",
}
UNIT_SCALE = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "ns": 1.0, "us": 1e3, "ms": 1e6, "s": 1e9,
              "usecond": 1e3, "msecond": 1e6, "nsecond": 1.0, "second": 1e9}


def source_hash() -> str:
    """sha256 over the CUDA sources and the C header, in sorted path order."""
    h = hashlib.sha256()
    files = sorted(glob.glob(os.path.join(ROOT, "paper_1712_09434_b200", "csrc", "*")))
    files.append(os.path.join(ROOT, "include", "tpc_tracker.h"))
    for f in files:
        if os.path.isfile(f):
            h.update(os.path.basename(f).encode())
            h.update(open(f, "rb").read())
    return h.hexdigest()[:16]


def parse_raw_csv(path):
    """Rows of `ncu --page raw --csv`: a header row, a units row, then one row per captured launch."""
    rows = list(csv.reader(open(path, newline="")))
    start = next(i for i, r in enumerate(rows) if "Kernel Name" in r)
    head, units = rows[start], rows[start + 1]
    col = {n: i for i, n in enumerate(head)}
    out = {}
    for r in rows[start + 2:]:
        if len(r) < len(head):
            continue
        name = r[col["Kernel Name"]]
        stage = next((s for k, s in STAGE_OF.items() if k in name), None)
        if stage is None:
            continue
        rec = {"kernel": name.split("(")[0]}
        for key, metric in METRICS.items():
            if metric not in col:
                continue
            txt = r[col[metric]].replace(",", "")
            try:
                v = float(txt)
            except ValueError:
                continue
            rec[key] = v * UNIT_SCALE.get(units[col[metric]].strip(), 1.0)
        if "thread_inst" not in rec and "warp_inst" in rec and "lanes_per_inst" in rec:
            rec["thread_inst"] = rec["warp_inst"] * rec["lanes_per_inst"]  # --set full carries the ratio, not the sum
        out.setdefault(stage, []).append(rec)
    return out


def main() -> int:
    ap = argparse.ArgumentParser()
    ap.add_argument("raw_csv")
    ap.add_argument("--workload", required=True, help="CONFIGS[...]['name'] of the bench run that was captured")
    ap.add_argument("--command", default="", help="the full ncu command, recorded in the summary")
    args = ap.parse_args()
    per_stage = parse_raw_csv(args.raw_csv)
    kernels = {}
    for stage, recs in per_stage.items():
        # a stage may be several kernels per step (the tracklet constructor): the kernels of the LAST captured step,
        # i.e. the last occurrence of every distinct kernel name, are summed
        last = {}
        for rec in recs:
            last[rec["kernel"]] = rec
        agg = {"kernels": sorted(last)}
        for key in ("dram_read", "dram_write", "thread_inst", "warp_inst", "duration_ns"):
            vals = [r[key] for r in last.values() if key in r]
            if vals:
                agg[key] = sum(vals)
        if "dram_read" in agg and "dram_write" in agg:
            agg["dram_bytes"] = agg["dram_read"] + agg["dram_write"]
        top = max(last.values(), key=lambda r: r.get("duration_ns", 0.0))
        for key in ("l2_hit_pct", "issue_active_pct"):
            if key in top:
                agg[key + "_of_longest"] = top[key]
        kernels[stage] = agg
    doc = {"workload": args.workload, "source_hash": source_hash(), "command": args.command,
           "note": "cold-cache, serialised ncu replay: durations are NOT bench values; bytes and instruction counts "
                   "are per launch", "kernels": kernels}
    json.dump(doc, open(OUT, "w"), indent=1)
    print(json.dumps(doc, indent=1))
    return 0


if __name__ == "__main__":
    sys.exit(main())
