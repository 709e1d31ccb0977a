"""Write profiles/r02_fp64_ops.json from ncu's per-launch CSV of the search kernels.

bench.py reports the FP64 roofline of reco_search_kernel in executed FP64 lane-operations, a count only ncu can take
(predicated-on DADD + DMUL + DFMA thread instructions).  This module turns the CSV of

    ncu --metrics <METRICS below> --clock-control none -k regex:reco_search -c 12 --csv --log-file gpurun_out/ops_cfg2.csv \
        python bench.py --workload cfg2 --steps 3 --warmup 3 --no-cpu-baseline --no-extra-configs

(and the same for --workload cfg3) into per-solve counts, keyed by a hash of the kernel sources, so that bench.py can refuse a
stale count:

    python -m paper_2211_14346_b200.ncu_counts --csv gpurun_out/ops_cfg2.csv --workload cfg2 \
           --bench-json gpurun_out/ops_cfg2_plain.json --profile profiles/r02a_reco_search.md

--bench-json is the JSON line of the same bench.py command run WITHOUT ncu (it carries solves_per_launch).  Existing entries
of other kernels are kept if they were written for the same source hash.  Nothing here runs on the product path.
"""
from __future__ import annotations

import argparse
import csv
import hashlib
import json
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
OPS_FILE = os.path.join(ROOT, "profiles", "r02_fp64_ops.json")
KERNEL_SOURCES = ("paper_2211_14346_b200/csrc/hepf_reco.cu", "paper_2211_14346_b200/csrc/hepf_common.cuh")
METRICS = ("gpu__time_duration.sum,smsp__inst_executed.sum,sm__cycles_elapsed.avg,"
           "smsp__sass_thread_inst_executed_op_dadd_pred_on.sum,smsp__sass_thread_inst_executed_op_dmul_pred_on.sum,"
           "smsp__sass_thread_inst_executed_op_dfma_pred_on.sum,sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active,"
           "sm__issue_active.avg.pct_of_peak_sustained_elapsed,dram__bytes_read.sum,dram__bytes_write.sum,"
           "launch__registers_per_thread,sm__warps_active.avg.per_cycle_active")


def source_hash() -> str:
    h = hashlib.sha256()
    for rel in KERNEL_SOURCES:
        with open(os.path.join(ROOT, rel), "rb") as f:
            h.update(f.read())
    return h.hexdigest()


def parse_launches(path: str) -> dict:
    """{short kernel name: [ {metric: value in base units} per launch ]} from ncu's long-format CSV."""
    rows = [r for r in csv.reader(open(path, newline="")) if r]
    head = next(i for i, r in enumerate(rows) if "Kernel Name" in r and "Metric Name" in r)
    col = {n: i for i, n in enumerate(rows[head])}
    scale = {"ms": 1e-3, "us": 1e-6, "ns": 1e-9, "s": 1.0, "msecond": 1e-3, "usecond": 1e-6, "nsecond": 1e-9, "second": 1.0,
             "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "byte": 1.0}
    out: dict = {}
    for r in rows[head + 1:]:
        if len(r) <= col["Metric Value"]:
            continue
        m = re.search(r"reco_search_kernel<\(?(?:int\))?(\d+), \(?(?:int\))?(\d+)", r[col["Kernel Name"]])
        if not m:
            continue
        name = f"reco_search_kernel<{m.group(1)},{m.group(2)}>"
        lid = int(r[col["ID"]])
        launches = out.setdefault(name, {})
        val = float(r[col["Metric Value"]].replace(",", "")) * scale.get(r[col["Metric Unit"]], 1.0)
        launches.setdefault(lid, {})[r[col["Metric Name"]]] = val
    return {k: [v[i] for i in sorted(v)] for k, v in out.items()}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--csv", required=True)
    ap.add_argument("--bench-json", required=True, help="JSON line of the same bench.py command run without ncu")
    ap.add_argument("--workload", required=True)
    ap.add_argument("--profile", required=True, help="the profiles/*.md file that documents this capture")
    args = ap.parse_args()
    bench = json.loads(open(args.bench_json).read().strip().splitlines()[-1])
    kernel = bench["roofline"]["kernel"]
    solves = int(bench["roofline"]["solves_per_launch"])
    launches = parse_launches(args.csv).get(kernel)
    if not launches:
        raise SystemExit(f"no launch of {kernel} in {args.csv}")
    full = [l for l in launches if l.get("gpu__time_duration.sum", 0.0) > 0.5 * max(x["gpu__time_duration.sum"] for x in launches)]
    mean = lambda k: sum(l[k] for l in full) / len(full)   # noqa: E731
    entry = {
        "workload": args.workload, "profile": args.profile, "launches_averaged": len(full), "solves_per_launch": solves,
        "dadd": mean("smsp__sass_thread_inst_executed_op_dadd_pred_on.sum") / solves,
        "dmul": mean("smsp__sass_thread_inst_executed_op_dmul_pred_on.sum") / solves,
        "dfma": mean("smsp__sass_thread_inst_executed_op_dfma_pred_on.sum") / solves,
        "warp_instructions_per_solve": mean("smsp__inst_executed.sum") / solves,
        "ncu_gpu_time_ms": 1e3 * mean("gpu__time_duration.sum"),
        "ncu_sm__pipe_fp64_cycles_active_pct": mean("sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active"),
        "ncu_sm__issue_active_pct": mean("sm__issue_active.avg.pct_of_peak_sustained_elapsed"),
        "dram_bytes_per_launch": mean("dram__bytes_read.sum") + mean("dram__bytes_write.sum"),
        "registers_per_thread": mean("launch__registers_per_thread"),
        "warps_active_per_sm": mean("sm__warps_active.avg.per_cycle_active"),
    }
    sha = source_hash()
    try:
        d = json.load(open(OPS_FILE))
    except (OSError, ValueError):
        d = {}
    if d.get("source_sha256") != sha:
        d = {"source_sha256": sha, "kernels": {}, "algorithmic_fp64_ops_per_solve": d.get("algorithmic_fp64_ops_per_solve", {})}
    d["kernels"][kernel] = entry
    with open(OPS_FILE, "w") as f:
        json.dump(d, f, indent=1)
        f.write("\n")
    print(json.dumps({kernel: entry}, indent=1))


if __name__ == "__main__":
    main()
