"""profiles/inst_counts.json: warp-instructions one chain-step executes, per workload, taken from ncu launch lists.

bench.py multiplies such a count by the chain-steps/s it measures to report the issue-slot fraction (`roofline.frac`).
A count is only meaningful for the kernel text and the launch geometry it was captured on, so every entry records both:

  source_id  FNV-1a-64 of the run-time compiled source of its kernel family (sa_kernel_source_id; `tree_source_id`
             computes the same number from the files under csrc/)
  geometry   chains per GPU and the launch shape the handle reported during the capture (`GEOMETRY_KEYS`)

`stale_reason(entry, ...)` says why an entry does not apply to a running handle (None if it does); bench.py then reports
`frac: null` with that reason.  tests/test_telemetry.py compares every entry's source_id with the tree, so a kernel
change without a fresh capture fails on the CPU box.

    python -m paper_2506_19866_b200.inst_counts update W profiles/r3_W_launches.csv profiles/r3_W_bench.json

rewrites workload W's entry from an ncu launch list (`--metrics gpu__time_duration.sum,smsp__inst_executed.sum --csv`) and
the JSON line of the same bench command run without ncu (its `config` gives the geometry and the chain-steps per launch).
"""
from __future__ import annotations

import csv
import json
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
PATH = os.path.join(ROOT, "profiles", "inst_counts.json")
CSRC = os.path.join(HERE, "csrc")
# kernel name -> (family number of sa_kernel_source_id, the files whose text NVRTC compiles, as build.py joins them)
KERNELS = {"tsa_run_static": (2, ("sa_static_params.h", "sa_static_kernel.cu")),
           "tsa_run_dense": (3, ("sa_dense_params.h", "sa_dense_kernel.cu")),
           "tsp_run": (4, ("sap_params.h", "sap_kernel.cu"))}
GEOMETRY_KEYS = ("variant", "threads_per_cta", "chains_per_cta", "grid", "smem_bytes", "static_regs", "team_warps",
                 "lanes_per_chain", "node_slots", "edge_slots", "regs", "ctas_per_sm", "sm_count")


def fnv1a64(data: bytes) -> int:
    h = 0xCBF29CE484222325
    for b in data:
        h = ((h ^ b) * 0x100000001B3) & 0xFFFFFFFFFFFFFFFF
    return h


def tree_source_id(kernel: str) -> str:
    parts = []
    for name in KERNELS[kernel][1]:
        with open(os.path.join(CSRC, name)) as f:
            parts.append(f.read())
    return f"{fnv1a64(chr(10).join(parts).encode()):016x}"


def load() -> dict:
    try:
        with open(PATH) as f:
            return json.load(f)
    except Exception:
        return {}


def geometry_of(chains: int, launch: dict) -> dict:
    g = {"chains": int(chains)}
    g.update({k: int(launch[k]) for k in GEOMETRY_KEYS if k in launch})
    return g


def stale_reason(entry: dict, kernel: str, library_source_id: str, chains: int, launch: dict):
    """None if `entry` (one workload of inst_counts.json) was captured on this kernel text and launch geometry."""
    if not entry or not entry.get("warp_inst_per_chain_step"):
        return "no instruction count for this workload in profiles/inst_counts.json"
    if entry.get("kernel") != kernel:
        return f"the instruction count is of kernel {entry.get('kernel')}, this run launches {kernel}"
    if entry.get("source_id") != library_source_id:
        return (f"stale instruction count: captured on kernel source {entry.get('source_id')}, "
                f"the loaded library carries {library_source_id}")
    want, have = entry.get("geometry") or {}, geometry_of(chains, launch)
    diff = {k: (v, have.get(k)) for k, v in want.items() if have.get(k) != v}
    if not want or diff:
        return f"stale instruction count: captured on another launch geometry {diff or '(none recorded)'}"
    return None


def update(workload: str, launches_csv: str, bench_json: str) -> dict:
    with open(bench_json) as f:
        line = [ln for ln in f.read().splitlines() if ln.startswith("{")][-1]
    cfg = json.loads(line)["config"]
    rows = []
    with open(launches_csv, newline="") as f:
        for row in csv.reader(ln for ln in f if ln.startswith('"')):
            rows.append(row)
    head = rows[0]
    col = {name: head.index(name) for name in ("ID", "Kernel Name", "Metric Name", "Metric Value")}
    per_launch = {}
    for row in rows[1:]:
        if row[col["Kernel Name"]] in KERNELS:
            per_launch.setdefault(row[col["ID"]], {"kernel": row[col["Kernel Name"]]})[row[col["Metric Name"]]] = float(row[col["Metric Value"]])
    last = per_launch[max(per_launch, key=int)]                      # the timed launch: the last full-length one
    chain_steps = cfg["chains_per_gpu"] * cfg["sa_steps"]
    launch = dict(cfg.get("launch") or cfg["paper"])
    entry = {"kernel": last["kernel"],
             "warp_inst_per_chain_step": round(last["smsp__inst_executed.sum"] / chain_steps, 1),
             "source": f"{os.path.relpath(launches_csv, ROOT)} ({last['smsp__inst_executed.sum']:.3e} warp-instructions / "
                       f"{chain_steps} chain-steps, {last['gpu__time_duration.sum'] * 1e-6:.3f} ms)",
             "source_id": tree_source_id(last["kernel"]),
             "geometry": geometry_of(cfg["chains_per_gpu"], launch)}
    data = load()
    keep = {k: v for k, v in data.get(workload, {}).items() if k.startswith("smem_")}
    entry.update(keep)
    data[workload] = entry
    with open(PATH, "w") as f:
        json.dump(data, f, indent=1)
        f.write("\n")
    return entry


if __name__ == "__main__":
    if len(sys.argv) == 5 and sys.argv[1] == "update":
        print(json.dumps(update(sys.argv[2], sys.argv[3], sys.argv[4]), indent=1))
    else:
        print(__doc__)
        sys.exit(2)
