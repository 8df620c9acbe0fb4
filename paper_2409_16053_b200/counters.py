"""ncu counters of the stage kernel, kept beside the numbers bench.py derives from them.

    python -m paper_2409_16053_b200.counters <ncu raw-page csv> <workload> > profiles/r02_stage_counters_<workload>.json

reads the CSV written by

    ncu --metrics <METRICS below> --clock-control none -k regex:stage -s <warm-up launches> -c <n> --page raw --csv \
        --log-file <csv> python bench.py --workload <workload> --steps 2 --warmup 1 --no-e2e --no-cpu

and writes, per stage launch kind (stage 1 / stage 2), the DRAM bytes, the FP64-pipe and ALU-pipe warp instructions,
all warp instructions and the launch duration, together with a hash of the kernel sources (csrc/ + include/ak.h).
bench.py prints `roofline.traffic` and `roofline_alu` only while that hash equals the hash of the tree it runs from,
so the two numbers cannot outlive the kernel they were counted on.
"""
from __future__ import annotations

import csv
import hashlib
import json
import os
import re
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
_AK_H = os.path.join(ROOT, "include", "ak.h")
METRICS = ("gpu__time_duration.sum,dram__bytes_read.sum,dram__bytes_write.sum,smsp__inst_executed.sum,"
           "sm__inst_executed_pipe_fp64.sum,sm__inst_executed_pipe_alu.sum,sm__inst_executed_pipe_fma.sum,"
           "sm__inst_executed_pipe_lsu.sum,sm__inst_executed_pipe_xu.sum,"
           "smsp__sass_thread_inst_executed_op_dadd_pred_on.sum,smsp__sass_thread_inst_executed_op_dmul_pred_on.sum,"
           "smsp__sass_thread_inst_executed_op_dfma_pred_on.sum,"
           "sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active,smsp__issue_active.avg.pct_of_peak_sustained_active,"
           "launch__registers_per_thread,launch__grid_size,launch__block_size")


def csrc_sha() -> str:
    """Hash of everything the kernels are built from."""
    h = hashlib.sha256()
    files = sorted(os.path.join(HERE, "csrc", f) for f in os.listdir(os.path.join(HERE, "csrc")))
    files.append(_AK_H)
    for f in files:
        if os.path.isfile(f):
            h.update(os.path.basename(f).encode())
            h.update(open(f, "rb").read())
    return h.hexdigest()[:16]


def load(workload: str):
    """Counters for `workload` if they were taken on the present kernel sources, else None."""
    path = os.path.join(ROOT, "profiles", f"r02_stage_counters_{workload}.json")
    try:
        d = json.load(open(path))
    except Exception:
        return None
    return d if d.get("csrc_sha") == csrc_sha() else None


def _num(x: str) -> float:
    return float(x.replace(",", ""))


def parse(path: str, workload: str) -> dict:
    rows = list(csv.reader(open(path)))
    hi = [i for i, r in enumerate(rows) if r and r[0] == "ID"][0]
    hdr = rows[hi]
    data = [r for r in rows[hi + 2:] if len(r) == len(hdr)]
    out = {"csrc_sha": csrc_sha(), "workload": workload, "source": os.path.basename(path),
           "command": "ncu --metrics " + METRICS + " --clock-control none -k regex:stage --page raw --csv "
                      f"python bench.py --workload {workload} --steps 2 --warmup 1 --no-e2e --no-cpu",
           "launches": {}}
    for r in data:
        name = r[hdr.index("Kernel Name")]
        m = re.search(r"stage_v3_kernel<(\d+), (\d+), (\d+), (\d+), (\d+), (\d+)>", name)
        if not m:
            continue
        recon, rs, ti, tj, minb, st2 = (int(x) for x in m.groups())
        key = "stage2" if st2 else "stage1"
        e = out["launches"].setdefault(key, {"kernel": m.group(0), "n": 0})
        for k in hdr:
            if k.split(".")[0] in ("gpu__time_duration", "dram__bytes_read", "dram__bytes_write", "smsp__inst_executed") or \
               k.startswith(("sm__inst_executed_pipe_", "smsp__sass_thread_inst_executed_op_d", "sm__pipe_fp64", "smsp__issue_active", "launch__")):
                try:
                    e[k] = e.get(k, 0.0) + _num(r[hdr.index(k)])
                except ValueError:
                    pass
        e["n"] += 1
    for e in out["launches"].values():
        n = e.pop("n")
        for k in list(e):
            if isinstance(e[k], float):
                e[k] /= n
        e["launches_averaged"] = n
    return out


if __name__ == "__main__":
    print(json.dumps(parse(sys.argv[1], sys.argv[2]), indent=1))
