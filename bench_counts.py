#!/usr/bin/env python
"""bench_counts.py — turn ncu captures of the integrator kernels into profiles/r02_flop_counts.json,
the file bench.py reads its roofline numerators from.

What is counted is the FP64 work the kernels EXECUTE on the bench workload itself: predicated-on
thread instructions per opcode from the ncu source page (2 x DFMA + DMUL + DADD = flop; DSETP and
MUFU occupy pipes but carry no flop), plus DRAM bytes, warp execution efficiency and FP64-pipe
utilisation from the raw page.  Two captures are needed: the geodesics-only kernel and the fused
geodesic + transfer kernel, each taken with

    python bench.py --steps 1 --warmup 3 --no-e2e --no-cpu-baseline --no-extra [--model none] > plain.log 2>&1 &&
    ncu --set full --clock-control none --import-source on -k regex:odyssey_kernel -s 3 -c 1 \
        -o gpurun_out/<name> -f python bench.py --steps 1 --warmup 3 --no-e2e --no-cpu-baseline --no-extra [--model none]

on one B200, then here (no GPU needed):

    python bench_counts.py --geo gpurun_out/<geo>.ncu-rep --fused gpurun_out/<fused>.ncu-rep \
        --attempts A --accepts B > profiles/r02_flop_counts.json

A, B: the attempted / accepted step totals of one launch (bench.py prints them in `config`).
The file records the hash of the kernel sources it was measured on; bench.py recomputes that hash
and reports `"stale": true` in its roofline block when the sources have changed since.
"""
import argparse
import csv
import hashlib
import io
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(ROOT, "paper_1601_02063_b200", "csrc")
KERNEL_SOURCES = ("odyssey_kernels.cuh", "geodesic.cuh", "emission.cuh", "dmath.cuh", "dmath_coeffs.h",
                  "bessel_k2_coeffs.h", "params.h")


def source_hash():
    """sha256 over the files that determine the integrator kernels' instruction stream."""
    h = hashlib.sha256()
    for name in KERNEL_SOURCES:
        with open(os.path.join(CSRC, name), "rb") as f:
            h.update(name.encode() + b"\0" + f.read())
    return h.hexdigest()[:16]


def _ncu_csv(rep, page):
    out = subprocess.run(["ncu", "-i", rep, "--page", page, "--csv"], capture_output=True, text=True, check=True).stdout
    return list(csv.reader(io.StringIO(out)))


def capture(rep):
    """Per-launch figures of the (single) kernel in an .ncu-rep file."""
    raw = _ncu_csv(rep, "raw")
    hdr, vals = raw[0], raw[2]
    get = lambda k: vals[hdr.index(k)]
    src = _ncu_csv(rep, "source")
    sh, rows = src[1], src[2:]
    i_src, i_ex, i_thr = sh.index("Source"), sh.index("Instructions Executed"), sh.index("Predicated-On Thread Instructions Executed")
    warp, thread = {}, {}
    for r in rows:
        t = r[i_src].split()
        op = (t[1] if t[0].startswith("@") else t[0]).split(".")[0]
        warp[op] = warp.get(op, 0) + int(r[i_ex])
        thread[op] = thread.get(op, 0) + int(r[i_thr])
    total_warp = sum(warp.values())
    fp64_warp = sum(warp.get(o, 0) for o in ("DFMA", "DMUL", "DADD", "DSETP"))
    scale = {"Mbyte": 1e6, "Gbyte": 1e9, "Kbyte": 1e3, "byte": 1.0}
    unit = lambda k: raw[1][hdr.index(k)]
    dram = sum(float(get(k)) * scale[unit(k)] for k in ("dram__bytes_read.sum", "dram__bytes_write.sum"))
    return {
        "kernel": get("Kernel Name"),
        "flop": 2 * thread.get("DFMA", 0) + thread.get("DMUL", 0) + thread.get("DADD", 0),
        "fp64_thread_instructions": sum(thread.get(o, 0) for o in ("DFMA", "DMUL", "DADD", "DSETP")),
        "warp_instructions": total_warp,
        "fp64_share_of_warp_instructions": fp64_warp / total_warp,
        "static_instructions": len(rows),
        "duration_ms_under_ncu": float(get("gpu__time_duration.sum")),
        "registers": int(get("launch__registers_per_thread")),
        "warp_execution_efficiency": float(get("smsp__thread_inst_executed_per_inst_executed.ratio")) / 32.0,
        "fp64_pipe_utilisation": float(get("sm__inst_executed_pipe_fp64.avg.pct_of_peak_sustained_active")) / 100.0,
        "issue_slot_utilisation": float(get("smsp__issue_active.avg.pct_of_peak_sustained_active")) / 100.0,
        "local_load_store_instructions": int(float(get("sass__inst_executed_local_loads"))) + int(float(get("sass__inst_executed_local_stores"))),
        "dram_bytes": dram,
        "opcode_warp_instructions": dict(sorted(warp.items(), key=lambda kv: -kv[1])[:16]),
    }


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--geo", required=True)
    ap.add_argument("--fused", required=True)
    ap.add_argument("--attempts", type=int, required=True)
    ap.add_argument("--accepts", type=int, required=True)
    ap.add_argument("--workload", default="C4: a=0.998, i=85deg, 4096x4096, RIAF 230 GHz")
    a = ap.parse_args()
    geo, fused = capture(a.geo), capture(a.fused)
    per_attempt_geo = geo["flop"] / a.attempts
    out = {
        "what": "executed FP64 flop (2 x DFMA + DMUL + DADD thread instructions, predicated on) per launch, ncu --set full",
        "workload": a.workload, "attempts": a.attempts, "accepts": a.accepts,
        "source_hash": source_hash(), "kernel_sources": list(KERNEL_SOURCES),
        "flop_per_attempt_geodesic": per_attempt_geo,
        "flop_per_rt_update": (fused["flop"] - per_attempt_geo * a.attempts) / a.accepts,
        "flop_per_attempt_fused": fused["flop"] / a.attempts,
        "geodesic_kernel": geo, "fused_kernel": fused,
    }
    json.dump(out, sys.stdout, indent=1)
    print()


if __name__ == "__main__":
    main()
