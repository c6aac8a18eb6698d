"""Turn an ncu report into one record of profiles/ncu_kernels.json, the file bench.py reads
its `roofline.traffic` and `roofline.executed_fp32_frac` from (so that no profiler figure is
pasted into source code).  Runs here, without a GPU:

    python -m paper_2501_04456_b200.ncu_summary REPORT.ncu-rep --kernel k_pair_force_rows \
        --workload C3 --start-step 0 --path list --command "<the committed ncu command>"

A record: kernel, workload, start_step, path (force path: list / cells / tile), source_hash
(content hash of csrc/ + lv.h at capture time), duration_us, dram_bytes (read + write per
launch), lts_bytes, thread-instruction counts fadd / fmul / ffma (+ the packed f32x2 forms
counted by ncu as two), sm_cycles, n_sms, issue_active_pct, warps_active_pct, registers.
"""
from __future__ import annotations

import argparse
import csv
import hashlib
import json
import os
import subprocess

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
OUT = os.path.join(ROOT, "profiles", "ncu_kernels.json")


def source_hash():
    h = hashlib.sha256()
    base = os.path.join(ROOT, "paper_2501_04456_b200", "csrc")
    for f in sorted(os.listdir(base)):
        with open(os.path.join(base, f), "rb") as fh:
            h.update(f.encode() + b"\0" + fh.read())
    with open(os.path.join(ROOT, "include", "lv.h"), "rb") as fh:
        h.update(fh.read())
    return h.hexdigest()[:16]


def raw_metrics(report, kernel):
    out = subprocess.run(["ncu", "-i", report, "--page", "raw", "--csv"], capture_output=True, text=True).stdout
    rows = list(csv.reader(out.splitlines()))
    hdr, units = rows[0], rows[1]
    kcol = hdr.index("Kernel Name")
    for r in rows[2:]:
        if kernel in r[kcol]:
            return {h: (u, v) for h, u, v in zip(hdr, units, r)}
    raise SystemExit(f"no launch of {kernel} in {report}")


def sass_flops(report, kernel):
    """FP32 flop per launch from the SASS page (predicated-on thread instructions by opcode):
    FADD + FMUL + 2 FFMA + 2 (FADD2 + FMUL2) + 4 FFMA2 -- ncu's op_fadd/fmul/ffma counters do
    not see the packed f32x2 forms."""
    out = subprocess.run(["ncu", "-i", report, "--page", "source", "--csv", "-k", "regex:" + kernel],
                         capture_output=True, text=True).stdout
    rows = list(csv.reader(out.splitlines()))
    k = next(i for i, r in enumerate(rows) if r and r[0] == "Address")
    hdr = rows[k]
    isrc, it = hdr.index("Source"), hdr.index("Predicated-On Thread Instructions Executed")
    w = {"FADD": 1, "FMUL": 1, "FFMA": 2, "FADD2": 2, "FMUL2": 2, "FFMA2": 4}
    ops, flops = {}, 0.0
    for r in rows[k + 1:]:
        if len(r) <= it or r[0] == "Address" or not r[0].startswith("0x"):
            if r and r[0] == "Kernel Name":
                break                       # next launch of the report
            continue
        tok = r[isrc].split()
        op = (tok[1] if tok[0].startswith("@") else tok[0]).split(".")[0]
        if op in w:
            ops[op] = ops.get(op, 0) + int(r[it])
            flops += w[op] * int(r[it])
    return flops, ops


def num(m, key, scale_units=True):
    u, v = m[key]
    x = float(v.replace(",", ""))
    if scale_units:
        for pre, f in (("K", 1e3), ("M", 1e6), ("G", 1e9), ("T", 1e12)):
            if u.startswith(pre) and u not in ("Mhz", "Ghz"):
                x *= f
    return x


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("report")
    ap.add_argument("--kernel", required=True)
    ap.add_argument("--workload", required=True)
    ap.add_argument("--start-step", type=int, required=True)
    ap.add_argument("--path", required=True)
    ap.add_argument("--command", default="")
    ap.add_argument("--source-hash", default=None, help="hash at capture time if the sources moved on since")
    a = ap.parse_args()
    m = raw_metrics(a.report, a.kernel)
    cyc = num(m, "sm__cycles_elapsed.avg")
    rec = {
        "kernel": a.kernel, "workload": a.workload, "start_step": a.start_step, "path": a.path,
        "source_hash": a.source_hash or source_hash(), "report": os.path.basename(a.report), "command": a.command,
        "duration_us": num(m, "gpu__time_duration.sum", False) * {"us": 1.0, "ms": 1e3, "ns": 1e-3}[m["gpu__time_duration.sum"][0]],
        "dram_bytes": num(m, "dram__bytes_read.sum") + num(m, "dram__bytes_write.sum"),
        "lts_bytes": 32.0 * num(m, "lts__t_sectors.sum") if "lts__t_sectors.sum" in m else None,
        # thread instructions per launch (ncu reports them per elapsed SM cycle, summed over the GPU)
        "fadd": num(m, "smsp__sass_thread_inst_executed_op_fadd_pred_on.sum.per_cycle_elapsed") * cyc,
        "fmul": num(m, "smsp__sass_thread_inst_executed_op_fmul_pred_on.sum.per_cycle_elapsed") * cyc,
        "ffma": num(m, "smsp__sass_thread_inst_executed_op_ffma_pred_on.sum.per_cycle_elapsed") * cyc,
        "sm_cycles": cyc,
        "n_sms": int(num(m, "device__attribute_multiprocessor_count")),
        "warp_instructions": num(m, "smsp__inst_executed.sum"),
        "issue_active_pct": num(m, "smsp__issue_active.avg.pct_of_peak_sustained_active"),
        "warps_active_pct": num(m, "sm__warps_active.avg.pct_of_peak_sustained_active"),
        "l1_data_pipe_pct": num(m, "l1tex__data_pipe_lsu_wavefronts.avg.pct_of_peak_sustained_elapsed"),
        "registers": int(num(m, "launch__registers_per_thread")),
    }
    # executed FP32 in flop terms per clock / (SMs x 128 lanes x 2), opcodes from the SASS page
    flops, ops = sass_flops(a.report, a.kernel)
    rec["fp32_flop"] = flops
    rec["fp32_thread_inst_by_opcode"] = ops
    rec["executed_fp32_frac"] = flops / cyc / (rec["n_sms"] * 128 * 2)
    recs = []
    if os.path.exists(OUT):
        with open(OUT) as f:
            recs = json.load(f)
    recs = [r for r in recs if not (r["kernel"] == rec["kernel"] and r["workload"] == rec["workload"]
                                    and r["start_step"] == rec["start_step"] and r["path"] == rec["path"])]
    recs.append(rec)
    recs.sort(key=lambda r: (r["workload"], r["start_step"], r["path"], r["kernel"]))
    with open(OUT, "w") as f:
        json.dump(recs, f, indent=1)
    print(json.dumps(rec, indent=1))


if __name__ == "__main__":
    main()
