"""Summarise one `ncu --set full --import-source on` capture of the march kernel into profiles/.

  python -m paper_2205_15000_b200.ncu_summary --rep gpurun_out/x.ncu-rep --key cfg4_f64_stepper0 \
         --units 131874160640 --json profiles/r2_march_ncu.json --md profiles/r2_march_fp64_cfg4.md --command "<how x was made>"

Reads the report with `ncu -i ... --page raw --csv` and `--page source --csv --print-source sass` (no GPU needed), and
writes (a) one entry of the JSON that bench.py quotes — keyed by the capture name, stamped with the sha256 of the kernel
sources so that bench.py drops the figures when the sources change — and (b) a Markdown summary with the pipe /
memory metrics, the executed SASS opcode mix per unit and the warp-stall shares.  `units` = (piece, energy, angle-pair)
units of the captured launch (bench.py prints it as roofline.units_per_launch).
"""
from __future__ import annotations

import argparse
import collections
import csv
import hashlib
import io
import json
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))


def source_hash() -> str:
    h = hashlib.sha256()
    d = os.path.join(HERE, "csrc")
    for f in ("sc_kernels.cuh", "sc_math.cuh"):            # the files the march kernel is compiled from
        h.update(f.encode()); h.update(open(os.path.join(d, f), "rb").read())
    return h.hexdigest()


def _ncu(rep, *args):
    return subprocess.run(["ncu", "-i", rep, *args], capture_output=True, text=True, check=True).stdout


def raw_metrics(rep):
    rows = list(csv.reader(io.StringIO(_ncu(rep, "--page", "raw", "--csv"))))
    names, units, vals = rows[0], rows[1], rows[2]
    return {n: (u, v) for n, u, v in zip(names, units, vals)}


SCALE = {"Tbyte": 1e12, "Gbyte": 1e9, "Mbyte": 1e6, "Kbyte": 1e3, "byte": 1.0, "s": 1.0, "ms": 1e-3, "us": 1e-6, "ns": 1e-9,
         "Ghz": 1e9, "Mhz": 1e6, "hz": 1.0}


def val(m, name):
    u, v = m[name]
    return float(v.replace(",", "")) * SCALE.get(u, 1.0)


def sass_table(rep):
    rows = list(csv.reader(io.StringIO(_ncu(rep, "--page", "source", "--csv", "--print-source", "sass"))))
    hdr, data = rows[1], rows[2:]
    ix = {h: i for i, h in enumerate(hdr)}
    ops = collections.Counter(); stalls = collections.Counter(); total = 0
    for r in data:
        src = r[ix["Source"]].split()
        op = (src[1] if src[0].startswith("@") else src[0]).split(".")[0]
        n = int(r[ix["Instructions Executed"]])
        ops[op] += n; total += n
        for h in hdr:
            if h.startswith("stall_") and "Not Issued" not in h:
                stalls[h] += int(r[ix[h]])
    return rows[0][1] if len(rows[0]) > 1 else "", ops, total, stalls


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--rep", required=True)
    ap.add_argument("--key", required=True)
    ap.add_argument("--units", type=float, required=True)
    ap.add_argument("--json", required=True)
    ap.add_argument("--md", required=True)
    ap.add_argument("--command", default="")
    a = ap.parse_args()
    m = raw_metrics(a.rep)
    kernel, ops, total, stalls = sass_table(a.rep)
    uw = a.units / 32.0                                             # unit-warps: one warp instruction serves 32 units
    fp64 = sum(ops[o] for o in ("DFMA", "DMUL", "DADD"))
    fp32 = sum(ops[o] for o in ("FFMA", "FMUL", "FADD"))
    is32 = fp32 > fp64
    dur = val(m, "gpu__time_duration.sum")
    rd, wr = val(m, "dram__bytes_read.sum"), val(m, "dram__bytes_write.sum")
    entry = {
        "source_sha256": source_hash(), "kernel": kernel, "duration_s": dur,
        "dram_bytes": rd + wr, "dram_bytes_read": rd, "dram_bytes_write": wr, "dram_gbs": (rd + wr) / dur / 1e9,
        "sm_clock_ghz": val(m, "sm__cycles_elapsed.avg.per_second") / 1e9,
        "pipe_fp64_cycles_active_pct": float(m["sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active"][1]),
        "pipe_fma_cycles_active_pct": float(m["sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_active"][1]),
        "pipe_xu_inst_pct": float(m["sm__inst_executed_pipe_xu.avg.pct_of_peak_sustained_active"][1]),
        "issue_active_pct": float(m["smsp__issue_active.avg.pct_of_peak_sustained_active"][1]),
        "registers_per_thread": int(float(m["launch__registers_per_thread"][1])),
        "warp_instr_per_unit": total / uw,
        "fp_pipe_warp_instr_per_unit": (fp32 if is32 else fp64) / uw,
        "mufu_per_unit": ops["MUFU"] / uw,
        "units": a.units,
    }
    j = {"captures": {}}
    if os.path.exists(a.json):
        j = json.load(open(a.json))
    j["captures"][a.key] = entry
    json.dump(j, open(a.json, "w"), indent=1, sort_keys=True)
    tot_st = sum(stalls.values()) or 1
    with open(a.md, "w") as f:
        f.write(f"# ncu --set full: `{kernel}`\n\nCapture key `{a.key}` of `{os.path.basename(a.json)}`; kernel sources sha256 `{entry['source_sha256'][:16]}…`.\n\n")
        if a.command:
            f.write("Command (one B200; the same command without ncu had exited 0 first):\n\n```\n" + a.command + "\n```\n\n")
        f.write("Summarised with `python -m paper_2205_15000_b200.ncu_summary` from `ncu -i <rep> --page raw --csv` and `--page source --csv --print-source sass`.\n\n")
        f.write("| metric | value |\n|---|---|\n")
        for k in ("duration_s", "sm_clock_ghz", "pipe_fp64_cycles_active_pct", "pipe_fma_cycles_active_pct", "pipe_xu_inst_pct", "issue_active_pct",
                  "registers_per_thread", "dram_bytes_read", "dram_bytes_write", "dram_gbs", "units", "warp_instr_per_unit", "fp_pipe_warp_instr_per_unit", "mufu_per_unit"):
            v = entry[k]
            f.write(f"| `{k}` | {v:.6g} |\n" if isinstance(v, float) else f"| `{k}` | {v} |\n")
        for extra in ("l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum", "lts__t_sector_hit_rate.pct", "sm__warps_active.avg.pct_of_peak_sustained_active",
                      "launch__occupancy_limit_registers", "smsp__thread_inst_executed_per_inst_executed.ratio"):
            if extra in m:
                f.write(f"| `{extra}` | {m[extra][1]} {m[extra][0]} |\n")
        f.write("\nExecuted SASS warp instructions per unit-warp (one warp instruction serves the 32 energies of a unit's round):\n\n| opcode | per unit |\n|---|---|\n")
        for op, n in ops.most_common(24):
            f.write(f"| {op} | {n / uw:.2f} |\n")
        f.write("\nWarp-state samples (share of all samples):\n\n| state | share |\n|---|---|\n")
        for s, n in sorted(stalls.items(), key=lambda kv: -kv[1])[:10]:
            f.write(f"| {s} | {n / tot_st:.3f} |\n")
    print(json.dumps(entry, indent=1))


if __name__ == "__main__":
    main()
