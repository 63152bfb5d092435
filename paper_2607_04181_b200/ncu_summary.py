"""Summarises an `ncu --set full` export as text for profiles/ (measurement aid; no arithmetic of the method).

    ncu -i gpurun_out/X.ncu-rep --page raw --csv > gpurun_out/X.raw.csv          # here, no GPU needed
    python -m paper_2607_04181_b200.ncu_summary gpurun_out/X.raw.csv --out profiles/X.md \
        --title "..." --command "..." [--traffic-replicas R]

Writes a markdown table (one column per profiled launch) of the metrics the roofline discussion uses, and with
--traffic-replicas R records dram__bytes_read/write per launch of every layer kernel in profiles/ncu_traffic.json
under "R<R>", with the commit the capture was taken at -- bench.py reads `roofline.traffic` from that file.
"""
from __future__ import annotations

import argparse
import csv
import json
import os
import re
import subprocess

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
METRICS = [
    "gpu__time_duration.sum",
    "dram__bytes_read.sum",
    "dram__bytes_write.sum",
    "gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed",
    "lts__throughput.avg.pct_of_peak_sustained_elapsed",
    "sm__pipe_tensor_cycles_active.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_tensor.sum",
    "launch__registers_per_thread",
    "launch__grid_size",
    "launch__cluster_size",
    "sm__warps_active.avg.pct_of_peak_sustained_active",
]
# kernel-name pattern -> the stage name bench.py uses
STAGES = [(r"k_prologue", "prologue"), (r"k_gemm(_cl)?<(\(int\))?0[,>]", "gemm_qkv"), (r"k_attn", "attention"),
          (r"k_gemm(_cl)?<(\(int\))?1[,>]", "gemm_o"), (r"k_gemm(_cl)?<(\(int\))?2[,>]", "gemm_gate_up"),
          (r"k_gemm(_cl)?<(\(int\))?3[,>]", "gemm_down"),
          (r"k_big_gemm<(\(int\))?0", "big_gemm_qkv"), (r"k_big_gemm<(\(int\))?1", "big_gemm_o"),
          (r"k_big_gemm<(\(int\))?2", "big_gemm_gate_up"), (r"k_big_gemm<(\(int\))?3", "big_gemm_down"),
          (r"k_prefill_attn", "prefill_attention"), (r"k_copy", "replica_copy")]


def stage_of(kernel: str) -> str:
    for pat, name in STAGES:
        if re.search(pat, kernel):
            return name
    m = re.search(r"(k_\w+)", kernel)
    return m.group(1) if m else kernel[:24]


def to_bytes(value: float, unit: str) -> float:
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}
    return value * scale.get(unit, 1.0)


def read_raw(path: str):
    """Rows of `--page raw --csv`: a header line, a units line, then one line per profiled launch."""
    with open(path, newline="") as f:
        rows = [r for r in csv.reader(f) if r and not r[0].startswith("==")]
    head, units, body = rows[0], rows[1], rows[2:]
    col = {h: i for i, h in enumerate(head)}
    return col, units, body


def main() -> int:
    ap = argparse.ArgumentParser()
    ap.add_argument("raw_csv")
    ap.add_argument("--out", required=True)
    ap.add_argument("--title", default="ncu --set full summary")
    ap.add_argument("--command", default="")
    ap.add_argument("--note", default="")
    ap.add_argument("--traffic-replicas", type=int, default=0)
    a = ap.parse_args()
    col, units, body = read_raw(a.raw_csv)
    kname = col.get("Kernel Name")
    names = [stage_of(r[kname]) for r in body]
    lines = [f"# {a.title}", ""]
    if a.command:
        lines += [f"Command: `{a.command}`, read here with `ncu -i … --page raw --csv` and "
                  f"`python -m paper_2607_04181_b200.ncu_summary`.", ""]
    lines += ["| metric | unit | " + " | ".join(names) + " |", "|---|---|" + "---|" * len(names)]
    for m in METRICS:
        if m not in col:
            continue
        i = col[m]
        lines.append(f"| `{m}` | {units[i]} | " + " | ".join(r[i] for r in body) + " |")
    traffic = {}
    if "dram__bytes_read.sum" in col and "dram__bytes_write.sum" in col:
        ir, iw = col["dram__bytes_read.sum"], col["dram__bytes_write.sum"]
        parts = []
        for n, r in zip(names, body):
            rd = to_bytes(float(r[ir].replace(",", "")), units[ir])
            wr = to_bytes(float(r[iw].replace(",", "")), units[iw])
            traffic[n] = {"dram_bytes_read": int(round(rd)), "dram_bytes_write": int(round(wr))}
            parts.append(f"{n} {(rd + wr) / 1e6:.1f} MB")
        lines += ["", "DRAM traffic (read + write) per launch: " + ", ".join(parts) + "."]
    if a.note:
        lines += ["", a.note]
    with open(a.out, "w") as f:
        f.write("\n".join(lines) + "\n")
    if a.traffic_replicas:
        path = os.path.join(ROOT, "profiles", "ncu_traffic.json")
        try:
            with open(path) as f:
                t = json.load(f)
        except Exception:
            t = {"kernels": {}}
        try:
            commit = subprocess.run(["git", "-C", ROOT, "rev-parse", "--short", "HEAD"], capture_output=True, text=True).stdout.strip()
        except Exception:
            commit = "unknown"
        t["commit"] = commit or "unknown"
        for n, e in traffic.items():
            e = dict(e, summary=os.path.relpath(os.path.abspath(a.out), ROOT))
            t.setdefault("kernels", {}).setdefault(n, {})[f"R{a.traffic_replicas}"] = e
        with open(path, "w") as f:
            json.dump(t, f, indent=1, sort_keys=True)
            f.write("\n")
    return 0


if __name__ == "__main__":
    raise SystemExit(main())
