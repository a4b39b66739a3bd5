"""Turn an `ncu --page raw --csv` export of one bench step into the summaries kept under profiles/.

  ncu -i step.ncu-rep --page raw --csv > step_raw.csv
  python -m paper_1405_2915_b200.ncu_summary step_raw.csv bench_line.json --csv profiles/rNN_ncu_traffic.csv --md profiles/rNN_ncu_step.md

The capture must hold the 16 kernel launches of ONE step of bench.py in launch order (bench.py's Workload.ops); the
bench JSON line (same tree, same plan) supplies the op names and the variant each op ran. Writes
  * the CSV bench.py reads `roofline.traffic` from: bench_op, variant, kernel, dram_bytes_read, dram_bytes_write;
  * a markdown table with the counters the design decisions rest on.
Text processing only; nothing here touches the GPU.
"""
from __future__ import annotations

import argparse
import csv
import json
import re


def num(v: str) -> float:
    try:
        return float(v.replace(",", ""))
    except ValueError:
        return float("nan")


def to_bytes(value: str, unit: str) -> float:
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}
    return num(value) * scale.get(unit, 1.0)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("raw_csv")
    ap.add_argument("bench_json")
    ap.add_argument("--csv", required=True)
    ap.add_argument("--md", required=True)
    ap.add_argument("--command", default="", help="the ncu command line, quoted verbatim in the markdown")
    args = ap.parse_args()
    rows = list(csv.reader(open(args.raw_csv)))
    hdr, units, data = rows[0], rows[1], rows[2:]
    col = {h: i for i, h in enumerate(hdr)}
    bench = json.loads([ln for ln in open(args.bench_json) if ln.startswith("{")][-1])
    ops = list(bench["per_skeleton"].items())
    assert len(data) >= len(ops), f"{len(data)} launches captured, {len(ops)} ops in a step"
    data = data[: len(ops)]

    def get(r, name):
        return r[col[name]] if name in col else ""

    out_rows, md = [], []
    md.append("| bench op | variant | kernel | us | DRAM rd MB | DRAM wr MB | DRAM / algorithmic | DRAM thr % | FMA pipe % | issue % | warps/SMSP | regs | top stalls (warps per issue) |")
    md.append("|---|---|---|---:|---:|---:|---:|---:|---:|---:|---:|---:|---|")
    for (op, info), r in zip(ops, data):
        kern = re.sub(r"\(.*", "", get(r, "Kernel Name"))
        rd = to_bytes(get(r, "dram__bytes_read.sum"), units[col["dram__bytes_read.sum"]])
        wr = to_bytes(get(r, "dram__bytes_write.sum"), units[col["dram__bytes_write.sum"]])
        dur = to_bytes(get(r, "gpu__time_duration.sum"), "byte")
        dur_unit = units[col["gpu__time_duration.sum"]]
        us = dur * {"ns": 1e-3, "us": 1.0, "ms": 1e3, "s": 1e6}.get(dur_unit, 1.0)
        alg = info["GB/s"] * info["us"] * 1e3  # algorithmic bytes of the op
        stalls = []
        for h, i in col.items():
            m = re.match(r"smsp__average_warps_issue_stalled_(.*)_per_issue_active\.ratio", h)
            if m and num(r[i]) == num(r[i]):
                stalls.append((num(r[i]), m.group(1)))
        stalls.sort(reverse=True)
        out_rows.append([op, info["variant"], kern, int(rd), int(wr)])
        md.append(f"| {op} | `{info['variant']}` | `{kern}` | {us:.1f} | {rd / 1e6:.1f} | {wr / 1e6:.1f} | {(rd + wr) / alg:.3f} | "
                  f"{num(get(r, 'gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed')):.0f} | "
                  f"{num(get(r, 'sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_active')):.0f} | "
                  f"{num(get(r, 'smsp__issue_active.avg.pct_of_peak_sustained_active')):.0f} | "
                  f"{num(get(r, 'smsp__warps_active.avg.per_cycle_active')):.1f} | {get(r, 'launch__registers_per_thread')} | "
                  + ", ".join(f"{n} {v:.1f}" for v, n in stalls[:3]) + " |")
    with open(args.csv, "w", newline="") as f:
        w = csv.writer(f)
        w.writerow(["bench_op", "variant", "kernel", "dram_bytes_read", "dram_bytes_write"])
        w.writerows(out_rows)
    with open(args.md, "w") as f:
        f.write("# ncu `--set full` capture of one bench step (16 launches, full sizes)\n\n")
        if args.command:
            f.write("Command (on the GPU box, after the same command had exited 0 without ncu):\n\n```\n" + args.command + "\n```\n\n")
        f.write("Per-launch values; durations under ncu are serialised and cold-cache (the CUDA-event numbers of the sustained run are "
                "in the bench JSON line). `DRAM / algorithmic` = (dram__bytes_read + dram__bytes_write) / algorithmic bytes of the op.\n\n")
        f.write("\n".join(md) + "\n")
    print("wrote", args.csv, args.md)


if __name__ == "__main__":
    main()
