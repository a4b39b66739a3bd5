"""Off-line tuning of the execution plan for this machine (plans are "recomputed
for each new target system"; L53: dispatch structures precomputed from sample executions).

  python -m paper_1405_2915_b200.tune [--out plans/b200.plan] [--reps 7]

Times every applicable kernel variant of the skeleton instances the bench configs use (and a few
neighbours, so that the plan's dispatch tree has more than one tuned radius per skeleton) at
n = 2^k under the conditions of a sustained run (skel_tune_instance: operands rotate through arenas
larger than L2, every timed launch follows a writer that leaves L2 dirty), stores the per-size
winners as breakpoints, prints the timing tables (microseconds) and writes the plan file that
bench.py and users load with skel_plan_load. The file is written by this program only: its first
line is a '#' comment that names the command, the GPU and the date; nobody edits breakpoints by hand.
"""
from __future__ import annotations

import argparse
import json
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))


def instances(S):
    I = S.SkelInstance
    out = []
    out.append(("map_saxpy_f32", I(skeleton=S.SK_MAP, fn=S.FN_SAXPY, dtype=S.F32, mode=1), 12, 26, 0))
    out.append(("map_mult_const_f32", I(skeleton=S.SK_MAP, fn=S.FN_MULT, dtype=S.F32, mode=0), 12, 26, 0))
    out.append(("map3_muladd_f32", I(skeleton=S.SK_MAP, fn=S.FN_MULADD, dtype=S.F32, mode=2), 12, 26, 0))
    out.append(("reduce_add_i32", I(skeleton=S.SK_REDUCE, fn=S.FN_ADD, dtype=S.I32), 12, 26, 0))
    out.append(("reduce_max_i32", I(skeleton=S.SK_REDUCE, fn=S.FN_MAX, dtype=S.I32), 12, 26, 0))
    out.append(("reduce_add_f32", I(skeleton=S.SK_REDUCE, fn=S.FN_ADD, dtype=S.F32), 12, 26, 0))
    out.append(("dot_f32", I(skeleton=S.SK_MAPREDUCE, fn=S.FN_MULT, fn2=S.FN_ADD, dtype=S.F32, mode=1), 12, 26, 0))
    for mode, mn in ((S.SCAN_INCLUSIVE, "incl"), (S.SCAN_EXCLUSIVE, "excl")):
        out.append((f"scan_add_i32_{mn}", I(skeleton=S.SK_SCAN, fn=S.FN_ADD, dtype=S.I32, mode=mode), 12, 28, 0))
    for r in (1, 4, 16):
        for edge in (S.EDGE_CONSTANT, S.EDGE_DUPLICATE):
            out.append((f"overlap1d_r{r}_e{edge}", I(skeleton=S.SK_OVERLAP1D, fn=S.FN_WSTENCIL, dtype=S.F32, r0=r, edge=edge), 12, 26, 0))
    for r in (2, 8):  # neighbours for the dispatch tree (not in a bench config)
        out.append((f"overlap1d_r{r}_e1", I(skeleton=S.SK_OVERLAP1D, fn=S.FN_WSTENCIL, dtype=S.F32, r0=r, edge=S.EDGE_DUPLICATE), 12, 26, 0))
    # rows of a matrix: shape class 1 of the dispatch tree (skel_instance.mode)
    out.append(("overlap1d_rows_r8", I(skeleton=S.SK_OVERLAP1D, fn=S.FN_WSTENCIL, dtype=S.F32, r0=8, edge=S.EDGE_DUPLICATE, mode=1), 20, 26, 8192))
    out.append(("overlap1d_cols_r8", I(skeleton=S.SK_OVERLAP1D_COL, fn=S.FN_WSTENCIL, dtype=S.F32, r0=8, edge=S.EDGE_DUPLICATE), 20, 26, 8192))
    for r in (1, 2, 4):
        out.append((f"overlap2d_{2*r+1}x{2*r+1}", I(skeleton=S.SK_OVERLAP2D, fn=S.FN_WSTENCIL, dtype=S.F32, r0=r, r1=r, edge=S.EDGE_DUPLICATE), 20, 26, 8192))
    # int32 containers (S:§8(f) f2): the same kernels on integer weights, IMAD instead of FFMA2
    out.append(("overlap1d_r4_e1_i32", I(skeleton=S.SK_OVERLAP1D, fn=S.FN_WSTENCIL, dtype=S.I32, r0=4, edge=S.EDGE_DUPLICATE), 12, 26, 0))
    out.append(("overlap2d_5x5_i32", I(skeleton=S.SK_OVERLAP2D, fn=S.FN_WSTENCIL, dtype=S.I32, r0=2, r1=2, edge=S.EDGE_DUPLICATE), 20, 26, 8192))
    out.append(("reduce_rows_add_f32", I(skeleton=S.SK_REDUCE_ROWS, fn=S.FN_ADD, dtype=S.F32), 20, 26, 8192))
    out.append(("separable_r8", I(skeleton=S.SK_SEPARABLE, fn=S.FN_WSTENCIL, dtype=S.F32, r0=8, r1=8, edge=S.EDGE_DUPLICATE), 20, 26, 8192))
    out.append(("separable_r8_const", I(skeleton=S.SK_SEPARABLE, fn=S.FN_WSTENCIL, dtype=S.F32, r0=8, r1=8, edge=S.EDGE_CONSTANT), 20, 26, 8192))
    return out


def selected(name: str, only: str | None) -> bool:
    """--only: comma-separated substrings; an instance is tuned when its name contains one of them (all when unset)."""
    if not only:
        return True
    return any(part and part in name for part in only.split(","))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default=os.path.join(HERE, "plans", "b200.plan"))
    ap.add_argument("--reps", type=int, default=11)
    ap.add_argument("--tables", default=None, help="write the timing tables as JSON here")
    ap.add_argument("--only", default=None, help="tune only the instances whose name contains this substring (several: comma-separated)")
    ap.add_argument("--base", default=None, help="start from this plan file (instances not tuned keep their entries)")
    args = ap.parse_args()
    sys.path.insert(0, os.path.dirname(HERE))
    from paper_1405_2915_b200 import skel as S

    ctx = S.Context()
    if args.base and os.path.exists(args.base):
        ctx.plan_load(args.base)
    tables = {}
    for name, inst, lo, hi, cols in instances(S):
        if not selected(name, args.only):
            continue
        t = ctx.tune(inst, lo, hi, cols, args.reps)
        names = S.variant_names(inst.skeleton)
        tables[name] = {"variants": names, "log2_lo": lo, "us": [[None if x != x else round(float(x), 2) for x in row] for row in t]}
        print(f"== {name}: " + ", ".join(f"{i}:{n}" for i, n in enumerate(names)))
        for k, row in enumerate(t):
            if all(x != x for x in row):
                continue
            best = min((x, i) for i, x in enumerate(row) if x == x)[1]
            print(f"  2^{lo + k:2d}  " + " ".join(f"{x:9.1f}" for x in row) + f"   -> {best}")
    # a partial re-tune (--only with --base) keeps the provenance lines of the plan it started from below its own
    # (read before the plan is saved: --out may be the same file as --base)
    earlier = ""
    if args.base and os.path.exists(args.base):
        earlier = "".join(ln for ln in open(args.base) if ln.startswith("#"))
    os.makedirs(os.path.dirname(os.path.abspath(args.out)), exist_ok=True)
    ctx.plan_save(args.out)
    # provenance: '#' lines are comments for the loader
    import datetime
    import torch
    body = open(args.out).read()
    cmd = "python -m paper_1405_2915_b200.tune " + " ".join(sys.argv[1:])
    note = (f"# generated by: {cmd.strip()}  (skel_tune_instance, reps={args.reps}; {torch.cuda.get_device_name(0)}, "
            f"{datetime.datetime.now(datetime.timezone.utc).strftime('%Y-%m-%d %H:%M UTC')}); not edited by hand\n")
    with open(args.out, "w") as f:
        f.write(note + earlier + body)
    if args.tables:
        with open(args.tables, "w") as f:
            json.dump(tables, f)
    ctx.close()
    print("plan written to", args.out)


if __name__ == "__main__":
    main()
