"""Turn ncu output into the text summaries kept under profiles/ (part of the profiling recipe; no GPU needed).

The captures themselves are made on the GPU box under `gpurun`, each only after the same command has exited 0
without ncu (/opt/skills/guides/B200_PROFILING.md):

    # launch list of one bench step (cold-cache, serialised per-launch times: compare SHARES, not absolutes)
    ncu --metrics gpu__time_duration.sum --clock-control none -c N --csv --log-file gpurun_out/launches.csv \
        python bench.py --steps 1 --warmup 1 --no-extras --no-cpu-baseline
    # one full capture of a kernel family
    ncu --set full --clock-control none --import-source on -k regex:orth_kernel -s SKIP -c COUNT \
        -o gpurun_out/NAME -f python bench.py --steps 1 --warmup 1 --no-extras --no-cpu-baseline

and are summarised here (the .ncu-rep is read with `ncu -i REP --page raw --csv` / `--page source --csv`):

    python -m paper_2009_12101_b200.profsummary launches RAW.csv OUT_PREFIX --cmd "..." [--note "..."]
    python -m paper_2009_12101_b200.profsummary full REP.ncu-rep OUT_PREFIX --cmd "..." [--note "..."]
    python -m paper_2009_12101_b200.profsummary source REP.ncu-rep OUT.md --launch I [--top 40] --cmd "..."
    python -m paper_2009_12101_b200.profsummary traffic OUT_PREFIX --n N --nnz NNZ --workload C5 REP:FMT [REP:FMT ...]

`traffic` writes OUT_PREFIX.csv / .md: per kernel family, ncu's dram__bytes_read.sum + dram__bytes_write.sum
of the captured launches over their ALGORITHMIC bytes (the basis size k of an orth launch
is inferred from its own read bytes).  bench.py multiplies that ratio into `roofline.traffic`.
"""
from __future__ import annotations

import argparse
import csv
import io
import os
import statistics
import subprocess
import sys
from collections import defaultdict

FORMAT_BYTES = {"fp64": 8, "fp32": 4, "fp16": 2, "int32": 4, "int16": 2}


def _short(name: str) -> str:
    return name.replace("(int)", "").replace("cbg::", "").split("(")[0].replace("void ", "")


def _family(kernel: str) -> str:
    k = _short(kernel)
    if "orth_fused" in k:  # the row-mapped fused update + multi-dot (template arguments: format, words per lane)
        return "update_multidot"
    if "orth" in k:
        kind = k.rstrip(">").split(",")[-1].strip()
        return {"0": "multidot", "1": "update", "2": "update_multidot"}.get(kind, k)
    if "spmv" in k:
        return "spmv"
    if "store" in k:
        return "store"
    return "other"


def launches(raw, out_prefix, cmd, note):
    rows = []
    with open(raw) as f:
        lines = [l for l in f if not l.startswith("==")]
    for r in csv.DictReader(io.StringIO("".join(lines))):
        if r.get("Metric Name") != "gpu__time_duration.sum":
            continue
        v = float(r["Metric Value"].replace(",", ""))
        ns = v * {"ns": 1, "us": 1e3, "ms": 1e6, "nsecond": 1, "usecond": 1e3, "msecond": 1e6}.get(r["Metric Unit"], 1)
        rows.append((_short(r["Kernel Name"]), r["Grid Size"].replace(" ", ""), r["Block Size"].replace(" ", ""), ns))
    agg = defaultdict(list)
    for k, g, b, ns in rows:
        agg[(k, g, b)].append(ns)
    tot = sum(ns for *_, ns in rows)
    with open(out_prefix + ".md", "w") as f:
        f.write("# ncu launch list summary\n\nCommand (run under gpurun, after the same command exited 0 without ncu):\n\n```\n" + cmd + "\n```\n\n")
        f.write("Summarised by `python -m paper_2009_12101_b200.profsummary launches` (the raw per-launch list is not kept).\n\n")
        f.write(note + "\n\n")
        f.write(f"{len(rows)} launches, {tot / 1e6:.3f} ms summed device time (cold-cache, serialised: compare shares).\n\n")
        f.write("| kernel | grid | block | launches | sum ms | share | min us | median us | max us |\n|---|---|---|---|---|---|---|---|---|\n")
        for (k, g, b), v in sorted(agg.items(), key=lambda kv: -sum(kv[1])):
            f.write(f"| `{k}` | {g} | {b} | {len(v)} | {sum(v) / 1e6:.3f} | {sum(v) / tot:.3f} | {min(v) / 1e3:.1f} | {statistics.median(v) / 1e3:.1f} | {max(v) / 1e3:.1f} |\n")
        fam = defaultdict(float)
        for (k, g, b), v in agg.items():
            fam[_family(k)] += sum(v)
        f.write("\nShares by kernel family:\n\n| family | sum ms | share |\n|---|---|---|\n")
        for k, v in sorted(fam.items(), key=lambda kv: -kv[1]):
            f.write(f"| {k} | {v / 1e6:.3f} | {v / tot:.3f} |\n")


COLS = [
    ("gpu__time_duration.sum", "us"), ("dram__bytes_read.sum", "dram read MB"), ("dram__bytes_write.sum", "dram write MB"),
    ("gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed", "dram %"), ("sm__throughput.avg.pct_of_peak_sustained_elapsed", "sm %"),
    ("lts__t_sector_hit_rate.pct", "L2 hit %"), ("smsp__issue_active.avg.pct_of_peak_sustained_active", "issue %"),
    ("sm__inst_executed_pipe_fp64.avg.pct_of_peak_sustained_active", "fp64 pipe %"),
    ("sm__inst_executed_pipe_alu.avg.pct_of_peak_sustained_active", "alu pipe %"),
    ("sm__inst_executed_pipe_lsu.avg.pct_of_peak_sustained_active", "lsu pipe %"),
    ("launch__registers_per_thread", "regs"), ("launch__shared_mem_per_block_dynamic", "dyn smem KB"),
    ("l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum", "smem bank conflicts"),
    ("l1tex__data_pipe_lsu_wavefronts_mem_shared.sum", "smem wavefronts"),
    ("smsp__inst_executed.sum", "warp instructions"),
]
STALLS = ["long_scoreboard", "short_scoreboard", "barrier", "wait", "math_pipe_throttle", "mio_throttle", "lg_throttle", "not_selected",
          "dispatch_stall", "membar", "sleeping", "branch_resolving", "no_instruction", "selected"]


def _raw_rows(rep):
    if rep.endswith(".csv"):  # the raw page already exported on the GPU box (`ncu -i REP --page raw --csv > REP_raw.csv`)
        with open(rep) as f:
            txt = f.read()
    else:
        txt = subprocess.run(["ncu", "-i", rep, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    rd = list(csv.reader(io.StringIO(txt)))
    hdr, units, data = rd[0], rd[1], rd[2:]
    idx = {h: i for i, h in enumerate(hdr)}

    def val(row, name):
        if name not in idx:
            return float("nan")
        s = row[idx[name]].replace(",", "")
        try:
            v = float(s)
        except ValueError:
            return float("nan")
        u = units[idx[name]]
        scale = {"ns": 1e-3, "us": 1, "ms": 1e3, "byte": 1e-6, "Kbyte": 1e-3, "Mbyte": 1, "Gbyte": 1e3}.get(u, 1)
        if name.startswith("launch__shared"):
            scale = {"byte": 1e-3, "Kbyte": 1}.get(u, 1)
        return v * scale

    return idx, data, val


def full(rep, out_prefix, cmd, note):
    idx, data, val = _raw_rows(rep)
    with open(out_prefix + ".csv", "w") as fc, open(out_prefix + ".md", "w") as fm:
        fc.write("id,kernel," + ",".join(c for c, _ in COLS) + "," + ",".join("stall_" + s for s in STALLS) + "\n")
        fm.write(f"# ncu --set full summary: `{os.path.basename(out_prefix)}.csv`\n\nCommand (under gpurun, after the same command exited 0 without ncu):\n\n```\n{cmd}\n```\n\n"
                 "Read with `ncu -i <rep> --page raw --csv` by `python -m paper_2009_12101_b200.profsummary full`; selected columns kept in the "
                 "`.csv` beside this file (times in us, bytes in MB, shared memory in KB).\n\n" + note + "\n\n")
        fm.write("| id | kernel | us | dram read MB | dram write MB | dram GB/s | dram % | sm % | L2 hit % | issue % | fp64 pipe % | alu pipe % | regs | warp inst (M) |\n|---|---|---|---|---|---|---|---|---|---|---|---|---|---|\n")
        stall_lines = []
        for i, row in enumerate(data):
            name = _short(row[idx["Kernel Name"]])
            v = {c: val(row, c) for c, _ in COLS}
            st = [val(row, f"smsp__average_warps_issue_stalled_{s}_per_issue_active.ratio") for s in STALLS]
            fc.write(f'{i},"{name}",' + ",".join(f"{v[c]:.6g}" for c, _ in COLS) + "," + ",".join(f"{x:.4g}" for x in st) + "\n")
            us, rd_mb, wr_mb = v["gpu__time_duration.sum"], v["dram__bytes_read.sum"], v["dram__bytes_write.sum"]
            fm.write(f"| {i} | `{name}` | {us:.1f} | {rd_mb:.1f} | {wr_mb:.1f} | {(rd_mb + wr_mb) / us * 1e3:.0f} | "
                     f"{v['gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed']:.1f} | {v['sm__throughput.avg.pct_of_peak_sustained_elapsed']:.1f} | "
                     f"{v['lts__t_sector_hit_rate.pct']:.1f} | {v['smsp__issue_active.avg.pct_of_peak_sustained_active']:.1f} | "
                     f"{v['sm__inst_executed_pipe_fp64.avg.pct_of_peak_sustained_active']:.1f} | {v['sm__inst_executed_pipe_alu.avg.pct_of_peak_sustained_active']:.1f} | "
                     f"{v['launch__registers_per_thread']:.0f} | {v['smsp__inst_executed.sum'] / 1e6:.2f} |\n")
            stall_lines.append(f"| {i} | " + " | ".join(f"{x:.2f}" for x in st) + " |\n")
        fm.write("\nWarp stall reasons (warps stalled per issue-active cycle, `smsp__average_warps_issue_stalled_*_per_issue_active`):\n\n| id | "
                 + " | ".join(STALLS) + " |\n|" + "---|" * (len(STALLS) + 1) + "\n" + "".join(stall_lines))


def source(rep, out_md, launch, top, cmd, note):
    """Hot spots of one captured launch: SASS instructions ranked by executed warp instructions."""
    if rep.endswith(".csv"):  # the source page already exported on the GPU box (`ncu -i REP --page source --csv --print-source sass`)
        with open(rep) as f:
            txt = f.read()
    else:
        txt = subprocess.run(["ncu", "-i", rep, "--page", "source", "--csv", "--print-source", "sass"],
                             capture_output=True, text=True).stdout
    rows = list(csv.reader(io.StringIO(txt)))
    starts = [i for i, r in enumerate(rows) if r and r[0] == "Kernel Name"]  # one section per captured launch
    if launch >= len(starts):
        raise SystemExit(f"{rep} has {len(starts)} launches")
    lo, hi = starts[launch], (starts[launch + 1] if launch + 1 < len(starts) else len(rows))
    kname = _short(rows[lo][1])
    h = rows[lo + 1]
    ci = {name: h.index(name) for name in h}
    col_inst = "Instructions Executed"
    col_samp = "# Samples" if "# Samples" in ci else None
    body = [r for r in rows[lo + 2:hi] if len(r) == len(h)]

    def num(s):
        try:
            return float(s.replace(",", ""))
        except ValueError:
            return 0.0

    total = sum(num(r[ci[col_inst]]) for r in body) or 1.0
    tot_s = sum(num(r[ci[col_samp]]) for r in body) if col_samp else 0.0
    by_op = defaultdict(float)
    for r in body:
        op = r[ci["Source"]].strip().split()
        op = [t for t in op if not t.startswith("@")]
        by_op[op[0].split(".")[0] if op else "?"] += num(r[ci[col_inst]])
    with open(out_md, "w") as f:
        f.write(f"# ncu source page, launch {launch} of `{os.path.basename(rep)}`: `{kname}`\n\nCommand:\n\n```\n{cmd}\n```\n\n{note}\n\n")
        f.write(f"{total / 1e6:.2f} M warp instructions executed.\n\nBy opcode:\n\n| opcode | warp inst (M) | share |\n|---|---|---|\n")
        for op, v in sorted(by_op.items(), key=lambda kv: -kv[1])[:25]:
            f.write(f"| {op} | {v / 1e6:.3f} | {v / total:.3f} |\n")
        f.write(f"\nTop {top} SASS lines by executed warp instructions"
                + (" (and their share of the stall samples)" if col_samp else "") + ":\n\n| # | share inst | share samples | SASS |\n|---|---|---|---|\n")
        ranked = sorted(enumerate(body), key=lambda ir: -num(ir[1][ci[col_inst]]))[:top]
        for i, r in ranked:
            ss = f"{num(r[ci[col_samp]]) / tot_s:.4f}" if col_samp and tot_s else ""
            f.write(f"| {i} | {num(r[ci[col_inst]]) / total:.4f} | {ss} | `{r[ci['Source']].strip()}` |\n")


def traffic(out_prefix, n, nnz, workload, reps):
    """traffic / algorithmic bytes per family from full captures (REP:FMT)."""
    acc = defaultdict(lambda: [0.0, 0.0, 0, set()])
    for item in reps:
        rep, fmt = item.rsplit(":", 1)
        B = FORMAT_BYTES[fmt]
        idx, data, val = _raw_rows(rep)
        for row in data:
            fam = _family(row[idx["Kernel Name"]])
            rd, wr = val(row, "dram__bytes_read.sum") * 1e6, val(row, "dram__bytes_write.sum") * 1e6
            if fam in ("multidot", "update", "update_multidot"):
                k = max(1, round((rd - 8 * n) / (n * B)))  # the basis size of this launch, from its own read bytes
                alg = k * n * B + (8 * n if fam == "multidot" else 16 * n)
            elif fam == "spmv":
                alg = 12 * nnz + 4 * (n + 1) + 16 * n
            elif fam == "store":
                alg = (16 + B) * n
            else:
                continue
            a = acc[fam]
            a[0] += rd + wr
            a[1] += alg
            a[2] += 1
            a[3].add(os.path.basename(rep))
    with open(out_prefix + ".csv", "w") as f:
        f.write("family,traffic_over_algorithmic,captured_launches,traffic_bytes_sum,algorithmic_bytes_sum,workload,capture\n")
        for fam, (t, a, c, names) in acc.items():
            f.write(f"{fam},{t / a:.4f},{c},{t:.0f},{a:.0f},{workload},{'+'.join(sorted(names))}\n")
    with open(out_prefix + ".md", "w") as f:
        f.write(f"# DRAM traffic over algorithmic bytes, per kernel family (`{os.path.basename(out_prefix)}.csv`)\n\n"
                f"`dram__bytes_read.sum + dram__bytes_write.sum` per launch from the `--set full` captures named in the table (workload {workload}, "
                f"n = {n}, nnz = {nnz}), divided by the algorithmic bytes of the same launches (DESIGN.md section 6; k of a Gram-Schmidt launch inferred "
                "from its own read bytes).  Written by `python -m paper_2009_12101_b200.profsummary traffic`; `bench.py` multiplies the ratio of the "
                "dominant family into `roofline.traffic`.\n\n| family | traffic / algorithmic | launches | captures |\n|---|---|---|---|\n")
        for fam, (t, a, c, names) in acc.items():
            f.write(f"| {fam} | {t / a:.4f} | {c} | {', '.join(sorted(names))} |\n")


def main(argv=None) -> int:
    ap = argparse.ArgumentParser()
    sub = ap.add_subparsers(dest="what", required=True)
    a = sub.add_parser("launches")
    a.add_argument("raw")
    a.add_argument("out_prefix")
    a = sub.add_parser("full")
    a.add_argument("rep")
    a.add_argument("out_prefix")
    a = sub.add_parser("source")
    a.add_argument("rep")
    a.add_argument("out_md")
    a.add_argument("--launch", type=int, default=0)
    a.add_argument("--top", type=int, default=40)
    a = sub.add_parser("traffic")
    a.add_argument("out_prefix")
    a.add_argument("--n", type=int, required=True)
    a.add_argument("--nnz", type=int, required=True)
    a.add_argument("--workload", default="C5")
    a.add_argument("reps", nargs="+")
    for p in sub.choices.values():
        p.add_argument("--cmd", default="")
        p.add_argument("--note", default="")
    args = ap.parse_args(argv)
    if args.what == "launches":
        launches(args.raw, args.out_prefix, args.cmd, args.note)
    elif args.what == "full":
        full(args.rep, args.out_prefix, args.cmd, args.note)
    elif args.what == "source":
        source(args.rep, args.out_md, args.launch, args.top, args.cmd, args.note)
    else:
        traffic(args.out_prefix, args.n, args.nnz, args.workload, args.reps)
    return 0


if __name__ == "__main__":
    sys.exit(main())
