#!/usr/bin/env python
"""Turns ncu exports into the text summaries kept under profiles/ (nothing here runs on the GPU).

  python -m paper_1711_07663_b200.profile_summary full  <raw.csv>      <config> <round-tag>   # from `ncu -i X.ncu-rep --page raw --csv`
  python -m paper_1711_07663_b200.profile_summary list  <launches.csv> <config> <round-tag>   # from `ncu --metrics gpu__time_duration.sum --csv`

`full` writes profiles/<tag>_kernels_full_config<C>.md (one row per captured launch) and, for config 2,
profiles/r2_dram_traffic.csv: DRAM bytes per launch of the kernels bench.py reports a roofline for, stamped with the
hash of the CUDA sources they were measured on (bench.py emits `traffic` only if that hash is the running code's).
`list` writes profiles/<tag>_launches_config<C>.md: every kernel of one cut in launch order and the shares per kernel.
The .md files carry the commands; fill in nothing by hand.
"""
from __future__ import annotations

import csv
import hashlib
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
BENCH_CMD = "python bench.py --config %d --steps 2 --warmup 3 --no-cpu-baseline --no-per-config"


def source_hash() -> str:
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_1711_07663_b200", "csrc")
    for name in sorted(os.listdir(d)):
        with open(os.path.join(d, name), "rb") as f:
            h.update(name.encode()); h.update(f.read())
    with open(os.path.join(ROOT, "include", "dc.h"), "rb") as f:
        h.update(f.read())
    return h.hexdigest()[:16]


def short(name: str) -> str:
    return name.split("(")[0].replace("void ", "")


def num(s: str) -> float:
    try:
        return float(s.replace(",", ""))
    except ValueError:
        return float("nan")


def do_full(path: str, cfg: int, tag: str):
    rows = list(csv.reader(open(path)))
    hdr, units = rows[0], rows[1]
    ix = {n: i for i, n in enumerate(hdr)}
    # ncu scales each column (us / ms, Mbyte / Gbyte ...): bring times to us and bytes to MB
    scale_of = {"ns": 1e-3, "us": 1.0, "ms": 1e3, "s": 1e6, "byte": 1e-6, "Kbyte": 1e-3, "Mbyte": 1.0, "Gbyte": 1e3}
    cols = [("gpu__time_duration.sum", "us", None), ("launch__registers_per_thread", "regs", 1.0),
            ("sm__warps_active.avg.pct_of_peak_sustained_active", "warps act %", 1.0),
            ("smsp__issue_active.avg.pct_of_peak_sustained_active", "issue %", 1.0),
            ("sm__inst_executed_pipe_fp64.avg.pct_of_peak_sustained_active", "fp64 pipe %", 1.0),
            ("smsp__thread_inst_executed_per_inst_executed.ratio", "lanes/inst", 1.0),
            ("dram__bytes_read.sum", "DRAM rd MB", None), ("dram__bytes_write.sum", "DRAM wr MB", None),
            ("gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed", "DRAM %", 1.0),
            ("smsp__average_warps_issue_stalled_long_scoreboard_per_issue_active.ratio", "stall long-sb", 1.0),
            ("smsp__average_warps_issue_stalled_wait_per_issue_active.ratio", "stall wait", 1.0),
            ("smsp__average_warps_issue_stalled_barrier_per_issue_active.ratio", "stall barrier", 1.0),
            ("smsp__inst_executed.sum", "warp inst M", 1e-6),
            ("smsp__sass_thread_inst_executed_op_dfma_pred_on.sum", "dfma", 1.0),
            ("smsp__sass_thread_inst_executed_op_dadd_pred_on.sum", "dadd", 1.0),
            ("smsp__sass_thread_inst_executed_op_dmul_pred_on.sum", "dmul", 1.0)]
    cols = [(c[0], c[1], c[2] if c[2] is not None else scale_of.get(units[ix[c[0]]], 1.0)) for c in cols if c[0] in ix]
    out = ["# Round 2: `ncu --set full` of the kernels of one cut, config %d" % cfg, "",
           "Commands (B200, under gpurun; the plain run exited 0 first, same call):", "", "```",
           BENCH_CMD % cfg + " > gpurun_out/plain.log 2>&1 &&",
           "ncu --set full --metrics smsp__sass_thread_inst_executed_op_dfma_pred_on.sum,smsp__sass_thread_inst_executed_op_dadd_pred_on.sum,"
           "smsp__sass_thread_inst_executed_op_dmul_pred_on.sum \\",
           "    --clock-control none --import-source on -k regex:'k_' --launch-skip 106 -c 35 \\",
           "    -f -o gpurun_out/prof_%s " % tag + BENCH_CMD % cfg,
           "ncu -i gpurun_out/prof_%s.ncu-rep --page raw --csv > raw.csv" % tag,
           "python -m paper_1711_07663_b200.profile_summary full raw.csv %d %s" % (cfg, tag), "```", "",
           "Sources: `src_sha16 = %s` (bench.py `config.src_sha16`).  Executed FP64 flops = 2 dfma + dadd + dmul "
           "(`smsp__sass_thread_inst_executed_op_*_pred_on.sum`, SURVEY.md 8(d)); the algorithmic ones are in the bench line.  "
           "Stall columns: warps stalled per issue slot (`smsp__average_warps_issue_stalled_*_per_issue_active.ratio`): long scoreboard = "
           "waiting for global / L2 data, wait = fixed-latency dependency, barrier = `__syncthreads`." % source_hash(), "",
           "| kernel | " + " | ".join(c[1] for c in cols if c[1] not in ("dfma", "dadd", "dmul")) + " | executed FP64 GFLOP |",
           "|---|" + "---:|" * (len([c for c in cols if c[1] not in ("dfma", "dadd", "dmul")]) + 1)]
    traffic = {}
    started = False
    for r in rows[2:]:
        if len(r) < len(hdr):
            continue
        name = short(r[ix["Kernel Name"]])
        if started and name == "k_reset_surface":
            break                                                # (the next cut begins: one cut only)
        started = started or name == "k_reset_surface"          # (rows before the cut's first kernel belong to the cut before)
        if not started:
            continue
        vals = {c[1]: num(r[ix[c[0]]]) * c[2] for c in cols}
        gf = (2 * vals.get("dfma", 0.0) + vals.get("dadd", 0.0) + vals.get("dmul", 0.0)) / 1e9
        out.append("| %s | " % name + " | ".join("%.1f" % vals[c[1]] for c in cols if c[1] not in ("dfma", "dadd", "dmul")) + " | %.3f |" % gf)
        key = "k_np_bound" if name.startswith("k_np_bound<") else ("k_np_solve" if name.startswith("k_np_solve") else name)
        t = traffic.setdefault(key, [0, 0.0, 0.0])
        t[0] += 1; t[1] += vals.get("DRAM rd MB", 0.0) * 1e6; t[2] += vals.get("DRAM wr MB", 0.0) * 1e6
    p = os.path.join(ROOT, "profiles", "%s_kernels_full_config%d.md" % (tag, cfg))
    open(p, "w").write("\n".join(out) + "\n")
    print("wrote", p)
    if cfg == 2:
        # bytes per launch; for the multi-launch kernels the SUM over the launches of one cut (bench.py's unit is one cut)
        p = os.path.join(ROOT, "profiles", "r2_dram_traffic.csv")
        with open(p, "w") as f:
            f.write("# src_sha16=%s config=%d source=%s_kernels_full_config%d.md\n" % (source_hash(), cfg, tag, cfg))
            f.write("kernel,launches_per_cut,dram_read_bytes_per_cut,dram_write_bytes_per_cut\n")
            for k in ("k_np_bound", "k_np_solve", "k_elem_boxes", "k_pairs", "k_uf_tiles"):
                if k in traffic:
                    f.write("%s,%d,%.0f,%.0f\n" % (k, traffic[k][0], traffic[k][1], traffic[k][2]))
        print("wrote", p)


def do_list(path: str, cfg: int, tag: str):
    rows = list(csv.reader(open(path)))
    h = [i for i, r in enumerate(rows) if r and r[0] == "ID"][0]
    hdr = rows[h]
    ix = {n: i for i, n in enumerate(hdr)}
    L = {}
    for r in rows[h + 1:]:
        if len(r) >= len(hdr) and r[ix["Metric Name"]] == "gpu__time_duration.sum":
            L[int(r[ix["ID"]])] = (short(r[ix["Kernel Name"]]), num(r[ix["Metric Value"]]) / 1000.0)
    ids = sorted(i for i in L if L[i][0] != "k_dfma_peak")
    starts = [i for i in ids if L[i][0] == "k_reset_surface"]
    s = starts[3] if len(starts) > 3 else starts[-1]
    e = [i for i in ids if i > s and L[i][0] == "k_uf_fix"][0]
    one = [L[i] for i in range(s, e + 1) if i in L]
    tot = sum(v for _, v in one)
    agg = {}
    for k, v in one:
        a = agg.setdefault(k, [0, 0.0]); a[0] += 1; a[1] += v
    out = ["# Round 2: ncu launch list, config %d" % cfg, "",
           "Commands (B200, under gpurun; the plain run exited 0 first, same call):", "", "```",
           BENCH_CMD % cfg + " > gpurun_out/plain.log 2>&1 &&",
           "ncu --metrics gpu__time_duration.sum --clock-control none -c 400 --csv --log-file gpurun_out/launches_%s.csv \\" % tag,
           "    " + BENCH_CMD % cfg,
           "python -m paper_1711_07663_b200.profile_summary list gpurun_out/launches_%s.csv %d %s" % (tag, cfg, tag), "```", "",
           "Per-launch times are cold-cache and serialised: compare SHARES with the CUDA-event times of the bench line "
           "(`cut.ms_full_cut_stages`, `cut.ms_S5_S6_kernels`).  Sources: `src_sha16 = %s`." % source_hash(), "",
           "One cut (the 4th `dc_cut` of the run = `dc_set_cut_surface` + `dc_classify(DC_FLAG_RECOMPUTE_BOXES)`, replayed from its CUDA "
           "graph: ncu profiles the graph's kernel nodes one by one): %d launches, %.1f us under ncu." % (len(one), tot), "",
           "| kernel | launches | sum us | share of the cut |", "|---|---:|---:|---:|"]
    for k, (n, v) in sorted(agg.items(), key=lambda kv: -kv[1][1]):
        out.append("| %s | %d | %.1f | %.1f%% |" % (k, n, v, 100.0 * v / tot))
    out += ["", "In launch order, us:", "", "```", ", ".join("%s %.1f" % (k, v) for k, v in one), "```"]
    p = os.path.join(ROOT, "profiles", "%s_launches_config%d.md" % (tag, cfg))
    open(p, "w").write("\n".join(out) + "\n")
    print("wrote", p)


if __name__ == "__main__":
    mode, path, cfg, tag = sys.argv[1], sys.argv[2], int(sys.argv[3]), sys.argv[4]
    (do_full if mode == "full" else do_list)(path, cfg, tag)
