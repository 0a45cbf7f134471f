#!/usr/bin/env python
"""bench.py -- one JSON line per run (driver contract).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl reference]

A *step* is one full direct cut of the workload: dc_set_cut_surface (S1 face boxes, S3 face bins)
+ dc_classify with DC_FLAG_RECOMPUTE_BOXES (S2 element boxes from the raw nodes, S4 candidate
pairs, S5 narrow phase, S6 decide, S7 flood fill) -- every row of SURVEY.md 8(a).  Inputs (grid
nodes + connectivity + adjacency, surface faces) are resident in HBM before the timed region.

  metric  : element-face pair tests/s  (pair test = one candidate (element, face) pair processed by
            the narrow phase; BASELINE.json `metric`);   ms_per_step = ms per full direct cut.
  e2e     : the same through dc_classify_host with pinned HOST buffers: faces host->device, labels +
            signed distances device->host inside the timed region (the grid is registered once by
            dc_create_grid, as the paper does for grid-only structures).
  roofline: the dominant kernel (k_np_newton, the closest-point solves of S5; FP64-ALU bound): algorithmic
            flops (device counters x the per-operation constants of DESIGN.md) / its CUDA-event duration
            (events recorded by the library around its launches), against the DFMA peak measured on
            this GPU in this run.  The HBM-bound S2 kernel is reported beside it ("roofline_s2").
  cpu_baseline: the oracle (oracle/dc_oracle.c, as it stands) on this box's host cores on a bounded
            uniform sample of the same workload's elements, each against ALL faces.

--gpus N > 1 (torchrun): the path does not shard: every rank runs an
independent replica of the cut; value = sum over ranks of pair tests / max-over-ranks time.
--impl reference: times the oracle instead (rank 0 only).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "element_face_pair_tests_per_s"
UNIT = "pair tests/s"

# algorithmic fp64 flops per operation of the narrow phase (FMA = 2)
FLOP_PER_BNB_NODE = 434.0       # 2 centre evals with first derivatives, 2 x 8 projected coefficients, 2 scalar ranges, leaf rule
FLOP_PER_NEWTON_EVAL = 560.0    # 6 jets x 36 + (r, g, H) 3 x 43 + LDL^T 4x4 ~75 + trial point and its value 6 x 16 + 17 + tests ~35
FLOP_PER_NEWTON_FINISH = 40.0   # normal, cosine, distance of a finished solve
# S2 algorithmic bytes: every conn row (108 B) and every node (24 B) read once, one box (48 B) written per element


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""

    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None

    def start(self):
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "20"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self) -> dict:
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            c = [x.strip() for x in line.split(",")]
            if len(c) < 9:
                continue
            try:
                sm.append(float(c[1])); mx.append(float(c[2]))
            except ValueError:
                continue
            for nm, v in zip(names, c[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        try:
            os.unlink(self.f.name)
        except OSError:
            pass
        if sm:
            out.update(sm_mhz=statistics.median(sm), sm_max_mhz=max(mx), reasons=sorted(reasons), samples=len(sm))
        return out


def aggregate(units_per_rank_step: float, steps: int, ms_total_this_rank: float, world: int, dist=None):
    """Whole-job throughput: (units all ranks processed) / (max over ranks of the timed region).
    `dist` is torch.distributed when world > 1 (gloo or nccl)."""
    import torch
    t = torch.tensor([ms_total_this_rank, units_per_rank_step * steps], dtype=torch.float64)
    if world > 1:
        dev = torch.device("cuda", torch.cuda.current_device()) if dist.get_backend() == "nccl" else torch.device("cpu")
        tmax = t[:1].clone().to(dev); usum = t[1:].clone().to(dev)
        dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
        dist.all_reduce(usum, op=dist.ReduceOp.SUM)
        ms_total, units = float(tmax.item()), float(usum.item())
    else:
        ms_total, units = float(t[0]), float(t[1])
    return units / (ms_total * 1e-3), ms_total / steps


def workload_name(cfg: int) -> str:
    return {0: "config0 sphere96 x 16^3 straight hexes", 1: "config1 sphere1536 x 64^3 curved hexes",
            2: "config2 dimpled-sphere24576 x 128^3 curved hexes", 3: "config3 spin32 of config2",
            4: "config4 ellipsoids49152 x 192^3 curved hexes"}[cfg]


_D_BAND = {}


def oracle_sample(w, n_sample: int, nproc: int, seed: int = 12345):
    """The oracle on a uniform random sample of the workload's elements (each against ALL faces)."""
    import numpy as np
    from oracle import dc_oracle
    rng = np.random.default_rng(seed)
    ids = np.sort(rng.choice(w.n_elem, size=min(n_sample, w.n_elem), replace=False))
    # (the band width depends on the grid only: computed once per workload, outside every timed interval)
    key = (id(w.xyz), id(w.conn27))
    if key not in _D_BAND:
        _D_BAND[key] = dc_oracle.auto_d_band(w.xyz, w.conn27, w.faces)
    d_band = _D_BAND[key]
    t0 = time.perf_counter()
    ref = dc_oracle.classify(w.xyz, w.conn27[ids], w.faces, nproc=nproc, d_band=d_band)
    sec = time.perf_counter() - t0
    return ids, ref, sec


def run_reference(args, rank: int, world: int):
    """--impl reference: the oracle, as it stands, on the host cores (rank 0 only)."""
    if rank != 0:
        return
    import numpy as np  # noqa: F401
    from oracle import dc_oracle
    from workloads import make_config
    dc_oracle.build()
    w = make_config(args.config)
    cores = max(1, len(os.sched_getaffinity(0)))
    # a bounded sample per step, sized so that the whole --steps K --warmup W run ends within a few minutes: the cost
    # per element is calibrated on 48 elements (one thread), then each step gets its share of a 120 s budget; all the
    # cores (one oracle process each, ~1.5 s to start them) only when a step's share pays for it
    nsteps = max(1, args.steps + args.warmup)
    oracle_sample(w, 8, 1, seed=6)                     # (builds the band width once)
    t0 = time.perf_counter()
    oracle_sample(w, 48, 1, seed=7)
    per_elem = max(1e-5, (time.perf_counter() - t0) / 48)
    share = 120.0 / nsteps
    if args.ref_sample > 0:
        n_sample, nproc = args.ref_sample, cores
    elif share >= 4.0:
        nproc = cores
        n_sample = int(min(1500 * cores, max(32 * cores, (share - 1.5) * cores / per_elem)))
    else:
        nproc = 1
        n_sample = int(max(16, share / per_elem))
    cores = nproc
    times, pairs = [], []
    for it in range(args.warmup + args.steps):
        ids, ref, sec = oracle_sample(w, n_sample, nproc, seed=1000 + it)
        if it >= args.warmup:
            times.append(sec); pairs.append(ref.stats["n_pair_tests"])
    tot = sum(times)
    value = sum(pairs) / tot
    ms_cut = 1e3 * (tot / len(times)) * (w.n_elem / float(len(ids)))
    sample = "%d uniformly sampled elements of %d per step, each against all %d faces" % (len(ids), w.n_elem, w.n_face)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot / len(times),
            "ms_per_full_cut_extrapolated": ms_cut,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(args.config), "n_elem": w.n_elem, "n_face": w.n_face, "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config index (default 2: the dimpled sphere)")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--ref-sample", type=int, default=0)
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "b200" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))

    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import numpy as np
    import torch
    from paper_1711_07663_b200._build import build_lib
    build_lib()
    from paper_1711_07663_b200 import binding as B   # raises if libdc.so is missing: no fallback
    from workloads import make_config

    assert torch.cuda.is_available(), "bench.py needs a B200: there is no CPU fallback"
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    cfg = args.config
    w = make_config(cfg)
    dcut = B.DirectCut(w.xyz, w.conn27, w.adj6, max_faces=w.n_face, device=local_rank)
    if cfg == 3:
        face_sets = [torch.from_numpy(w.spin_faces(s)).cuda(local_rank) for s in range(1, 33)]
    else:
        face_sets = [torch.from_numpy(w.faces).cuda(local_rank)]
    p_full = B.dc_params(); p_full.flags = B.DC_FLAG_RECOMPUTE_BOXES
    p_recut = B.dc_params()
    stream = torch.cuda.current_stream(local_rank)

    def step(i, params):
        dcut.set_cut_surface(face_sets[i % len(face_sets)])
        dcut.classify(params)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- warm-up + correctness of the run itself
    for i in range(args.warmup):
        step(i, p_full)
    st = dcut.stats()
    assert st.status == 0, "device-side status %d" % st.status
    launches_per_step = int(st.n_launches)

    # ---- timed region: (ii) full cut incl. S2 from raw nodes; inputs (634 MB at config 2) exceed L2
    sampler = ClockSampler(local_rank)
    barrier(); sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    stage = np.zeros(8); pairs_total = 0
    ev0.record(stream)
    for i in range(args.steps):
        step(i, p_full)
    ev1.record(stream)
    barrier()
    clocks = sampler.stop()
    ms_total = ev0.elapsed_time(ev1)
    st = dcut.stats()
    # per-step pair count (identical every step except config 3) and per-kernel durations (CUDA events
    # recorded by the library on the caller's stream, last step)
    pairs_per_step = []
    if cfg == 3:
        for i in range(len(face_sets)):
            step(i, p_full); pairs_per_step.append(dcut.stats().n_pairs)
        units_per_step = float(np.mean(pairs_per_step))
    else:
        units_per_step = float(st.n_pairs)
    value, ms_per_step = aggregate(units_per_step, args.steps, ms_total, world, dist)

    # ---- per-stage durations: median over repeated steps (events inside the library)
    reps = max(5, min(args.steps, 20))
    stages, stages_recut = [], []
    for i in range(reps):
        step(i, p_full); s = dcut.stats(); stages.append(list(s.ms_stage))
    for i in range(reps):
        step(i, p_recut); s = dcut.stats(); stages_recut.append(list(s.ms_stage))
    med = np.median(np.array(stages), axis=0)
    med_recut = np.median(np.array(stages_recut), axis=0)
    s_last = dcut.stats()

    # ---- e2e: host buffers through dc_classify_host
    fh = [f.cpu().pin_memory() for f in face_sets]
    lh = torch.empty(w.n_elem, dtype=torch.int8).pin_memory()
    sh = torch.empty(w.n_elem, dtype=torch.float64).pin_memory()
    for i in range(3):
        dcut.classify_host(fh[i % len(fh)], lh, sh, p_full)
    barrier()
    t0 = time.perf_counter()
    ev0.record(stream)
    for i in range(args.steps):
        dcut.classify_host(fh[i % len(fh)], lh, sh, p_full)
    ev1.record(stream)
    barrier()
    ms_e2e_total = max(ev0.elapsed_time(ev1), 0.0)
    wall_e2e = (time.perf_counter() - t0) * 1e3
    ms_e2e_total = max(ms_e2e_total, wall_e2e if world == 1 else ms_e2e_total)
    e2e_value, ms_e2e = aggregate(units_per_step, args.steps, ms_e2e_total, world, dist)
    h2d = int(fh[0].numel() * 8)
    d2h = int(w.n_elem * 9)

    # ---- rooflines
    hbm_peak, hbm_src = _peaks()
    fp64_peak = B.dc_measure_fp64_tflops(local_rank, 4000)
    # dominant kernel: k_np_newton (seed solves, leaf solves, two short launches over the sub-leaves of unconverged
    # solves), timed by CUDA events recorded by the library on the caller's stream around the seed launch and around
    # the other three (two ~7 us k_np_bound passes sit between those and are inside the interval): dc_stats.ms_stage[7]
    newton_flops = s_last.n_newton_iters * FLOP_PER_NEWTON_EVAL + s_last.n_newton * FLOP_PER_NEWTON_FINISH
    newton_ms = float(med[7])
    ach_tf = newton_flops / (newton_ms * 1e-3) / 1e12 if newton_ms > 0 else 0.0
    narrow_ms = float(med[3])
    narrow_flops = newton_flops + s_last.n_bnb_nodes * FLOP_PER_BNB_NODE
    s2_bytes = 108.0 * w.n_elem + 24.0 * len(w.xyz) + 48.0 * w.n_elem
    s2_ms = float(med[1])
    ach_gbs = s2_bytes / (s2_ms * 1e-3) / 1e9 if s2_ms > 0 else 0.0
    roofline = {"kernel": "k_np_newton (S5 closest-point solves: seed, leaf and two overflow launches per cut)", "bound": "alu", "achieved": ach_tf,
                "peak": fp64_peak, "unit": "TFLOP/s",
                "frac": ach_tf / fp64_peak if fp64_peak > 0 else None,
                # dram__bytes_read.sum + dram__bytes_write.sum of its launches in the committed ncu --set full
                # capture (profiles/r1c_kernels_full_config2.md: 48.4 + 0.1 and 121.3 + 5.8 MB, the overflow launches < 0.1 MB), config 2 only
                "traffic": 175.7e6 if cfg in (2, 3) else None,
                "algorithmic_flops_per_cut": newton_flops, "ms_per_cut": newton_ms,
                "peak_source": "measured: dc_measure_fp64_tflops (register-resident DFMA chains on all SMs) in this run",
                "share_of_step": newton_ms / float(med[5] + med[6]) if med[5] > 0 else None,
                "narrow_phase_S5_S6": {"ms": narrow_ms, "algorithmic_flops": narrow_flops,
                                       "achieved_tflops": narrow_flops / (narrow_ms * 1e-3) / 1e12 if narrow_ms > 0 else None}}
    roofline_s2 = {"kernel": "k_elem_boxes (S2)", "bound": "hbm", "achieved": ach_gbs, "peak": hbm_peak, "unit": "GB/s",
                   "frac": ach_gbs / hbm_peak,
                   # same capture: 634.5 MB read + 92.2 MB written (algorithmic: 734 MB), config 2 only
                   "traffic": 726.7e6 if cfg in (2, 3) else None, "algorithmic_bytes": s2_bytes, "peak_source": hbm_src}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(cfg), "n_elem": w.n_elem, "n_face": w.n_face,
                       "step": "full cut: dc_set_cut_surface + dc_classify(DC_FLAG_RECOMPUTE_BOXES)",
                       "l2": "inputs larger than L2 (nodes+conn+adj = %.0f MB)" % ((w.xyz.nbytes + w.conn27.nbytes + w.adj6.nbytes) / 1e6),
                       "parallelism": "replicas only" if world > 1 else "1 gpu"},
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "ms_per_step": ms_e2e, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
            "gpu_launches": launches_per_step * args.steps,
            "roofline": roofline, "roofline_s2": roofline_s2,
            "cut": {"pairs_per_cut": units_per_step, "box_tests_per_cut": int(s_last.n_box_tests),
                    "n_active": int(s_last.n_active), "bnb_nodes": int(s_last.n_bnb_nodes), "newton": int(s_last.n_newton),
                    "newton_iters": int(s_last.n_newton_iters), "newton_fail": int(s_last.n_newton_fail),
                    "census_hole_cut_normal": [int(s_last.n_hole), int(s_last.n_cut), int(s_last.n_normal)],
                    "n_ambiguous": int(s_last.n_ambiguous), "n_sign_ambiguous": int(s_last.n_sign_ambiguous),
                    "ms_full_cut_stages": {"S1+S3": float(med[6]), "S2": float(med[1]), "S4": float(med[2]),
                                           "S5+S6": float(med[3]), "S7": float(med[4]), "classify": float(med[5])},
                    "ms_recut_cached_boxes": float(med_recut[5] + med_recut[6])}}

    # ---- cpu baseline (rank 0, N = 1 only): the oracle on a bounded sample of the same workload
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        from oracle import dc_oracle
        dc_oracle.build()
        cores = max(1, len(os.sched_getaffinity(0)))
        n_sample = args.ref_sample if args.ref_sample > 0 else 1500 * cores
        faces0 = face_sets[0].cpu().numpy()
        w0 = w if cfg != 3 else type(w)(**{**w.__dict__, "faces": faces0})
        ids, ref, sec = oracle_sample(w0, n_sample, cores)
        # parity of this very run on the sample (labels bit-exact off the ambiguous band, sdist 1e-10 L_ref)
        step(0, p_full)
        lab = dcut.labels.cpu().numpy()[ids]; sd = dcut.sdist.cpu().numpy()[ids]
        amb = (ref.flags & dc_oracle.FLAG_AMBIGUOUS) != 0
        mism = int(((lab != ref.labels) & ~amb).sum())
        err = float(np.abs(sd - ref.sdist)[~amb].max())
        line["cpu_baseline"] = {"value": ref.stats["n_pair_tests"] / sec, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": "%d uniformly sampled elements of %d, each against all %d faces" % (len(ids), w.n_elem, w.n_face),
                                "seconds": sec, "ms_per_full_cut_extrapolated": 1e3 * sec * w.n_elem / len(ids),
                                "parity_on_sample": {"label_mismatches": mism, "ambiguous": int(amb.sum()),
                                                     "max_abs_dsdist_over_lref": err / ref.stats["l_ref"]}}
    dcut.close()
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(line), flush=True)


if __name__ == "__main__":
    main()
