#!/usr/bin/env python
"""bench.py -- one JSON line per run (driver contract).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl reference]

A *step* is one full direct cut of the workload: dc_set_cut_surface (S1 face boxes, S3 face bins)
+ dc_classify with DC_FLAG_RECOMPUTE_BOXES (S2 element boxes from the raw nodes, S4 candidate
pairs, S5 narrow phase, S6 decide, S7 flood fill) -- every row of SURVEY.md 8(a).  Inputs (grid
nodes + connectivity + adjacency, surface faces) are resident in HBM before the timed region.

  metric  : element-face pair tests/s.  A pair test = one candidate (element, face) pair -- face box within
            `reach` = d_band + 2 tau + t_tie of the element box, Algorithm A.2 -- resolved by the narrow phase
            (BASELINE.json `metric`).  The count grows with d_band, so `config.d_band` is part of the unit;
            ms_per_step = ms per full direct cut is the figure that does not.
  e2e     : the same through dc_classify_host with pinned HOST buffers: faces host->device, labels +
            signed distances device->host inside the timed region (the grid is registered once by
            dc_create_grid, as the paper does for grid-only structures).
  roofline: the dominant kernel by time (k_np_bound, the branch and bound of S5; FP64-ALU bound): algorithmic
            flops (device counter x the per-node constant of DESIGN.md) / its CUDA-event duration (events the
            library records around its launches, dc_stats.ms_kernel), against the DFMA peak measured on this GPU in
            this run.  Beside it: `roofline_solve` (every k_np_solve launch, ALU), `roofline_s2` (k_elem_boxes, HBM)
            and the phase-level `roofline_broad` (S1-S4 algorithmic bytes / their event time, HBM).
  cpu_baseline: the oracle (oracle/dc_oracle.c, as it stands) on this box's host cores on a bounded
            uniform sample of the same workload's elements, each against ALL faces; `value` counts the SAME
            candidate pairs as the GPU line (those of the sampled elements), per oracle second.
  paper_mode: the paper's own approximate cut (DC_FLAG_PAPER_MODE) on the same context: ms, labels differing from the exact mode.
  exact_far: DC_FLAG_EXACT_FAR on the same context (exact distance beyond the band too, "d_band = infinity"): ms of the far pass,
            far elements, candidate pairs, passes.
  donor_search: the paper's other GPU algorithm (4.3: ADT stack search + Newton point containment), 1 M points.
  per_config: the other BASELINE.json configs (0, 1, 3 incl. the sum over its 32 steps, 4), a few seconds each,
            every one with its own clock record over a timed region of at least 200 ms.

--gpus N > 1 (torchrun): the path does not shard: every rank runs an
independent replica of the cut; value = sum over ranks of pair tests / max-over-ranks time.
--impl reference: times the oracle instead (rank 0 only).
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import statistics
import subprocess
import sys
import tempfile
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "element_face_pair_tests_per_s"
UNIT = "pair tests/s"

# algorithmic fp64 flops per operation of the narrow phase (FMA = 2)
FLOP_PER_BNB_NODE = 920.0       # centre evals with first derivatives 183, norms + leaf rule 45, model closest pair 320 (4 sweeps), true patches there 120,
#                                 2 x 8 projected coefficients 80, 2 Bernstein ranges 170
FLOP_PER_BNB_ROOT = 655.0       # a whole patch pair (round 0): no centre evaluation (-180), no re-centring in the two ranges (-85)
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


def source_hash() -> str:
    """sha256 (first 16 hex digits) of the CUDA sources + the C ABI: what a stored ncu figure belongs to."""
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_1711_07663_b200", "csrc")
    for name in sorted(os.listdir(d)):
        with open(os.path.join(d, name), "rb") as f:
            h.update(name.encode()); h.update(f.read())
    with open(os.path.join(ROOT, "include", "dc.h"), "rb") as f:
        h.update(f.read())
    return h.hexdigest()[:16]


def stored_traffic(cfg: int) -> dict:
    """DRAM bytes per launch of the rooflined kernels from the committed ncu capture (profiles/r2_dram_traffic.csv,
    written by paper_1711_07663_b200/profile_summary.py): only if it was taken on THESE sources and this config."""
    p = os.path.join(ROOT, "profiles", "r2_dram_traffic.csv")
    out = {}
    if not os.path.exists(p):
        return out
    with open(p) as f:
        lines = f.read().splitlines()
    meta = dict(kv.split("=") for kv in lines[0].lstrip("# ").split() if "=" in kv) if lines else {}
    if meta.get("src_sha16") != source_hash() or int(meta.get("config", -1)) != cfg:
        return out
    for ln in lines[2:]:
        c = ln.split(",")
        if len(c) >= 4:
            out[c[0]] = float(c[2]) + float(c[3])
    return out


class ClockSampler:
    """SM clock and clock-event reasons DURING the timed region: NVML polled from a thread (about 1 kHz: a 30 ms
    region still gets tens of samples); `nvidia-smi -lms 20` (B200_PROFILING.md recipe) if NVML is not importable."""

    REASONS = ((0x8, "hw_slowdown"), (0x40, "hw_thermal_slowdown"), (0x20, "sw_thermal_slowdown"), (0x4, "sw_power_cap"))
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.h = None
        self.sm, self.bits, self.mx = [], 0, None
        self.stop_flag = False
        self.t = None
        self.p = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            h = None
            try:
                import torch
                uuid = str(torch.cuda.get_device_properties(index).uuid)
                h = pynvml.nvmlDeviceGetHandleByUUID(("GPU-" + uuid) if not uuid.startswith("GPU-") else uuid)
            except Exception:
                h = None
            self.h = h if h is not None else pynvml.nvmlDeviceGetHandleByIndex(index)
            self.mx = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.h = None

    def _poll(self):
        nv = self.nv
        get_reasons = getattr(nv, "nvmlDeviceGetCurrentClocksEventReasons", None) or nv.nvmlDeviceGetCurrentClocksThrottleReasons
        while not self.stop_flag:
            try:
                self.sm.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                self.bits |= int(get_reasons(self.h))
            except Exception:
                pass
            time.sleep(0.0005)

    def start(self):
        if self.h is not None:
            self.t = threading.Thread(target=self._poll, daemon=True)
            self.t.start()
            return
        try:
            self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "20"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self) -> dict:
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0, "source": "nvml"}
        if self.t is not None:
            self.stop_flag = True
            self.t.join(timeout=2)
            if self.sm:
                out.update(sm_mhz=statistics.median(self.sm), sm_max_mhz=self.mx, samples=len(self.sm),
                           reasons=[n for b, n in self.REASONS if self.bits & b])
            return out
        out["source"] = "nvidia-smi"
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush(); self.f.seek(0)
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


def candidate_pairs_by_oracle_boxes(w, ids, reach: float, max_elems: int = 1500):
    """The metric's unit counted WITHOUT the GPU (for --impl reference): candidate pairs = (element, face) whose
    Bezier boxes are within `reach` (Algorithm A.2).  Boxes come from the oracle's own exported routines; the
    count is taken on at most `max_elems` of the sampled elements and scaled."""
    import ctypes as C
    import numpy as np
    from oracle import dc_oracle
    L = dc_oracle.lib()
    dp = C.POINTER(C.c_double)
    sub = ids if len(ids) <= max_elems else ids[np.linspace(0, len(ids) - 1, max_elems).astype(int)]
    xyz = np.ascontiguousarray(w.xyz, np.float64)
    eb = np.empty((len(sub), 6))
    for i, e in enumerate(sub):
        row = np.ascontiguousarray(w.conn27[e], np.int32)
        L.orc_element_box(xyz.ctypes.data_as(dp), row.ctypes.data_as(C.POINTER(C.c_int)), eb[i].ctypes.data_as(dp))
    faces = np.ascontiguousarray(w.faces, np.float64)
    bez = np.empty((w.n_face, 9, 3))
    for f in range(w.n_face):
        L.orc_lagrange_to_bezier(faces[f].ctypes.data_as(dp), bez[f].ctypes.data_as(dp))
    flo, fhi = bez.min(axis=1), bez.max(axis=1)
    n = 0
    for i in range(len(sub)):
        g = np.maximum(0.0, np.maximum(flo - eb[i, 3:], eb[i, :3] - fhi))
        n += int(((g * g).sum(axis=1) <= reach * reach).sum())
    return n * (len(ids) / float(len(sub)))


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
    times, own_pairs, cand_per_elem = [], [], None
    for it in range(args.warmup + args.steps):
        ids, ref, sec = oracle_sample(w, n_sample, nproc, seed=1000 + it)
        if it >= args.warmup:
            times.append(sec); own_pairs.append(ref.stats["n_pair_tests"])
            if cand_per_elem is None:
                # (outside the timed interval, once: the samples are uniform, so one of them gives the candidates per element)
                reach = ref.stats["d_band"] + 2.0 * ref.stats["tau_cut"] + 1e-9 * ref.stats["l_ref"]
                cand_per_elem = candidate_pairs_by_oracle_boxes(w, ids, reach) / float(len(ids))
    tot = sum(times)
    value = cand_per_elem * len(ids) * len(times) / tot
    ms_cut = 1e3 * (tot / len(times)) * (w.n_elem / float(len(ids)))
    sample = "%d uniformly sampled elements of %d per step, each against all %d faces" % (len(ids), w.n_elem, w.n_face)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot / len(times),
            "ms_per_full_cut_extrapolated": ms_cut,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(args.config), "n_elem": w.n_elem, "n_face": w.n_face, "sample": sample,
                       "d_band": _D_BAND[(id(w.xyz), id(w.conn27))],
                       "unit_note": "candidate pairs (boxes within reach, A.2) of the sampled elements per oracle second; "
                                    "the oracle's own count of faces it refines is in cpu_baseline.oracle_pair_tests_per_s"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                             "oracle_pair_tests_per_s": sum(own_pairs) / tot},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def time_cuts(dcut, face_sets, params, n_cuts: int, stream, torch):
    """n_cuts cuts back to back between two CUDA events on the caller's stream -> total ms."""
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record(stream)
    for i in range(n_cuts):
        dcut.cut(face_sets[i % len(face_sets)], params)
    ev1.record(stream)
    torch.cuda.synchronize()
    return ev0.elapsed_time(ev1)


def measure_paper_mode(dcut, faces, B, stream, torch, np, n_cuts: int = 10):
    """the paper's own approximate cut (DC_FLAG_PAPER_MODE: A.1, A.3, A.4, 16 -> 4 faces, linear
    triangles, L215) on the same context: ms per full cut, and how its labels and distances differ from the exact mode's
    (which is element-by-element equal to the oracle in the -m gpu tests)."""
    p_exact = B.dc_params(); p_exact.flags = B.DC_FLAG_RECOMPUTE_BOXES
    p_paper = B.dc_params(); p_paper.flags = B.DC_FLAG_RECOMPUTE_BOXES | B.DC_FLAG_PAPER_MODE
    dcut.set_cut_surface(faces); dcut.classify(p_exact)
    lab0 = dcut.labels.clone(); sd0 = dcut.sdist.clone()
    st0 = dcut.stats()
    for _ in range(2):
        dcut.set_cut_surface(faces); dcut.classify(p_paper)
    ms = time_cuts(dcut, [faces], p_paper, n_cuts, stream, torch) / n_cuts
    st = dcut.stats()
    lab1, sd1 = dcut.labels, dcut.sdist
    diff = lab1 != lab0
    out = {"ms_per_full_cut": ms, "ms_S5_S6": float(st.ms_stage[3]), "ms_S5_S6_exact_mode": float(st0.ms_stage[3]),
           "labels_differing_from_exact": int(diff.sum().item()), "band_elements": int(st.band_needed),
           "cut_in_exact_only": int(((lab0 == 2) & (lab1 != 2)).sum().item()), "cut_in_paper_only": int(((lab1 == 2) & (lab0 != 2)).sum().item()),
           "hole_normal_swapped": int((diff & (lab0 != 2) & (lab1 != 2)).sum().item()),
           "max_abs_dsdist_over_lref": float((sd1 - sd0).abs().max().item() / st.l_ref),
           "census_hole_cut_normal": [int(st.n_hole), int(st.n_cut), int(st.n_normal)]}
    dcut.set_cut_surface(faces); dcut.classify(p_exact)
    return out


def measure_exact_far(dcut, faces, B, stream, torch, np, n_cuts: int = 3):
    """SURVEY.md 8(f) NEXT-4 (second half): DC_FLAG_EXACT_FAR on the same context -- the banded cut, then the exact distance
    of every element it left clamped.  Wall clock of the far pass (it synchronises after each of its passes), its
    element and pair counts, and that the labels and the band's distances are those of the banded cut."""
    p_band = B.dc_params(); p_band.flags = B.DC_FLAG_RECOMPUTE_BOXES
    p_far = B.dc_params(); p_far.flags = B.DC_FLAG_RECOMPUTE_BOXES | B.DC_FLAG_EXACT_FAR
    dcut.set_cut_surface(faces); dcut.classify(p_band)
    lab0 = dcut.labels.clone(); sd0 = dcut.sdist.clone()
    st0 = dcut.stats()
    ms_far, ms_all = [], []
    for i in range(n_cuts + 1):
        torch.cuda.synchronize(); t0 = time.perf_counter()
        dcut.set_cut_surface(faces); dcut.classify(p_far)
        torch.cuda.synchronize(); t1 = time.perf_counter()
        st = dcut.stats()
        if i:
            ms_far.append(float(st.ms_far)); ms_all.append((t1 - t0) * 1e3)
    lab1, sd1 = dcut.labels, dcut.sdist
    inband = sd0.abs() < st0.d_band
    out = {"ms_far_pass": statistics.median(ms_far), "ms_full_cut_with_far_pass_wall": statistics.median(ms_all),
           "ms_banded_cut": float(st0.ms_stage[5]) + float(st0.ms_stage[0]),
           "far_elements": int(st.n_far), "far_elements_done": int(st.n_far_done), "far_pairs": int(st.far_pairs),
           "passes": int(st.far_passes), "max_pairs": int(dcut.max_pairs),
           "far_elements_per_s": st.n_far / (statistics.median(ms_far) * 1e-3) if st.n_far else 0.0,
           "labels_equal_banded": bool((lab1 == lab0).all().item()),
           "band_sdist_equal_banded": bool((sd1[inband] == sd0[inband]).all().item()),
           "min_abs_far_sdist_over_d_band": float((sd1[~inband & (lab1 != 2)].abs().min().item() / st0.d_band)) if bool((~inband & (lab1 != 2)).any().item()) else None,
           "max_abs_sdist": float(sd1.abs().max().item())}
    dcut.set_cut_surface(faces); dcut.classify(p_band)
    return out


def measure_other_config(cfg: int, B, local_rank: int, torch, np, min_ms: float = 200.0):
    """One of the other BASELINE.json configs: full cut and re-cut, each over a timed region of at least `min_ms` with its
    own clock record; config 3: every one of its 32 steps and their sum (re-cut path: the grid is fixed)."""
    from workloads import make_config
    w = make_config(2 if cfg == 3 else cfg)
    dcut = B.DirectCut(w.xyz, w.conn27, w.adj6, max_faces=w.n_face, device=local_rank)
    stream = torch.cuda.current_stream(local_rank)
    if cfg == 3:
        face_sets = [torch.from_numpy(w.spin_faces(s)).cuda(local_rank) for s in range(1, 33)]
    else:
        face_sets = [torch.from_numpy(w.faces).cuda(local_rank)]
    p_full = B.dc_params(); p_full.flags = B.DC_FLAG_RECOMPUTE_BOXES | B.DC_FLAG_GRAPH
    p_recut = B.dc_params(); p_recut.flags = B.DC_FLAG_GRAPH
    for i in range(3):
        dcut.cut(face_sets[i % len(face_sets)], p_full)
    probe = time_cuts(dcut, face_sets, p_full, len(face_sets), stream, torch) / len(face_sets)
    n = max(len(face_sets), int(np.ceil(min_ms / max(probe, 1e-3))))
    n = ((n + len(face_sets) - 1) // len(face_sets)) * len(face_sets)
    out = {"workload": workload_name(cfg), "n_elem": w.n_elem, "n_face": w.n_face}
    for name, prm in (("full_cut", p_full), ("recut_cached_boxes", p_recut)):
        sampler = ClockSampler(local_rank); torch.cuda.synchronize(); sampler.start()
        ms = time_cuts(dcut, face_sets, prm, n, stream, torch)
        out[name] = {"ms_per_cut": ms / n, "cuts_timed": n, "clocks": sampler.stop()}
    st = dcut.stats()
    assert st.status == 0
    out.update(pairs_per_cut=int(st.n_pairs), d_band=st.d_band,
               census_hole_cut_normal=[int(st.n_hole), int(st.n_cut), int(st.n_normal)],
               n_ambiguous=int(st.n_ambiguous), n_sign_ambiguous=int(st.n_sign_ambiguous))
    if cfg == 3:
        # every step once per sweep, 5 sweeps, median per step: (i) re-cut with cached grid data per step, (ii) full for step 1
        sweeps = []
        for _ in range(5):
            row = []
            for s in range(32):
                row.append(time_cuts(dcut, [face_sets[s]], p_recut, 1, stream, torch))
            sweeps.append(row)
        per_step = np.median(np.array(sweeps), axis=0)
        first_full = statistics.median(time_cuts(dcut, [face_sets[0]], p_full, 1, stream, torch) for _ in range(5))
        out["spin32"] = {"ms_per_step_recut": [round(float(x), 4) for x in per_step],
                         "ms_sum_32_steps_recut": float(per_step.sum()),
                         "ms_step1_full_cut": float(first_full),
                         "ms_sum_32_steps_step1_full": float(per_step[1:].sum() + first_full)}
    if cfg != 3:
        out["paper_mode"] = measure_paper_mode(dcut, face_sets[0], B, stream, torch, np)
        out["exact_far"] = measure_exact_far(dcut, face_sets[0], B, stream, torch, np)
    dcut.close()
    del dcut, face_sets
    torch.cuda.empty_cache()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config index (default 2: the dimpled sphere)")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-per-config", action="store_true", help="skip the per_config block (configs 0, 1, 3, 4)")
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
    # everything below runs on ONE stream of our own, not the legacy default stream: dc_cut replays the cut's launch
    # sequence from a CUDA graph (DC_FLAG_GRAPH), and the default stream cannot be captured
    torch.cuda.set_stream(torch.cuda.Stream(local_rank))
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
    p_full = B.dc_params(); p_full.flags = B.DC_FLAG_RECOMPUTE_BOXES | B.DC_FLAG_GRAPH
    p_recut = B.dc_params(); p_recut.flags = B.DC_FLAG_GRAPH
    stream = torch.cuda.current_stream(local_rank)

    def step(i, params):
        dcut.cut(face_sets[i % len(face_sets)], params)

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

    # ---- per-stage and per-kernel durations: median over repeated steps (events inside the library)
    reps = max(5, min(args.steps, 20))
    stages, kernels, stages_recut = [], [], []
    # (plain launches: the library's stage events are left out of the replayed graph)
    p_full_ev = B.dc_params(); p_full_ev.flags = B.DC_FLAG_RECOMPUTE_BOXES
    p_recut_ev = B.dc_params()
    for i in range(reps):
        step(i, p_full_ev); s = dcut.stats(); stages.append(list(s.ms_stage)); kernels.append(list(s.ms_kernel))
    for i in range(reps):
        step(i, p_recut_ev); s = dcut.stats(); stages_recut.append(list(s.ms_stage))
    med = np.median(np.array(stages), axis=0)
    medk = np.median(np.array(kernels), axis=0)
    med_recut = np.median(np.array(stages_recut), axis=0)
    n_rc = max(20, len(face_sets))
    for i in range(len(face_sets)):
        step(i, p_recut)
    ms_recut_graph = time_cuts(dcut, face_sets, p_recut, n_rc, stream, torch) / n_rc
    step(0, p_full_ev)
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
    fp64_src = "measured: dc_measure_fp64_tflops (register-resident DFMA chains on all SMs) in this run"
    traffic = stored_traffic(cfg)
    step_ms = float(med[5] + med[6])
    # dominant kernel by time: k_np_bound (all rounds: four grids and the one-CTA tail; round 0 holds 97 % of the nodes)
    n_root = min(int(s_last.n_root_nodes), int(s_last.n_bnb_nodes))
    bound_flops = n_root * FLOP_PER_BNB_ROOT + (s_last.n_bnb_nodes - n_root) * FLOP_PER_BNB_NODE
    bound_ms = float(medk[3])
    ach_b = bound_flops / (bound_ms * 1e-3) / 1e12 if bound_ms > 0 else 0.0
    roofline = {"kernel": "k_np_bound (S5 branch and bound: 4 grid rounds + tail, round 0 = 97 % of the nodes)", "bound": "alu",
                "achieved": ach_b, "peak": fp64_peak, "unit": "TFLOP/s", "frac": ach_b / fp64_peak if fp64_peak > 0 else None,
                "traffic": traffic.get("k_np_bound"),
                "algorithmic_flops_per_cut": bound_flops, "flop_per_node": FLOP_PER_BNB_NODE, "flop_per_root_node": FLOP_PER_BNB_ROOT,
                "nodes_per_cut": int(s_last.n_bnb_nodes), "root_nodes_per_cut": n_root,
                "ms_per_cut": bound_ms, "peak_source": fp64_src, "share_of_step": bound_ms / step_ms if step_ms > 0 else None}
    # every k_np_solve launch (seeds, three leaf passes, two overflow rounds -- the latter with their two short bound passes)
    newton_flops = s_last.n_newton_iters * FLOP_PER_NEWTON_EVAL + s_last.n_newton * FLOP_PER_NEWTON_FINISH
    newton_ms = float(med[7])
    ach_tf = newton_flops / (newton_ms * 1e-3) / 1e12 if newton_ms > 0 else 0.0
    leaf_ms = float(medk[5])
    narrow_ms = float(med[3])
    narrow_flops = newton_flops + bound_flops
    roofline_solve = {"kernel": "k_np_solve (S5 closest-point solves: seeds, three leaf passes, two overflow rounds)", "bound": "alu",
                      "achieved": ach_tf, "peak": fp64_peak, "unit": "TFLOP/s", "frac": ach_tf / fp64_peak if fp64_peak > 0 else None,
                      "traffic": traffic.get("k_np_solve"), "algorithmic_flops_per_cut": newton_flops, "ms_per_cut": newton_ms,
                      "ms_leaf_passes": leaf_ms, "ms_seeds": float(medk[1]), "ms_overflow_rounds": float(medk[6]),
                      "evaluations_per_cut": int(s_last.n_newton_iters), "solves_per_cut": int(s_last.n_newton),
                      "share_of_step": newton_ms / step_ms if step_ms > 0 else None, "peak_source": fp64_src,
                      "narrow_phase_S5_S6": {"ms": narrow_ms, "algorithmic_flops": narrow_flops,
                                             "achieved_tflops": narrow_flops / (narrow_ms * 1e-3) / 1e12 if narrow_ms > 0 else None,
                                             "frac": narrow_flops / (narrow_ms * 1e-3) / 1e12 / fp64_peak if narrow_ms > 0 and fp64_peak > 0 else None}}
    s2_bytes = 108.0 * w.n_elem + 24.0 * len(w.xyz) + 48.0 * w.n_elem
    s2_ms = float(med[1])
    ach_gbs = s2_bytes / (s2_ms * 1e-3) / 1e9 if s2_ms > 0 else 0.0
    roofline_s2 = {"kernel": "k_elem_boxes (S2)", "bound": "hbm", "achieved": ach_gbs, "peak": hbm_peak, "unit": "GB/s",
                   "frac": ach_gbs / hbm_peak, "traffic": traffic.get("k_elem_boxes"), "algorithmic_bytes": s2_bytes, "peak_source": hbm_src}
    # the broad PHASE S1-S4: faces read + boxes/coefficients written (27 + 6 + 6 + 28 doubles per face), S2 as above, element
    # boxes read once more by S4, the pair list written (face id 4 B, key 8 B, band index 4 B per pair)
    broad_bytes = 8.0 * (27 + 6 + 6 + 28) * w.n_face + s2_bytes + 48.0 * w.n_elem + 16.0 * units_per_step
    broad_ms = float(med[6] + med[1] + med[2])
    broad_gbs = broad_bytes / (broad_ms * 1e-3) / 1e9 if broad_ms > 0 else 0.0
    roofline_broad = {"phase": "S1-S4 (dc_set_cut_surface + k_elem_boxes + k_filter + k_pairs)", "bound": "hbm", "achieved": broad_gbs,
                      "peak": hbm_peak, "unit": "GB/s", "frac": broad_gbs / hbm_peak, "algorithmic_bytes": broad_bytes, "ms": broad_ms,
                      "peak_source": hbm_src}

    names_k = ["k_np_stage", "k_np_solve seeds", "k_np_roots", "k_np_bound rounds", "k_np_compact", "k_np_solve leaf passes",
               "overflow rounds", "k_np_decide"]
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(cfg), "n_elem": w.n_elem, "n_face": w.n_face,
                       "step": "full cut: dc_cut = dc_set_cut_surface + dc_classify(DC_FLAG_RECOMPUTE_BOXES); its launch sequence replayed from a CUDA graph (DC_FLAG_GRAPH), every kernel runs every step",
                       "d_band": float(s_last.d_band), "reach": float(s_last.d_band + 2 * s_last.tau_cut + 1e-9 * s_last.l_ref),
                       "unit_note": "a pair test is a candidate pair (boxes within reach): the count is tied to d_band; ms_per_step is not",
                       "l2": "inputs larger than L2 (nodes+conn+adj = %.0f MB)" % ((w.xyz.nbytes + w.conn27.nbytes + w.adj6.nbytes) / 1e6),
                       "parallelism": "replicas only" if world > 1 else "1 gpu", "src_sha16": source_hash()},
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "ms_per_step": ms_e2e, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
            "gpu_launches": launches_per_step * args.steps,
            "roofline": roofline, "roofline_solve": roofline_solve, "roofline_s2": roofline_s2, "roofline_broad": roofline_broad,
            "cut": {"pairs_per_cut": units_per_step, "box_tests_per_cut": int(s_last.n_box_tests),
                    "n_active": int(s_last.n_active), "bnb_nodes": int(s_last.n_bnb_nodes), "newton": int(s_last.n_newton),
                    "newton_iters": int(s_last.n_newton_iters), "newton_fail": int(s_last.n_newton_fail),
                    "census_hole_cut_normal": [int(s_last.n_hole), int(s_last.n_cut), int(s_last.n_normal)],
                    "n_ambiguous": int(s_last.n_ambiguous), "n_sign_ambiguous": int(s_last.n_sign_ambiguous),
                    "ms_full_cut_stages": {"S1+S3": float(med[6]), "S2": float(med[1]), "S4": float(med[2]),
                                           "S5+S6": float(med[3]), "S7": float(med[4]), "classify": float(med[5])},
                    "ms_S5_S6_kernels": {n: float(v) for n, v in zip(names_k, medk)},
                    "ms_full_cut_plain_launches": float(med[5] + med[6]),
                    "ms_recut_cached_boxes_plain_launches": float(med_recut[5] + med_recut[6]),
                    "ms_recut_cached_boxes": float(ms_recut_graph),
                    "note": "stage and kernel times: plain launches with the library's CUDA events (they are left out of the "
                            "replayed graph); ms_per_step and ms_recut_cached_boxes: graph replay"}}

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
        # the SAME unit as the GPU line: the candidate pairs of the sampled elements (this cut's own pair list)
        pe, _pf = dcut.pairs()
        sel = np.zeros(w.n_elem, bool); sel[ids] = True
        cand = int(sel[pe].sum())
        line["cpu_baseline"] = {"value": cand / sec, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": "%d uniformly sampled elements of %d, each against all %d faces" % (len(ids), w.n_elem, w.n_face),
                                "seconds": sec, "ms_per_full_cut_extrapolated": 1e3 * sec * w.n_elem / len(ids),
                                "candidate_pairs_of_sample": cand,
                                "oracle_box_tests_per_s": ref.stats["n_box_tests"] / sec,
                                "oracle_pair_tests_per_s": ref.stats["n_pair_tests"] / sec,
                                "oracle_patchpair_calls_per_s": ref.stats["n_patchpair"] / sec,
                                "gpu_box_tests_per_s": float(s_last.n_box_tests) / (ms_per_step * 1e-3),
                                "parity_on_sample": {"label_mismatches": mism, "ambiguous": int(amb.sum()),
                                                     "max_abs_dsdist_over_lref": err / ref.stats["l_ref"]}}
    if rank == 0 and world == 1 and cfg != 3 and not args.no_per_config:
        line["paper_mode"] = measure_paper_mode(dcut, face_sets[0], B, stream, torch, np)
        line["exact_far"] = measure_exact_far(dcut, face_sets[0], B, stream, torch, np)
        # the paper's other GPU algorithm (4.3): ADT stack search + Newton point containment, 1 M query points
        t0 = time.perf_counter(); dcut.build_adt(); t_build = time.perf_counter() - t0
        q = (torch.rand((1 << 20, 3), dtype=torch.float64, device="cuda:%d" % local_rank) * 1.9 - 0.95)
        dcut.find_donors(q)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(5):
            donor, _ref = dcut.find_donors(q)
        e1.record(stream); torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / 5
        line["donor_search"] = {"points": int(q.shape[0]), "ms": ms, "points_per_s": q.shape[0] / (ms * 1e-3),
                                "found": int((donor >= 0).sum().item()), "adt_build_host_s": t_build}
    dcut.close()
    del dcut
    torch.cuda.empty_cache()

    # ---- the other configs, a few seconds each (rank 0, N = 1, default config only)
    if rank == 0 and world == 1 and cfg == 2 and not args.no_per_config:
        line["per_config"] = {}
        for c in (0, 1, 3, 4):
            line["per_config"]["config%d" % c] = measure_other_config(c, B, local_rank, torch, np)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(line), flush=True)


if __name__ == "__main__":
    main()
