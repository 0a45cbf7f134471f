#!/usr/bin/env python
"""Writes tests/golden/fullsize_config<C>.npz: the ORACLE's result on BASELINE.json's full-size configs,
so that the -m gpu parity tests can compare EVERY element (config 1, 2) or every band element plus a
large random far sample (config 4) without re-paying the oracle (config 2: ~25 min on 8 cores).

Calls only `oracle/` (the CPU oracle) and `workloads/` (the seeded input generator).  No value in the
files it writes comes from the CUDA path.  SURVEY.md 8(d) "Oracle timing": "Oracle results are cached on
disk keyed by a hash of the input arrays".

    python tests/golden/make_fullsize_golden.py --config 1 [--nproc 8]

Stored per config (np.savez_compressed):
    input_sha256   hash of xyz | conn27 | faces bytes (the test refuses a golden whose inputs differ)
    ids            int64 [n]   global element ids covered (config 1, 2: all elements, stored as empty = "all")
    labels         int8  [n]   HOLE 0 / NORMAL 1 / CUT 2
    flags          uint8 [n]   ORC_FLAG_* (1 ambiguous, 2 sign-ambiguous, 4 far, 8 depth)
    near_pos       int64 [m]   positions (into ids) of the elements with |sdist| < d_band
    near_sdist     f64   [m]   their signed distance (every other element has sdist = +-d_band by its label)
    l_ref, tau_cut, d_band, seconds, nproc, n_pair_tests, n_box_tests, n_patchpair

Config 4 (7.1 M elements x 49 152 faces): the candidates are the elements whose centroid lies within
`3.0 * h` (h = 2 / N) of the ANALYTIC surface (workloads' surf_margin: no method arithmetic), a superset of
the band by a wide margin (d_band ~ 1.5 h); the test asserts that every element the CUDA path puts inside
the band is covered.  20 000 uniformly random other elements are added.
"""
from __future__ import annotations

import argparse
import hashlib
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from oracle import dc_oracle as O          # noqa: E402
from workloads import make_config          # noqa: E402


def input_hash(xyz, conn27, faces) -> str:
    h = hashlib.sha256()
    for a in (xyz, conn27, faces):
        h.update(np.ascontiguousarray(a).tobytes())
    return h.hexdigest()


def golden_path(config: int) -> str:
    return os.path.join(HERE, "fullsize_config%d.npz" % config)


def candidate_ids(w, n_far: int, seed: int) -> np.ndarray:
    """Config 4: centroid within 3 h of the analytic surface + n_far random others."""
    cen = w.xyz[w.conn27[:, 13]]
    h = 2.0 / w.N
    near = np.zeros(w.n_elem, bool)
    step = 1 << 20
    for s in range(0, w.n_elem, step):
        near[s:s + step] = w.surf_margin(cen[s:s + step]) < 3.0 * h
    rng = np.random.default_rng(seed)
    far = rng.choice(np.nonzero(~near)[0], size=n_far, replace=False)
    return np.sort(np.concatenate([np.nonzero(near)[0], far])).astype(np.int64)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, required=True, choices=[1, 2, 4])
    ap.add_argument("--nproc", type=int, default=max(1, len(os.sched_getaffinity(0))))
    ap.add_argument("--n-far", type=int, default=20000)
    args = ap.parse_args()
    O.build()
    w = make_config(args.config)
    d_band = O.auto_d_band(w.xyz, w.conn27, w.faces)
    t0 = time.perf_counter()
    if args.config == 4:
        ids = candidate_ids(w, args.n_far, seed=4)
        ref = O.classify(w.xyz, w.conn27, w.faces, elem_ids=ids, nproc=args.nproc, d_band=d_band)
    else:
        ids = np.empty(0, np.int64)             # = all elements
        ref = O.classify(w.xyz, w.conn27, w.faces, nproc=args.nproc, d_band=d_band)
    sec = time.perf_counter() - t0
    assert ref.stats["n_depth_exceeded"] == 0
    near = np.nonzero(np.abs(ref.sdist) < d_band)[0].astype(np.int64)
    # every other element sits exactly on the clamp
    rest = np.ones(ref.sdist.size, bool); rest[near] = False
    sign = np.where(ref.labels == O.HOLE, -1.0, 1.0)
    assert np.array_equal(ref.sdist[rest], (sign * d_band)[rest])
    np.savez_compressed(golden_path(args.config),
                        input_sha256=np.array(input_hash(w.xyz, w.conn27, w.faces)),
                        ids=ids, labels=ref.labels.astype(np.int8), flags=ref.flags.astype(np.uint8),
                        near_pos=near, near_sdist=ref.sdist[near],
                        l_ref=ref.stats["l_ref"], tau_cut=ref.stats["tau_cut"], d_band=d_band,
                        seconds=sec, nproc=ref.nproc, n_pair_tests=ref.stats["n_pair_tests"],
                        n_box_tests=ref.stats["n_box_tests"], n_patchpair=ref.stats["n_patchpair"])
    print("config %d: %d elements in %.1f s on %d processes -> %s (%.2f MB); census hole/normal/cut = %s, "
          "ambiguous %d, sign-ambiguous %d, in band %d"
          % (args.config, ref.labels.size, sec, ref.nproc, golden_path(args.config),
             os.path.getsize(golden_path(args.config)) / 1e6, np.bincount(ref.labels, minlength=3).tolist(),
             int(((ref.flags & O.FLAG_AMBIGUOUS) != 0).sum()), int(((ref.flags & O.FLAG_SIGN_AMBIG) != 0).sum()),
             near.size))


if __name__ == "__main__":
    main()
