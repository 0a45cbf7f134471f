"""ctypes front end of the CPU oracle (oracle/dc_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It never imports the CUDA package and the CUDA package never imports it.
"""
from __future__ import annotations

import ctypes as C
import multiprocessing as mp
import os
import subprocess
import time
from dataclasses import dataclass
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dc_oracle.c")
_SRC_PAPER = os.path.join(_HERE, "paper_oracle.c")     # the paper's approximate mode (oracle/paper_oracle.py)
_LIB = os.path.join(_HERE, "liboracle_dc.so")

HOLE, NORMAL, CUT = 0, 1, 2
FLAG_AMBIGUOUS, FLAG_SIGN_AMBIG, FLAG_FAR, FLAG_DEPTH = 1, 2, 4, 8


class OrcParams(C.Structure):
    _fields_ = [("tau_cut_rel", C.c_double), ("d_band", C.c_double), ("l_ref", C.c_double),
                ("eps_rel", C.c_double), ("eps_far_rel", C.c_double), ("tie_rel", C.c_double),
                ("max_depth", C.c_int), ("reserved", C.c_int)]


class OrcStats(C.Structure):
    _fields_ = [("n_box_tests", C.c_longlong), ("n_pair_tests", C.c_longlong),
                ("n_patchpair", C.c_longlong), ("n_subpairs", C.c_longlong),
                ("n_depth_exceeded", C.c_longlong),
                ("n_cut", C.c_longlong), ("n_hole", C.c_longlong), ("n_normal", C.c_longlong),
                ("n_ambiguous", C.c_longlong), ("n_sign_ambiguous", C.c_longlong), ("n_far", C.c_longlong),
                ("l_ref", C.c_double), ("tau_cut", C.c_double), ("d_band", C.c_double)]


def build(force: bool = False) -> str:
    """gcc -O2 (no fast-math) -> oracle/liboracle_dc.so; rebuilt when the source is newer."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= max(os.path.getmtime(_SRC), os.path.getmtime(_SRC_PAPER))):
        return _LIB
    tmp = _LIB + ".tmp%d" % os.getpid()
    subprocess.check_call(["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-o", tmp, _SRC, _SRC_PAPER, "-lm"])
    os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        dp = C.POINTER(C.c_double)
        L.orc_shape.argtypes = [C.c_double, dp, dp, dp]
        L.orc_patch_eval.argtypes = [dp, C.c_double, C.c_double, dp, dp, dp]
        L.orc_hex_eval.argtypes = [dp, C.c_double, C.c_double, C.c_double, dp]
        L.orc_lagrange_to_bezier.argtypes = [dp, dp]
        L.orc_bezier_eval.argtypes = [dp, C.c_double, C.c_double, dp]
        L.orc_bezier_split.argtypes = [dp, C.c_int, dp, dp]
        L.orc_box_dist.argtypes = [dp, dp]
        L.orc_box_dist.restype = C.c_double
        L.orc_tri_tri_dist.argtypes = [dp, dp, dp, dp]
        L.orc_tri_tri_dist.restype = C.c_double
        L.orc_patch_pair_flat.argtypes = [dp, dp, C.c_double, C.c_double, C.c_double, C.c_int, dp]
        L.orc_hex_face_nodes.argtypes = [C.c_int, C.POINTER(C.c_int)]
        L.orc_element_box.argtypes = [dp, C.POINTER(C.c_int), dp]
        L.orc_classify.argtypes = [C.c_longlong, dp, C.c_longlong, C.POINTER(C.c_int),
                                   C.c_longlong, dp, C.POINTER(OrcParams),
                                   C.c_longlong, C.c_longlong,
                                   C.POINTER(C.c_byte), dp, dp, dp, C.POINTER(C.c_int),
                                   C.POINTER(C.c_ubyte), C.POINTER(OrcStats)]
        L.orc_classify.restype = C.c_int
        _lib = L
    return _lib


def _dp(a: np.ndarray):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64))


# ----------------------------------------------------------------------------- primitives
def shape(t: float):
    l, d, dd = np.empty(3), np.empty(3), np.empty(3)
    lib().orc_shape(float(t), _dp(l), _dp(d), _dp(dd))
    return l, d, dd


def patch_eval(X, u, v):
    X = _f64(X).reshape(9, 3)
    P, Pu, Pv = np.empty(3), np.empty(3), np.empty(3)
    lib().orc_patch_eval(_dp(X), float(u), float(v), _dp(P), _dp(Pu), _dp(Pv))
    return P, Pu, Pv


def hex_eval(X, xi, eta, zeta):
    X = _f64(X).reshape(27, 3)
    P = np.empty(3)
    lib().orc_hex_eval(_dp(X), float(xi), float(eta), float(zeta), _dp(P))
    return P


def lagrange_to_bezier(X):
    X = _f64(X).reshape(9, 3)
    B = np.empty((9, 3))
    lib().orc_lagrange_to_bezier(_dp(X), _dp(B))
    return B


def bezier_eval(B, a, b):
    B = _f64(B).reshape(9, 3)
    P = np.empty(3)
    lib().orc_bezier_eval(_dp(B), float(a), float(b), _dp(P))
    return P


def bezier_split(B, direction):
    B = _f64(B).reshape(9, 3)
    lo, hi = np.empty((9, 3)), np.empty((9, 3))
    lib().orc_bezier_split(_dp(B), int(direction), _dp(lo), _dp(hi))
    return lo, hi


def box_dist(b1, b2) -> float:
    b1, b2 = _f64(b1).reshape(6), _f64(b2).reshape(6)
    return float(lib().orc_box_dist(_dp(b1), _dp(b2)))


def tri_tri_dist(A, B):
    A, B = _f64(A).reshape(3, 3), _f64(B).reshape(3, 3)
    wa, wb = np.empty(3), np.empty(3)
    d = float(lib().orc_tri_tri_dist(_dp(A), _dp(B), _dp(wa), _dp(wb)))
    return d, wa, wb


@dataclass
class PatchPairResult:
    hi: float
    params: np.ndarray   # (u, v, s, t)
    r: np.ndarray
    n: np.ndarray
    status: int          # 0 enclosure [hi-eps, hi]; 1 pruned (> cutoff); 2 early exit (hi <= tau_exit)
    depth_exceeded: int
    n_subpairs: int


def patch_pair(PX, QX, cutoff=np.inf, eps=1e-12, tau_exit=-1.0, max_depth=60) -> PatchPairResult:
    PX, QX = _f64(PX).reshape(9, 3), _f64(QX).reshape(9, 3)
    out = np.empty(14)
    lib().orc_patch_pair_flat(_dp(PX), _dp(QX), float(cutoff), float(eps), float(tau_exit),
                              int(max_depth), _dp(out))
    return PatchPairResult(out[0], out[1:5].copy(), out[5:8].copy(), out[8:11].copy(),
                           int(out[11]), int(out[12]), int(out[13]))


def hex_face_nodes(k: int) -> np.ndarray:
    ids = (C.c_int * 9)()
    lib().orc_hex_face_nodes(int(k), ids)
    return np.array(list(ids), dtype=np.int64)


def element_box(xyz, conn27_e) -> np.ndarray:
    xyz = _f64(xyz)
    c = np.ascontiguousarray(np.asarray(conn27_e, dtype=np.int32))
    out = np.empty(6)
    lib().orc_element_box(_dp(xyz), c.ctypes.data_as(C.POINTER(C.c_int)), _dp(out))
    return out


# ----------------------------------------------------------------------------- whole pass
@dataclass
class OracleResult:
    labels: np.ndarray      # int8 [n]   HOLE=0 NORMAL=1 CUT=2
    sdist: np.ndarray       # f64 [n]    0 for CUT, else +-min(d, d_band)
    dmin: np.ndarray        # f64 [n]    unclamped upper end of the enclosure of d_e
    width: np.ndarray       # f64 [n]    enclosure width used
    nearest: np.ndarray     # i32 [n]    nearest face id (PARITY UNPINNED: not unique)
    flags: np.ndarray       # u8 [n]
    stats: dict
    seconds: float
    nproc: int
    elem_ids: np.ndarray    # which elements (global ids)


def _params(tau_cut_rel=1e-7, d_band=0.0, l_ref=0.0, eps_rel=1e-12, eps_far_rel=1e-6,
            tie_rel=1e-9, max_depth=60) -> OrcParams:
    return OrcParams(tau_cut_rel, d_band, l_ref, eps_rel, eps_far_rel, tie_rel, max_depth, 0)


_G = {}


def _run_range(args):
    e0, e1, pkw = args
    xyz, conn, faces = _G["xyz"], _G["conn"], _G["faces"]
    n = e1 - e0
    labels = np.empty(n, np.int8); sdist = np.empty(n); dmin = np.empty(n); width = np.empty(n)
    nearest = np.empty(n, np.int32); flags = np.empty(n, np.uint8)
    st = OrcStats()
    prm = _params(**pkw)
    rc = lib().orc_classify(xyz.shape[0], _dp(xyz), conn.shape[0],
                            conn.ctypes.data_as(C.POINTER(C.c_int)), faces.shape[0], _dp(faces),
                            C.byref(prm), e0, e1,
                            labels.ctypes.data_as(C.POINTER(C.c_byte)), _dp(sdist), _dp(dmin), _dp(width),
                            nearest.ctypes.data_as(C.POINTER(C.c_int)),
                            flags.ctypes.data_as(C.POINTER(C.c_ubyte)), C.byref(st))
    if rc != 0:
        raise RuntimeError("orc_classify failed rc=%d" % rc)
    sd = {k: getattr(st, k) for k, _ in OrcStats._fields_}
    return labels, sdist, dmin, width, nearest, flags, sd


def classify(xyz, conn27, faces, *, e_begin: int = 0, e_end: Optional[int] = None,
             elem_ids: Optional[np.ndarray] = None, nproc: int = 1, **pkw) -> OracleResult:
    """Run the oracle on elements [e_begin, e_end) (or on the explicit `elem_ids`), every one
    against ALL faces.  nproc > 1 runs that many single-threaded processes over disjoint
    contiguous chunks (fork; results concatenated).

    NOTE: when d_band <= 0 (auto) every process recomputes it over the WHOLE grid, so pass
    an explicit d_band (e.g. from a first 1-element call's stats) for large grids.
    """
    lib()
    xyz = _f64(xyz).reshape(-1, 3)
    conn = np.ascontiguousarray(np.asarray(conn27, dtype=np.int32)).reshape(-1, 27)
    faces = _f64(faces).reshape(-1, 9, 3)
    n_elem = conn.shape[0]
    t0 = time.perf_counter()
    if elem_ids is not None:
        elem_ids = np.asarray(elem_ids, dtype=np.int64)
        # resolve auto d_band / l_ref once on the whole grid, then run on the gathered elements
        if not pkw.get("d_band", 0.0) > 0.0:
            pkw = dict(pkw, d_band=auto_d_band(xyz, conn, faces, **pkw))
        conn_sub = np.ascontiguousarray(conn[elem_ids])
        res = classify(xyz, conn_sub, faces, nproc=nproc, **pkw)
        res.elem_ids = elem_ids
        res.seconds = time.perf_counter() - t0
        return res
    if e_end is None:
        e_end = n_elem
    n = e_end - e_begin
    nproc = max(1, min(int(nproc), max(1, n // 8)))
    if nproc > 1 and not pkw.get("d_band", 0.0) > 0.0:
        pkw = dict(pkw, d_band=auto_d_band(xyz, conn, faces, **pkw))
    _G["xyz"], _G["conn"], _G["faces"] = xyz, conn, faces
    if nproc == 1:
        parts = [_run_range((e_begin, e_end, pkw))]
    else:
        nchunk = nproc * 8
        edges = np.linspace(e_begin, e_end, nchunk + 1).astype(np.int64)
        jobs = [(int(edges[i]), int(edges[i + 1]), pkw) for i in range(nchunk) if edges[i + 1] > edges[i]]
        ctx = mp.get_context("fork")
        with ctx.Pool(nproc) as pool:
            parts = pool.map(_run_range, jobs, chunksize=1)
    _G.clear()
    cat = lambda i: np.concatenate([p[i] for p in parts])  # noqa: E731
    stats = {}
    for p in parts:
        for k, v in p[6].items():
            if k in ("l_ref", "tau_cut", "d_band"):
                stats[k] = v
            else:
                stats[k] = stats.get(k, 0) + v
    return OracleResult(cat(0), cat(1), cat(2), cat(3), cat(4), cat(5), stats,
                        time.perf_counter() - t0, nproc, np.arange(e_begin, e_end, dtype=np.int64))


def auto_d_band(xyz, conn27, faces, **pkw) -> float:
    """The oracle's own auto d_band (max element Bezier-box diagonal): a zero-element call."""
    xyz = _f64(xyz).reshape(-1, 3)
    conn = np.ascontiguousarray(np.asarray(conn27, dtype=np.int32)).reshape(-1, 27)
    faces = _f64(faces).reshape(-1, 9, 3)
    st = OrcStats()
    kw = {k: v for k, v in pkw.items() if k != "d_band"}
    prm = _params(**kw)
    lab = np.empty(1, np.int8); sd = np.empty(1)
    rc = lib().orc_classify(xyz.shape[0], _dp(xyz), conn.shape[0],
                            conn.ctypes.data_as(C.POINTER(C.c_int)), faces.shape[0], _dp(faces),
                            C.byref(prm), 0, 0, lab.ctypes.data_as(C.POINTER(C.c_byte)), _dp(sd),
                            None, None, None, None, C.byref(st))
    if rc != 0:
        raise RuntimeError("orc_classify failed rc=%d" % rc)
    return float(st.d_band)
