"""ctypes front end of oracle/paper_oracle.c: the CPU oracle of the paper's own approximate direct cut
(Algorithms A.1-A.4, N_F^1 = 16, N_F^2 = 4).  TEST INFRASTRUCTURE ONLY, like dc_oracle.py.
"""
from __future__ import annotations

import ctypes as C
import multiprocessing as mp
from dataclasses import dataclass
from typing import Optional

import numpy as np

from . import dc_oracle as O

FLAG_FAR = 4


class PmStats(C.Structure):
    _fields_ = [("n_a1", C.c_longlong), ("n_tritri", C.c_longlong), ("n_cut", C.c_longlong), ("n_hole", C.c_longlong),
                ("n_normal", C.c_longlong), ("n_far", C.c_longlong), ("l_ref", C.c_double), ("tol", C.c_double),
                ("d_band", C.c_double)]


_set = False


def lib():
    global _set
    L = O.lib()
    if not _set:
        dp = C.POINTER(C.c_double)
        L.orc_pm_eig3.argtypes = [dp, dp]
        L.orc_pm_obb.argtypes = [dp, dp, dp, dp]
        L.orc_pm_a1.argtypes = [dp, dp, dp, dp]
        L.orc_pm_a1.restype = C.c_double
        L.orc_paper_classify.argtypes = [C.c_longlong, dp, C.c_longlong, C.POINTER(C.c_int), C.c_longlong, dp,
                                         C.c_double, C.c_double, C.c_longlong, C.c_longlong,
                                         C.POINTER(C.c_byte), dp, C.POINTER(C.c_int), C.POINTER(C.c_ubyte), C.POINTER(PmStats)]
        L.orc_paper_classify.restype = C.c_int
        _set = True
    return L


def eig3(A) -> np.ndarray:
    A = O._f64(A).reshape(9)
    R = np.empty(9)
    lib().orc_pm_eig3(O._dp(A), O._dp(R))
    return R.reshape(3, 3)          # rows = axes


def obb(X8):
    X8 = O._f64(X8).reshape(8, 3)
    R, ext, ecg = np.empty(9), np.empty(6), np.empty(3)
    lib().orc_pm_obb(O._dp(X8), O._dp(R), O._dp(ext), O._dp(ecg))
    return R.reshape(3, 3), ext, ecg


def a1(R, ext, ecg, F4) -> float:
    R, ext, ecg, F4 = O._f64(R).reshape(9), O._f64(ext), O._f64(ecg), O._f64(F4).reshape(12)
    return float(lib().orc_pm_a1(O._dp(R), O._dp(ext), O._dp(ecg), O._dp(F4)))


@dataclass
class PaperResult:
    labels: np.ndarray      # int8: HOLE 0 / NORMAL 1 / CUT 2, -1 = no candidate face (not computed)
    sdist: np.ndarray
    nearest: np.ndarray
    flags: np.ndarray
    stats: dict
    elem_ids: Optional[np.ndarray] = None


_G = {}


def _run(args):
    e0, e1, d_band, l_ref = args
    xyz, conn, faces = _G["xyz"], _G["conn"], _G["faces"]
    n = e1 - e0
    labels = np.empty(n, np.int8); sdist = np.empty(n); nearest = np.empty(n, np.int32); flags = np.empty(n, np.uint8)
    st = PmStats()
    rc = lib().orc_paper_classify(xyz.shape[0], O._dp(xyz), conn.shape[0], conn.ctypes.data_as(C.POINTER(C.c_int)),
                                  faces.shape[0], O._dp(faces), float(d_band), float(l_ref), e0, e1,
                                  labels.ctypes.data_as(C.POINTER(C.c_byte)), O._dp(sdist),
                                  nearest.ctypes.data_as(C.POINTER(C.c_int)), flags.ctypes.data_as(C.POINTER(C.c_ubyte)),
                                  C.byref(st))
    if rc != 0:
        raise RuntimeError("orc_paper_classify failed rc=%d" % rc)
    return labels, sdist, nearest, flags, {k: getattr(st, k) for k, _ in PmStats._fields_}


def classify(xyz, conn27, faces, *, d_band: float, l_ref: float, elem_ids=None, nproc: int = 1) -> PaperResult:
    """The paper's approximate cut of the given elements (all by default), every one against all faces."""
    lib()
    xyz = O._f64(xyz).reshape(-1, 3)
    conn = np.ascontiguousarray(np.asarray(conn27, dtype=np.int32)).reshape(-1, 27)
    faces = O._f64(faces).reshape(-1, 9, 3)
    if elem_ids is not None:
        elem_ids = np.asarray(elem_ids, dtype=np.int64)
        conn = np.ascontiguousarray(conn[elem_ids])
    n = conn.shape[0]
    _G["xyz"], _G["conn"], _G["faces"] = xyz, conn, faces
    nproc = max(1, min(int(nproc), max(1, n // 8)))
    if nproc == 1:
        parts = [_run((0, n, d_band, l_ref))]
    else:
        edges = np.linspace(0, n, nproc * 8 + 1).astype(np.int64)
        jobs = [(int(edges[i]), int(edges[i + 1]), d_band, l_ref) for i in range(nproc * 8) if edges[i + 1] > edges[i]]
        with mp.get_context("fork").Pool(nproc) as pool:
            parts = pool.map(_run, jobs)
    stats = {}
    for p in parts:
        for k, v in p[4].items():
            stats[k] = v if k in ("l_ref", "tol", "d_band") else stats.get(k, 0) + v
    return PaperResult(np.concatenate([p[0] for p in parts]), np.concatenate([p[1] for p in parts]),
                       np.concatenate([p[2] for p in parts]), np.concatenate([p[3] for p in parts]), stats, elem_ids)
