"""ctypes binding of libdc.so: same names as include/dc.h, argument marshalling only.

Every step of the hot path runs in the library's CUDA kernels.  Tensors are passed as raw
device pointers (`tensor.data_ptr()`), streams as `torch.cuda.current_stream().cuda_stream`.
There is NO CPU fallback: if libdc.so is missing this module raises on import; if the device
is not sm_100 `dc_create_grid` returns DC_ERR_UNSUPPORTED and `DirectCut` raises.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

from ._build import LIB

DC_HOLE, DC_NORMAL, DC_CUT = 0, 1, 2
DC_OK, DC_ERR_ARG, DC_ERR_WORKSPACE, DC_ERR_UNSUPPORTED, DC_ERR_CUDA, DC_ERR_STATE, DC_ERR_RESULT = 0, -1, -2, -3, -4, -5, -6
DC_STATUS_PAIR_OVERFLOW, DC_STATUS_QUEUE_OVERFLOW, DC_STATUS_FILL_CONFLICT, DC_STATUS_SEEDLESS_OVERFLOW = 1, 2, 4, 8
DC_STATUS_BAND_OVERFLOW, DC_STATUS_SURFACE_SMALL = 16, 32
DC_FLAG_RECOMPUTE_BOXES = 1
DC_FLAG_PAPER_MODE = 2
DC_FLAG_EXACT_FAR = 4
DC_FLAG_GRAPH = 8
DC_MODE_WALL, DC_MODE_OVERSET = 0, 1
DC_NOALLOC_MAX_POINTS = 65536

EXPORTS = ["dc_workspace_bytes", "dc_create_grid", "dc_set_cut_surface", "dc_classify", "dc_cut",
           "dc_classify_host", "dc_get_element_boxes", "dc_get_adjacency", "dc_get_pairs",
           "dc_get_stats", "dc_destroy", "dc_error_string", "dc_measure_fp64_tflops", "dc_version",
           "dc_union_labels", "dc_unblank", "dc_ab_faces",
           "dc_adt_bytes", "dc_donor_scratch_bytes", "dc_adt_build", "dc_find_donors", "dc_find_donors_noalloc"]


class dc_params(C.Structure):
    _fields_ = [("tau_cut_rel", C.c_double), ("d_band", C.c_double), ("l_ref", C.c_double),
                ("theta_leaf", C.c_double), ("max_level", C.c_int), ("flags", C.c_int)]


class dc_stats(C.Structure):
    _fields_ = [("n_elem", C.c_longlong), ("n_face", C.c_longlong), ("n_active", C.c_longlong),
                ("n_box_tests", C.c_longlong), ("n_pairs", C.c_longlong), ("n_bnb_nodes", C.c_longlong),
                ("n_newton", C.c_longlong), ("n_newton_iters", C.c_longlong), ("n_newton_fail", C.c_longlong),
                ("n_depth_exceeded", C.c_longlong), ("n_cut", C.c_longlong), ("n_hole", C.c_longlong),
                ("n_normal", C.c_longlong), ("n_ambiguous", C.c_longlong), ("n_sign_ambiguous", C.c_longlong),
                ("n_seedless_components", C.c_longlong), ("n_fill_conflicts", C.c_longlong),
                ("pairs_needed", C.c_longlong), ("queue_peak", C.c_longlong),
                ("n_root_nodes", C.c_longlong), ("band_needed", C.c_longlong), ("queue_needed", C.c_longlong),
                ("n_far", C.c_longlong), ("n_far_done", C.c_longlong), ("n_far_unresolved", C.c_longlong),
                ("far_pairs", C.c_longlong), ("far_passes", C.c_longlong),
                ("l_ref", C.c_double), ("tau_cut", C.c_double), ("d_band", C.c_double),
                ("ms_stage", C.c_float * 8), ("ms_kernel", C.c_float * 8), ("status", C.c_int), ("n_launches", C.c_int),
                ("ms_far", C.c_float), ("reserved", C.c_int)]

    def as_dict(self) -> dict:
        d = {}
        for k, _ in self._fields_:
            v = getattr(self, k)
            d[k] = list(v) if k in ("ms_stage", "ms_kernel") else v
        return d


if not os.path.exists(LIB):
    raise ImportError("libdc.so is not built (%s): run `python -c 'import __graft_entry__ as g; g.build()'`; "
                      "there is no CPU fallback" % LIB)

_lib = C.CDLL(LIB)
_vp = C.c_void_p
_lib.dc_workspace_bytes.argtypes = [C.c_longlong] * 4
_lib.dc_workspace_bytes.restype = C.c_size_t
_lib.dc_create_grid.argtypes = [C.POINTER(_vp), C.c_int, C.c_longlong, _vp, C.c_longlong, _vp, _vp,
                                _vp, C.c_size_t, C.c_longlong, C.c_longlong, _vp]
_lib.dc_set_cut_surface.argtypes = [_vp, C.c_longlong, _vp, _vp]
_lib.dc_classify.argtypes = [_vp, C.POINTER(dc_params), _vp, _vp, _vp]
_lib.dc_cut.argtypes = [_vp, C.POINTER(dc_params), C.c_longlong, _vp, _vp, _vp, _vp]
_lib.dc_classify_host.argtypes = [_vp, C.POINTER(dc_params), C.c_longlong, _vp, _vp, _vp, _vp]
_lib.dc_get_element_boxes.argtypes = [_vp, _vp, _vp]
_lib.dc_get_adjacency.argtypes = [_vp, _vp, _vp]
_lib.dc_get_pairs.argtypes = [_vp, _vp, _vp, C.c_longlong]
_lib.dc_get_pairs.restype = C.c_longlong
_lib.dc_get_stats.argtypes = [_vp, C.POINTER(dc_stats)]
_lib.dc_destroy.argtypes = [_vp]
_lib.dc_destroy.restype = None
_lib.dc_error_string.argtypes = [C.c_int]
_lib.dc_error_string.restype = C.c_char_p
_lib.dc_measure_fp64_tflops.argtypes = [C.c_int, C.c_int]
_lib.dc_measure_fp64_tflops.restype = C.c_double
_lib.dc_version.restype = C.c_int
_lib.dc_union_labels.argtypes = [C.c_longlong, _vp, _vp, _vp, _vp]
_lib.dc_unblank.argtypes = [C.c_int, C.c_int, C.c_longlong, _vp, _vp, _vp, _vp, _vp, _vp, C.c_longlong, _vp, _vp]
_lib.dc_ab_faces.argtypes = [C.c_longlong, _vp, _vp, _vp, _vp, _vp]
_lib.dc_adt_bytes.argtypes = [C.c_longlong]
_lib.dc_adt_bytes.restype = C.c_size_t
_lib.dc_donor_scratch_bytes.argtypes = [C.c_longlong]
_lib.dc_donor_scratch_bytes.restype = C.c_size_t
_lib.dc_adt_build.argtypes = [_vp, _vp, C.c_size_t, _vp]
_lib.dc_find_donors.argtypes = [_vp, C.c_longlong, _vp, C.POINTER(C.c_double), C.POINTER(C.c_double), _vp, _vp, _vp, C.c_size_t, _vp]
_lib.dc_find_donors_noalloc.argtypes = [_vp, C.c_longlong, _vp, C.POINTER(C.c_double), C.POINTER(C.c_double), _vp, _vp, _vp]


class DcError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        super().__init__("%s: %s (%d)" % (where, _lib.dc_error_string(code).decode(), code))


def _ck(code: int, where: str):
    if code != DC_OK:
        raise DcError(code, where)


# ---- 1:1 wrappers (names of include/dc.h) ------------------------------------------------------
def dc_workspace_bytes(n_nodes, n_elem, max_faces, max_pairs) -> int:
    return int(_lib.dc_workspace_bytes(n_nodes, n_elem, max_faces, max_pairs))


def dc_create_grid(device, n_nodes, xyz_ptr, n_elem, conn_ptr, adj_ptr, ws_ptr, ws_bytes, max_faces, max_pairs, stream):
    ctx = _vp()
    _ck(_lib.dc_create_grid(C.byref(ctx), device, n_nodes, xyz_ptr, n_elem, conn_ptr, adj_ptr or None,
                            ws_ptr, ws_bytes, max_faces, max_pairs, stream or None), "dc_create_grid")
    return ctx


def dc_set_cut_surface(ctx, n_face, faces_ptr, stream):
    _ck(_lib.dc_set_cut_surface(ctx, n_face, faces_ptr, stream or None), "dc_set_cut_surface")


def dc_classify(ctx, params: Optional[dc_params], labels_ptr, sdist_ptr, stream):
    _ck(_lib.dc_classify(ctx, C.byref(params) if params is not None else None, labels_ptr, sdist_ptr,
                         stream or None), "dc_classify")


def dc_cut(ctx, params: Optional[dc_params], n_face, faces_ptr, labels_ptr, sdist_ptr, stream):
    _ck(_lib.dc_cut(ctx, C.byref(params) if params is not None else None, n_face, faces_ptr, labels_ptr, sdist_ptr,
                    stream or None), "dc_cut")


def dc_classify_host(ctx, params: Optional[dc_params], n_face, faces_host_ptr, labels_host_ptr, sdist_host_ptr, stream):
    _ck(_lib.dc_classify_host(ctx, C.byref(params) if params is not None else None, n_face, faces_host_ptr,
                              labels_host_ptr, sdist_host_ptr, stream or None), "dc_classify_host")


def dc_get_stats(ctx, allow_status: bool = False, return_code: bool = False):
    st = dc_stats()
    rc = _lib.dc_get_stats(ctx, C.byref(st))
    if rc != DC_OK and not (allow_status and rc in (DC_ERR_WORKSPACE, DC_ERR_RESULT, DC_ERR_UNSUPPORTED)):
        raise DcError(rc, "dc_get_stats (status=%d, pairs_needed=%d)" % (st.status, st.pairs_needed))
    return (st, rc) if return_code else st


def dc_destroy(ctx):
    _lib.dc_destroy(ctx)


def dc_measure_fp64_tflops(device: int = 0, iters: int = 2000) -> float:
    v = float(_lib.dc_measure_fp64_tflops(device, iters))
    if v < 0:
        raise DcError(DC_ERR_CUDA, "dc_measure_fp64_tflops")
    return v


def dc_version() -> int:
    return int(_lib.dc_version())


# ---- blanking logic on torch CUDA tensors (argument marshalling only; include/dc.h documents the calls) ----------
def _stream(t):
    import torch
    return C.c_void_p(torch.cuda.current_stream(t.device).cuda_stream)


def dc_union_labels(a, b, out=None):
    import torch
    out = torch.empty_like(a) if out is None else out
    rc = _lib.dc_union_labels(a.numel(), a.data_ptr(), b.data_ptr(), out.data_ptr(), _stream(a))
    if rc:
        raise DcError(rc, "dc_union_labels")
    return out


def dc_unblank(mode: int, cut_is_hole: bool, iblank_prev, labels_t, labels_tplus, list_cap: Optional[int] = None,
               want_tohole: bool = True):
    """Returns (iblank_new int8 tensor, must_unblank ids, to_hole ids) -- the id lists in no particular order."""
    import torch
    n = iblank_prev.numel()
    cap = n if list_cap is None else int(list_cap)
    out = torch.empty(n, dtype=torch.int8, device=iblank_prev.device)
    unb = torch.empty(max(cap, 1), dtype=torch.int32, device=iblank_prev.device)
    toh = torch.empty(max(cap, 1), dtype=torch.int32, device=iblank_prev.device) if want_tohole else None
    counts = torch.zeros(2, dtype=torch.int64, device=iblank_prev.device)
    rc = _lib.dc_unblank(int(mode), int(bool(cut_is_hole)), n, iblank_prev.data_ptr(), labels_t.data_ptr(),
                         labels_tplus.data_ptr(), out.data_ptr(), unb.data_ptr(),
                         toh.data_ptr() if toh is not None else None, cap, counts.data_ptr(), _stream(iblank_prev))
    if rc:
        raise DcError(rc, "dc_unblank")
    c = counts.cpu().tolist()
    return out, unb[:min(c[0], cap)], (toh[:min(c[1], cap)] if toh is not None else None), c


def dc_ab_faces(iblank, adj6):
    import torch
    n = iblank.numel()
    mask = torch.empty(n, dtype=torch.uint8, device=iblank.device)
    count = torch.zeros(1, dtype=torch.int64, device=iblank.device)
    rc = _lib.dc_ab_faces(n, iblank.data_ptr(), adj6.data_ptr(), mask.data_ptr(), count.data_ptr(), _stream(iblank))
    if rc:
        raise DcError(rc, "dc_ab_faces")
    return mask, int(count.item())


# ---- convenience owner of the torch buffers ----------------------------------------------------
class DirectCut:
    """Owns the caller-side torch buffers (grid arrays, workspace, outputs) around one dc_ctx.

    torch is imported lazily: it provides device memory and the stream, nothing else.
    """

    def __init__(self, xyz, conn27, adj6=None, *, max_faces: int, max_pairs: Optional[int] = None, device: int = 0):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1711_07663_b200 needs a CUDA device (sm_100); there is no CPU fallback")
        self.torch = torch
        self.device = device
        dev = torch.device("cuda", device)
        self.xyz = torch.as_tensor(xyz, dtype=torch.float64).contiguous().to(dev)
        self.conn = torch.as_tensor(conn27, dtype=torch.int32).contiguous().to(dev)
        self.adj = None if adj6 is None else torch.as_tensor(adj6, dtype=torch.int32).contiguous().to(dev)
        self.n_nodes, self.n_elem = int(self.xyz.shape[0]), int(self.conn.shape[0])
        self.max_faces = int(max_faces)
        self.max_pairs = int(max_pairs) if max_pairs else max(1 << 20, 8 * self.n_elem)
        self.ws_bytes = dc_workspace_bytes(self.n_nodes, self.n_elem, self.max_faces, self.max_pairs)
        if self.ws_bytes == 0:
            raise DcError(DC_ERR_ARG, "dc_workspace_bytes")
        self.ws = torch.empty(self.ws_bytes + 256, dtype=torch.uint8, device=dev)
        off = (-self.ws.data_ptr()) % 256
        self.ws_ptr = self.ws.data_ptr() + off
        self.labels = torch.empty(self.n_elem, dtype=torch.int8, device=dev)
        self.sdist = torch.empty(self.n_elem, dtype=torch.float64, device=dev)
        self.faces = None
        with torch.cuda.device(dev):
            self.ctx = dc_create_grid(device, self.n_nodes, self.xyz.data_ptr(), self.n_elem, self.conn.data_ptr(),
                                      self.adj.data_ptr() if self.adj is not None else None,
                                      self.ws_ptr, self.ws_bytes, self.max_faces, self.max_pairs, self._stream())

    def _stream(self):
        return self.torch.cuda.current_stream(self.device).cuda_stream

    def set_cut_surface(self, faces):
        t = self.torch
        if not (isinstance(faces, t.Tensor) and faces.is_cuda):
            faces = t.as_tensor(faces, dtype=t.float64).contiguous().to(self.xyz.device)
        self.faces = faces.contiguous()
        dc_set_cut_surface(self.ctx, int(self.faces.shape[0]), self.faces.data_ptr(), self._stream())

    def classify(self, params: Optional[dc_params] = None):
        dc_classify(self.ctx, params, self.labels.data_ptr(), self.sdist.data_ptr(), self._stream())
        return self.labels, self.sdist

    def cut(self, faces, params: Optional[dc_params] = None):
        """dc_cut: set_cut_surface + classify in one call; with DC_FLAG_GRAPH in params.flags the launch sequence is
        replayed from a CUDA graph (needs a current stream other than the legacy default stream)."""
        t = self.torch
        if not (isinstance(faces, t.Tensor) and faces.is_cuda):
            faces = t.as_tensor(faces, dtype=t.float64).contiguous().to(self.xyz.device)
        self.faces = faces.contiguous()
        dc_cut(self.ctx, params, int(self.faces.shape[0]), self.faces.data_ptr(), self.labels.data_ptr(),
               self.sdist.data_ptr(), self._stream())
        return self.labels, self.sdist

    def classify_host(self, faces_host, labels_host, sdist_host, params: Optional[dc_params] = None):
        """faces_host / labels_host / sdist_host: pinned CPU torch tensors (f64 [n,9,3], int8 [n_elem], f64 [n_elem])."""
        dc_classify_host(self.ctx, params, int(faces_host.shape[0]), faces_host.data_ptr(),
                         labels_host.data_ptr(), sdist_host.data_ptr(), self._stream())

    def stats(self, allow_status: bool = False, return_code: bool = False):
        return dc_get_stats(self.ctx, allow_status, return_code)

    def element_boxes(self):
        out = self.torch.empty((self.n_elem, 6), dtype=self.torch.float64, device=self.xyz.device)
        _ck(_lib.dc_get_element_boxes(self.ctx, out.data_ptr(), self._stream()), "dc_get_element_boxes")
        return out

    def adjacency(self):
        out = self.torch.empty((self.n_elem, 6), dtype=self.torch.int32, device=self.xyz.device)
        _ck(_lib.dc_get_adjacency(self.ctx, out.data_ptr(), self._stream()), "dc_get_adjacency")
        return out

    def pairs(self):
        import numpy as np
        st = self.stats(allow_status=True)
        cap = max(1, int(st.n_pairs))
        e = np.empty(cap, np.int32); f = np.empty(cap, np.int32)
        n = _lib.dc_get_pairs(self.ctx, e.ctypes.data, f.ctypes.data, cap)
        if n < 0:
            raise DcError(int(n), "dc_get_pairs")
        return e[:n], f[:n]

    def build_adt(self):
        """dc_adt_build: the donor-search tree over the element boxes (host build, once)."""
        t = self.torch
        nbytes = int(_lib.dc_adt_bytes(self.n_elem))
        self.adt = t.empty(nbytes + 16, dtype=t.uint8, device=self.xyz.device)
        off = (-self.adt.data_ptr()) % 16
        _ck(_lib.dc_adt_build(self.ctx, self.adt.data_ptr() + off, nbytes, self._stream()), "dc_adt_build")

    def find_donors(self, pts, rot=None, offset=None):
        """dc_find_donors: pts [n][3] (torch CUDA f64 or numpy) -> (donor int32 [n], ref f64 [n][3]) on the device."""
        t = self.torch
        if not (isinstance(pts, t.Tensor) and pts.is_cuda):
            pts = t.as_tensor(pts, dtype=t.float64).contiguous().to(self.xyz.device)
        pts = pts.contiguous()
        n = int(pts.shape[0])
        donor = t.empty(n, dtype=t.int32, device=pts.device)
        ref = t.empty((n, 3), dtype=t.float64, device=pts.device)
        sb = int(_lib.dc_donor_scratch_bytes(n))
        scratch = t.empty(max(sb, 4), dtype=t.uint8, device=pts.device)
        R = (C.c_double * 9)(*[float(x) for x in rot.reshape(-1)]) if rot is not None else None
        o = (C.c_double * 3)(*[float(x) for x in offset]) if offset is not None else None
        _ck(_lib.dc_find_donors(self.ctx, n, pts.data_ptr(), R, o, donor.data_ptr(), ref.data_ptr(), scratch.data_ptr(), sb,
                                self._stream()), "dc_find_donors")
        return donor, ref

    def find_donors_noalloc(self, pts, donor, ref, rot=None, offset=None, return_code: bool = False):
        """dc_find_donors_noalloc: pts [n][3] CUDA f64, donor int32 [n] and ref f64 [n][3] CUDA tensors of the caller's;
        the library's built-in scratch (n <= DC_NOALLOC_MAX_POINTS), nothing allocated here or there."""
        R = (C.c_double * 9)(*[float(x) for x in rot.reshape(-1)]) if rot is not None else None
        o = (C.c_double * 3)(*[float(x) for x in offset]) if offset is not None else None
        rc = _lib.dc_find_donors_noalloc(self.ctx, int(pts.shape[0]), pts.data_ptr(), R, o, donor.data_ptr(), ref.data_ptr(),
                                         self._stream())
        if return_code:
            return rc
        _ck(rc, "dc_find_donors_noalloc")

    def close(self):
        if getattr(self, "ctx", None):
            dc_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
