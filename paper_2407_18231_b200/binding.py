"""Thin ctypes binding of include/lst.h (argument marshalling only; all compute runs in the CUDA
kernels of csrc/).  There is NO CPU fallback: a missing library or a missing GPU raises.

Function names mirror the C ABI: lst_load_geometry, lst_run_event, lst_free, lst_ctx_*.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liblst_b200.so")

LST_OK, LST_ERR_ARG, LST_ERR_CUDA, LST_ERR_CAPACITY, LST_ERR_GEOMETRY, LST_ERR_LIMIT = 0, -1, -2, -3, -4, -5
LST_SCAN_STATIC_MAX_N = 1 << 24  # include/lst.h
N_STAGES = 7
STAGES = ("md", "ls", "t3", "t5", "pt3", "pt5", "t4")
_EXT_FIELDS = ("t4_tol0", "t4_tol1", "t5_mlp_scale", "t5_mlp_thr")

_FLOAT_FIELDS = (
    "b_field", "pt_min", "z0_max", "md_b_phi_tol", "md_z_tol", "md_e_slope", "md_e_tol",
    "ls_kappa_max", "ls_z_tol", "ls_dir_tol", "t3_kappa_max", "t3_z_tol0", "t3_z_tol1",
    "t5_tol0", "t5_tol1", "pt_gate_tol", "pt_k_tol0", "pt_k_tol1", "pt_z_tol", "near_rel",
)
_fp = C.POINTER(C.c_float)
_ip = C.POINTER(C.c_int32)


class LstError(RuntimeError):
    def __init__(self, status, where=""):
        self.status = int(status)
        msg = _lib().lst_strerror(int(status)).decode() if _LIB is not None else str(status)
        super().__init__(f"{where}: {msg} (status {status})")


class lst_module(C.Structure):
    _fields_ = [("subdet", C.c_int32), ("layer", C.c_int32), ("side", C.c_int32), ("ring", C.c_int32)]


class lst_params(C.Structure):
    _fields_ = [(f, C.c_float) for f in _FLOAT_FIELDS] + [("stage_mask", C.c_int32)] + \
               [(f, C.c_float) for f in _EXT_FIELDS] + [("t5_mlp", C.c_float * 65)]

    def as_dict(self):
        d = {f: float(np.float32(getattr(self, f))) for f in _FLOAT_FIELDS + _EXT_FIELDS}
        d["stage_mask"] = int(self.stage_mask)
        return d


class lst_caps(C.Structure):
    _fields_ = [(f, C.c_int32) for f in ("max_events", "max_hits", "max_pls", "max_md", "max_ls", "max_t3",
                                          "max_t5", "max_pt3", "max_pt5", "max_tc", "max_t4")]


class lst_hits(C.Structure):
    _fields_ = [("x", C.c_void_p), ("y", C.c_void_p), ("z", C.c_void_p), ("sensor", C.c_void_p),
                ("n", C.c_int32), ("event_offsets", C.c_void_p), ("on_device", C.c_int32), ("sensor_u16", C.c_int32)]


class lst_pls(C.Structure):
    _fields_ = [("pt", C.c_void_p), ("q", C.c_void_p), ("x0", C.c_void_p), ("y0", C.c_void_p), ("z0", C.c_void_p),
                ("x1", C.c_void_p), ("y1", C.c_void_p), ("z1", C.c_void_p), ("n", C.c_int32),
                ("event_offsets", C.c_void_p), ("on_device", C.c_int32)]


class lst_event_out(C.Structure):
    _fields_ = [("magic", C.c_uint64)] + \
        [(f, C.c_int32) for f in ("n_md", "n_ls", "n_t3", "n_t5", "n_pt3", "n_pt5", "n_tc")] + \
        [("near", C.c_int64 * N_STAGES), ("n_tests", C.c_int64 * N_STAGES),
         ("md_hits", _ip), ("md_module", _ip), ("md_f", _fp), ("ls_md", _ip), ("ls_kappa", _fp),
         ("t3_ls", _ip), ("t3_md", _ip), ("t3_k", _fp), ("t5_t3", _ip), ("t5_md", _ip), ("t5_score", _fp),
         ("pt3", _ip), ("pt3_score", _fp), ("pt5", _ip), ("pt5_score", _fp), ("tc", _ip),
         ("n_t4", C.c_int32), ("t4_t3", _ip), ("t4_md", _ip), ("t4_score", _fp)]


class lst_batch_summary(C.Structure):
    _fields_ = [(f, C.c_int32) for f in ("n_events", "n_hits", "n_pls", "n_md", "n_ls", "n_t3", "n_t5", "n_pt3",
                                          "n_pt5", "n_tc", "n_t4")] + \
        [("near", C.c_int64 * N_STAGES), ("n_tests", C.c_int64 * N_STAGES)]

    def as_dict(self):
        d = {f: int(getattr(self, f)) for f, _ in self._fields_[:11]}
        d["near"] = [int(v) for v in self.near]
        d["n_tests"] = [int(v) for v in self.n_tests]
        return d


class lst_audit_report(C.Structure):
    _fields_ = [(f, C.c_int64 * 4) for f in ("candidates", "accepted", "near", "chain_candidates", "chain_objects",
                                              "chain_near")] + \
        [("hash_exact", C.c_uint64 * 4), ("hash_chain", C.c_uint64 * 4), ("mismatches", C.c_int64)]

    def as_dict(self):
        d = {f: [int(v) for v in getattr(self, f)] for f, _ in self._fields_[:8]}
        d["mismatches"] = int(self.mismatches)
        return d


# every symbol include/lst.h declares (tests check the library exports all of them)
ABI_SYMBOLS = (
    "lst_strerror", "lst_default_params", "lst_default_caps", "lst_workspace_bytes", "lst_load_geometry",
    "lst_run_event", "lst_free", "lst_ctx_create", "lst_ctx_run", "lst_ctx_sync", "lst_ctx_fetch_event",
    "lst_ctx_fetch_tc", "lst_ctx_set_blocks_per_sm", "lst_ctx_set_graph", "lst_ctx_set_timing", "lst_ctx_kernel_times", "lst_ctx_launch_count", "lst_ctx_stat",
    "lst_scan_counts", "lst_scan_counts_static", "lst_ctx_audit",
)

_LIB = None


def library_path() -> str:
    return _SO


def _lib():
    """Loads the CUDA library; raises if it has not been built (no fallback of any kind)."""
    global _LIB
    if _LIB is not None:
        return _LIB
    if not os.path.exists(_SO):
        raise RuntimeError(f"{_SO} is missing: build it with `python -m paper_2407_18231_b200.build` "
                           "(__graft_entry__.build()); there is no CPU fallback")
    L = C.CDLL(_SO)
    vp = C.c_void_p
    L.lst_strerror.restype = C.c_char_p
    L.lst_strerror.argtypes = [C.c_int]
    L.lst_default_params.argtypes = [C.POINTER(lst_params)]
    L.lst_default_params.restype = None
    L.lst_default_caps.argtypes = [C.POINTER(lst_caps)]
    L.lst_default_caps.restype = None
    L.lst_workspace_bytes.argtypes = [C.POINTER(lst_caps), C.c_int32]
    L.lst_workspace_bytes.restype = C.c_size_t
    L.lst_load_geometry.argtypes = [C.POINTER(lst_module), C.c_int32, _ip, _ip, C.POINTER(lst_params), C.POINTER(vp)]
    L.lst_run_event.argtypes = [vp, C.POINTER(lst_hits), C.POINTER(lst_pls), C.POINTER(C.POINTER(lst_event_out))]
    L.lst_free.argtypes = [vp]
    L.lst_free.restype = None
    L.lst_ctx_create.argtypes = [vp, C.POINTER(lst_caps), vp, C.POINTER(vp)]
    L.lst_ctx_run.argtypes = [vp, C.c_int32, C.POINTER(lst_hits), C.POINTER(lst_pls)]
    L.lst_ctx_sync.argtypes = [vp, C.POINTER(lst_batch_summary)]
    L.lst_ctx_fetch_event.argtypes = [vp, C.c_int32, C.POINTER(C.POINTER(lst_event_out))]
    L.lst_ctx_fetch_tc.argtypes = [vp, _ip, C.c_int32, _ip]
    L.lst_ctx_set_timing.argtypes = [vp, C.c_int32]
    L.lst_ctx_set_blocks_per_sm.argtypes = [vp, C.c_int32]
    L.lst_ctx_set_graph.argtypes = [vp, C.c_int32]
    L.lst_ctx_kernel_times.argtypes = [vp, _fp, C.POINTER(C.c_char_p), C.c_int32]
    L.lst_ctx_launch_count.argtypes = [vp]
    L.lst_ctx_stat.argtypes = [vp, C.c_int32]
    L.lst_ctx_stat.restype = C.c_int64
    L.lst_scan_counts.argtypes = [vp, C.c_int32, vp, vp]
    L.lst_ctx_audit.argtypes = [vp, C.POINTER(lst_audit_report)]
    L.lst_scan_counts_static.argtypes = [vp, C.c_int32, vp, vp]
    _LIB = L
    return L


def _check(status, where):
    if status != LST_OK:
        raise LstError(status, where)


def lst_default_params(**overrides) -> lst_params:
    p = lst_params()
    _lib().lst_default_params(C.byref(p))
    for k, v in overrides.items():
        if not hasattr(p, k):
            raise KeyError(k)
        if k == "t5_mlp":
            w = np.asarray(v, dtype=np.float32).ravel()
            if w.shape[0] != 65:
                raise ValueError("t5_mlp holds 65 weights (CUTS.md section 11)")
            for i in range(65):
                p.t5_mlp[i] = float(w[i])
        else:
            setattr(p, k, v)
    return p


def lst_default_caps(**overrides) -> lst_caps:
    c = lst_caps()
    _lib().lst_default_caps(C.byref(c))
    for k, v in overrides.items():
        if not hasattr(c, k):
            raise KeyError(k)
        setattr(c, k, int(v))
    return c


def lst_workspace_bytes(caps: lst_caps | None, n_modules: int) -> int:
    return int(_lib().lst_workspace_bytes(C.byref(caps) if caps is not None else None, int(n_modules)))


def lst_free(handle) -> None:
    if handle:
        _lib().lst_free(handle)


def lst_load_geometry(module_table, conn_offsets, conn_targets, params: lst_params | None = None):
    """module_table: int32 [n_modules, 4] (subdet, layer, side, ring).  Returns an opaque handle."""
    mt = np.ascontiguousarray(np.asarray(module_table, dtype=np.int32).reshape(-1, 4))
    off = np.ascontiguousarray(np.asarray(conn_offsets, dtype=np.int32))
    tgt = np.ascontiguousarray(np.asarray(conn_targets, dtype=np.int32))
    if off.shape[0] != mt.shape[0] + 1:
        raise LstError(LST_ERR_ARG, "lst_load_geometry")
    out = C.c_void_p()
    st = _lib().lst_load_geometry(mt.ctypes.data_as(C.POINTER(lst_module)), mt.shape[0], off.ctypes.data_as(_ip),
                                  tgt.ctypes.data_as(_ip), C.byref(params) if params is not None else None,
                                  C.byref(out))
    _check(st, "lst_load_geometry")
    return out
