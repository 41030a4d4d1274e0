"""Marshalling of events into the C ABI structs and of lst_event_out into numpy arrays.

Inputs may be numpy arrays (host pointers) or CUDA torch tensors (device pointers); nothing is
computed here.  Result dictionaries use the same keys as the oracle's so tests can compare them.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from .binding import (LST_OK, N_STAGES, LstError, _check, _fp, _ip, _lib, lst_audit_report, lst_batch_summary, lst_caps,
                      lst_event_out, lst_hits, lst_pls)

_PLS_F = ("pt", "x0", "y0", "z0", "x1", "y1", "z1")


def _is_torch(a):
    return type(a).__module__.startswith("torch")


def _ptr(a, dtype, keep):
    """(pointer, n, on_device) of a numpy array or torch tensor; `keep` pins the converted object."""
    if a is None:
        return None, 0, 0
    if _is_torch(a):
        import torch

        want = torch.float32 if dtype == np.float32 else torch.int32
        if a.dtype != want or not a.is_contiguous():
            a = a.to(want).contiguous()
        keep.append(a)
        return C.c_void_p(a.data_ptr()), int(a.numel()), int(a.is_cuda)
    b = np.ascontiguousarray(np.asarray(a, dtype=dtype))
    keep.append(b)
    return C.c_void_p(b.ctypes.data), int(b.shape[0]), 0


def make_hits(x, y, z, sensor, event_offsets=None, keep=None):
    keep = keep if keep is not None else []
    h = lst_hits()
    h.x, n, dev = _ptr(x, np.float32, keep)
    h.y, n2, dev2 = _ptr(y, np.float32, keep)
    h.z, n3, dev3 = _ptr(z, np.float32, keep)
    u16 = (sensor.dtype == np.uint16) if isinstance(sensor, np.ndarray) else str(getattr(sensor, "dtype", "")) == "torch.uint16"
    if u16 and _is_torch(sensor):
        keep.append(sensor)
        h.sensor, n4, dev4 = C.c_void_p(sensor.data_ptr()), int(sensor.numel()), int(sensor.is_cuda)
    else:
        h.sensor, n4, dev4 = _ptr(sensor, np.uint16 if u16 else np.int32, keep)
    h.sensor_u16 = int(u16)
    if not (n == n2 == n3 == n4) or not (dev == dev2 == dev3 == dev4):
        raise ValueError("hit arrays must have equal length and live on the same side")
    h.n = n
    h.on_device = dev
    if event_offsets is not None:
        eo = np.ascontiguousarray(np.asarray(event_offsets, dtype=np.int32))
        keep.append(eo)
        h.event_offsets = C.c_void_p(eo.ctypes.data)
    else:
        h.event_offsets = None
    return h, keep


def make_pls(pls: dict | None, event_offsets=None, keep=None):
    keep = keep if keep is not None else []
    if not pls or len(pls["pt"]) == 0:
        return None, keep
    s = lst_pls()
    n = dev = None
    for f in _PLS_F:
        p, k, dv = _ptr(pls[f], np.float32, keep)
        setattr(s, f, p)
        if n is not None and (k != n or dv != dev):
            raise ValueError("pLS arrays must have equal length and live on the same side")
        n, dev = k, dv
    s.q, k, dv = _ptr(pls["q"], np.int32, keep)
    if k != n or dv != dev:
        raise ValueError("pLS arrays must have equal length and live on the same side")
    s.n = n
    s.on_device = dev
    if event_offsets is not None:
        eo = np.ascontiguousarray(np.asarray(event_offsets, dtype=np.int32))
        keep.append(eo)
        s.event_offsets = C.c_void_p(eo.ctypes.data)
    else:
        s.event_offsets = None
    return s, keep


def _np(ptr, shape, dtype):
    n = int(np.prod(shape))
    if n == 0:
        return np.zeros(shape, dtype=dtype)
    return np.ctypeslib.as_array(ptr, shape=(n,)).astype(dtype, copy=True).reshape(shape)


def event_out_to_dict(o: lst_event_out) -> dict:
    return {
        "md_hits": _np(o.md_hits, (o.n_md, 2), np.int32), "md_module": _np(o.md_module, (o.n_md,), np.int32),
        "md_f": _np(o.md_f, (o.n_md, 6), np.float32),
        "ls_md": _np(o.ls_md, (o.n_ls, 2), np.int32), "ls_kappa": _np(o.ls_kappa, (o.n_ls,), np.float32),
        "t3_ls": _np(o.t3_ls, (o.n_t3, 2), np.int32), "t3_md": _np(o.t3_md, (o.n_t3, 3), np.int32),
        "t3_k": _np(o.t3_k, (o.n_t3,), np.float32),
        "t5_t3": _np(o.t5_t3, (o.n_t5, 2), np.int32), "t5_md": _np(o.t5_md, (o.n_t5, 5), np.int32),
        "t5_score": _np(o.t5_score, (o.n_t5,), np.float32),
        "pt3": _np(o.pt3, (o.n_pt3, 2), np.int32), "pt3_score": _np(o.pt3_score, (o.n_pt3,), np.float32),
        "pt5": _np(o.pt5, (o.n_pt5, 2), np.int32), "pt5_score": _np(o.pt5_score, (o.n_pt5,), np.float32),
        "tc": _np(o.tc, (o.n_tc, 16), np.int32),
        "t4_t3": _np(o.t4_t3, (o.n_t4, 2), np.int32), "t4_md": _np(o.t4_md, (o.n_t4, 4), np.int32),
        "t4_score": _np(o.t4_score, (o.n_t4,), np.float32),
        "near": np.array([o.near[i] for i in range(N_STAGES)], dtype=np.int64),
        "n_tests": np.array([o.n_tests[i] for i in range(N_STAGES)], dtype=np.int64),
    }


def lst_run_event(geometry, x, y, z, sensor, pls: dict | None = None) -> dict:
    """One event through the whole chain (synchronous); returns every object array as numpy."""
    h, keep = make_hits(x, y, z, sensor)
    s, keep = make_pls(pls, keep=keep)
    out = C.POINTER(lst_event_out)()
    st = _lib().lst_run_event(geometry, C.byref(h), C.byref(s) if s is not None else None, C.byref(out))
    _check(st, "lst_run_event")
    try:
        return event_out_to_dict(out.contents)
    finally:
        _lib().lst_free(out)


def lst_ctx_create(geometry, caps: lst_caps | None = None, cuda_stream: int | None = None):
    ctx = C.c_void_p()
    st = _lib().lst_ctx_create(geometry, C.byref(caps) if caps is not None else None,
                               C.c_void_p(cuda_stream) if cuda_stream else None, C.byref(ctx))
    _check(st, "lst_ctx_create")
    return ctx


def lst_ctx_run(ctx, n_events: int, hits: lst_hits, seeds: lst_pls | None = None) -> None:
    st = _lib().lst_ctx_run(ctx, int(n_events), C.byref(hits), C.byref(seeds) if seeds is not None else None)
    _check(st, "lst_ctx_run")


def lst_ctx_sync(ctx) -> dict:
    s = lst_batch_summary()
    st = _lib().lst_ctx_sync(ctx, C.byref(s))
    _check(st, "lst_ctx_sync")
    return s.as_dict()


def lst_ctx_fetch_event(ctx, event: int) -> dict:
    out = C.POINTER(lst_event_out)()
    st = _lib().lst_ctx_fetch_event(ctx, int(event), C.byref(out))
    _check(st, "lst_ctx_fetch_event")
    try:
        return event_out_to_dict(out.contents)
    finally:
        _lib().lst_free(out)


def lst_ctx_fetch_tc(ctx, tc_buf: np.ndarray, n_events: int):
    """tc_buf: int32 [cap, 16] host array (e.g. pinned).  Returns (tc view, event offsets)."""
    off = np.zeros(n_events + 1, dtype=np.int32)
    st = _lib().lst_ctx_fetch_tc(ctx, tc_buf.ctypes.data_as(_ip), int(tc_buf.shape[0]), off.ctypes.data_as(_ip))
    _check(st, "lst_ctx_fetch_tc")
    return tc_buf[: off[-1]], off


def lst_ctx_set_blocks_per_sm(ctx, blocks: int) -> None:
    """Resident blocks per SM a kernel of this context may take (include/lst.h); 0 = default (fill the GPU)."""
    _check(_lib().lst_ctx_set_blocks_per_sm(ctx, int(blocks)), "lst_ctx_set_blocks_per_sm")


def lst_ctx_set_graph(ctx, enable: bool) -> None:
    """Replay the captured CUDA graph per batch (default on a caller's stream) or launch kernel by kernel."""
    _check(_lib().lst_ctx_set_graph(ctx, int(bool(enable))), "lst_ctx_set_graph")


def lst_ctx_set_timing(ctx, enable: bool) -> None:
    _check(_lib().lst_ctx_set_timing(ctx, int(bool(enable))), "lst_ctx_set_timing")


def lst_ctx_kernel_times(ctx) -> list:
    ms = (C.c_float * 64)()
    names = (C.c_char_p * 64)()
    n = _lib().lst_ctx_kernel_times(ctx, ms, names, 64)
    if n < 0:
        raise LstError(n, "lst_ctx_kernel_times")
    return [(names[i].decode(), float(ms[i])) for i in range(n)]


def lst_ctx_launch_count(ctx) -> int:
    return int(_lib().lst_ctx_launch_count(ctx))


LST_STAT_PT_QUEUE, LST_STAT_WORKSPACE_MB = 0, 1


def lst_ctx_stat(ctx, which: int) -> int:
    v = int(_lib().lst_ctx_stat(ctx, int(which)))
    if v < 0:
        raise LstError(v, "lst_ctx_stat")
    return v


def _scan_args(counts, offsets, where):
    """Device pointers of two CUDA int32 torch tensors (counts [n], offsets [n + 1]); nothing is copied or allocated."""
    import torch

    for t in (counts, offsets):
        if not (_is_torch(t) and t.is_cuda and t.dtype == torch.int32 and t.is_contiguous() and t.dim() == 1):
            raise ValueError(f"{where}: counts and offsets must be contiguous 1-d CUDA int32 tensors")
    n = int(counts.numel())
    if int(offsets.numel()) != n + 1:
        raise ValueError(f"{where}: offsets must hold len(counts) + 1 entries")
    return C.c_void_p(counts.data_ptr() if n else None), n, C.c_void_p(offsets.data_ptr())


def lst_scan_counts(counts, offsets, cuda_stream: int | None = None) -> None:
    """offsets[i] = counts[0] + ... + counts[i-1] with the chain's scan kernel; scratch from cudaMalloc, returns
    when the result is there (include/lst.h)."""
    c, n, o = _scan_args(counts, offsets, "lst_scan_counts")
    _check(_lib().lst_scan_counts(c, n, o, C.c_void_p(cuda_stream) if cuda_stream else None), "lst_scan_counts")


def lst_scan_counts_static(counts, offsets, cuda_stream: int | None = None) -> None:
    """The same scan for callers that may not allocate device memory (a framework that owns the device memory and
    bans cudaMalloc / cudaFree from its event loop because they stall every stream of the device): the scratch is a
    fixed array inside the library, so len(counts) is limited to LST_SCAN_STATIC_MAX_N (LstError with
    LST_ERR_LIMIT beyond it).  Asynchronous on `cuda_stream`; both tensors are the caller's and nothing is
    allocated here either.  Calls that could overlap on the GPU share the array and race: keep them ordered.
    Make the first call on a device outside any stream capture (it looks up the array's address)."""
    c, n, o = _scan_args(counts, offsets, "lst_scan_counts_static")
    _check(_lib().lst_scan_counts_static(c, n, o, C.c_void_p(cuda_stream) if cuda_stream else None),
           "lst_scan_counts_static")


AUDIT_STAGES = ("md", "ls", "pt3", "pt5")


def lst_ctx_audit(ctx) -> dict:
    """Re-evaluates every MD, LS, pT3 and pT5 candidate of the last synchronised batch with the exact cuts on the GPU
    and compares counts, near flags and a hash of the accepted set with what the chain produced (include/lst.h)."""
    rep = lst_audit_report()
    _check(_lib().lst_ctx_audit(ctx, C.byref(rep)), "lst_ctx_audit")
    return rep.as_dict()
