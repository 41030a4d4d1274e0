"""ctypes loader for oracle/lst_oracle.c -- TEST INFRASTRUCTURE ONLY (see lst_oracle.h)."""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lst_oracle.c")
_HDR = os.path.join(_HERE, "lst_oracle.h")
_SO = os.path.join(_HERE, "liblst_oracle.so")

STAGES = ("md", "ls", "t3", "t5", "pt3", "pt5", "t4")
KINDS = ("md", "ls", "t3", "t5", "pt3", "pt5", "tc", "t4")
_KIND_W = (3, 2, 5, 7, 2, 2, 16, 6)
_KIND_FW = (6, 1, 1, 1, 1, 1, 0, 1)
N_STAGES = len(STAGES)
_EXT_FIELDS = ("t4_tol0", "t4_tol1", "t5_mlp_scale", "t5_mlp_thr")

_FLOAT_FIELDS = (
    "b_field", "pt_min", "z0_max", "md_b_phi_tol", "md_z_tol", "md_e_slope", "md_e_tol",
    "ls_kappa_max", "ls_z_tol", "ls_dir_tol", "t3_kappa_max", "t3_z_tol0", "t3_z_tol1",
    "t5_tol0", "t5_tol1", "pt_gate_tol", "pt_k_tol0", "pt_k_tol1", "pt_z_tol", "near_rel",
)


class Params(C.Structure):
    _fields_ = [(f, C.c_float) for f in _FLOAT_FIELDS] + [("stage_mask", C.c_int)] + \
               [(f, C.c_float) for f in _EXT_FIELDS] + [("t5_mlp", C.c_float * 65)]

    def as_dict(self):
        d = {f: float(np.float32(getattr(self, f))) for f in _FLOAT_FIELDS + _EXT_FIELDS}
        d["stage_mask"] = int(self.stage_mask)
        return d


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (no FMA contraction, no fast-math)."""
    if not force and os.path.exists(_SO):
        if os.path.getmtime(_SO) >= max(os.path.getmtime(_SRC), os.path.getmtime(_HDR)):
            return _SO
    tmp = _SO + f".tmp{os.getpid()}"
    cmd = ["gcc", "-O2", "-ffp-contract=off", "-fno-fast-math", "-std=c99", "-Wall", "-shared", "-fPIC",
           "-o", tmp, _SRC, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, _SO)
    return _SO


_lib = None


def _load():
    global _lib
    if _lib is not None:
        return _lib
    lib = C.CDLL(build())
    fp = C.POINTER(C.c_float)
    ip = C.POINTER(C.c_int)
    pp = C.POINTER(Params)
    lib.orc_default_params.argtypes = [pp]
    lib.orc_derived.argtypes = [pp, fp]
    lib.orc_g.argtypes = [C.c_float]
    lib.orc_g.restype = C.c_float
    lib.orc_kappa3.argtypes = [C.c_float] * 6 + [fp]
    lib.orc_kappa3.restype = C.c_float
    lib.orc_md_test.argtypes = [pp, C.c_int] + [C.c_float] * 6 + [fp, ip]
    lib.orc_ls_test.argtypes = [pp, fp, C.c_int, fp, C.c_int, fp, ip]
    lib.orc_t3_test.argtypes = [pp, fp, C.c_int, fp, C.c_int, fp, C.c_int, fp, ip]
    lib.orc_t5_test.argtypes = [pp, C.c_float, C.c_float, fp, fp, fp, fp, ip]
    lib.orc_t4_test.argtypes = [pp, C.c_float, C.c_float, fp, ip]
    lib.orc_pt_test.argtypes = [pp, fp, fp, C.c_int, fp, C.c_int, fp, C.c_int, C.c_float, fp, ip]
    cp = C.POINTER(C.c_char)
    lib.orc_dedup.argtypes = [ip, ip, C.c_int, ip, C.c_int, fp, ip, C.c_int, fp, ip, C.c_int, fp, C.c_int,
                              cp, cp, cp, cp]
    lib.orc_dedup_t4.argtypes = [ip, ip, ip, C.c_int, ip, C.c_int, ip, C.c_int, cp, cp, cp, ip, C.c_int, fp, cp]
    lib.orc_run_event.restype = C.c_void_p
    lib.orc_run_event.argtypes = [pp, C.c_int, ip, ip, ip, C.c_int, fp, fp, fp, ip, C.c_int, fp, ip,
                                  fp, fp, fp, fp, fp, fp]
    lib.orc_free_event.argtypes = [C.c_void_p]
    lib.orc_count.argtypes = [C.c_void_p, C.c_int]
    lib.orc_copy_i32.argtypes = [C.c_void_p, C.c_int, ip]
    lib.orc_copy_f32.argtypes = [C.c_void_p, C.c_int, fp]
    lib.orc_counters.argtypes = [C.c_void_p, C.POINTER(C.c_longlong), C.POINTER(C.c_longlong)]
    _lib = lib
    return lib


def default_params(**overrides) -> Params:
    p = Params()
    _load().orc_default_params(C.byref(p))
    for k, v in overrides.items():
        if not hasattr(p, k):
            raise KeyError(k)
        if k == "t5_mlp":
            w = np.asarray(v, dtype=np.float32).ravel()
            assert w.shape[0] == 65
            for i in range(65):
                p.t5_mlp[i] = float(w[i])
        else:
            setattr(p, k, v)
    return p


def _params(p):
    return p if p is not None else default_params()


def derived(p: Params | None = None):
    out = (C.c_float * 3)()
    _load().orc_derived(C.byref(_params(p)), out)
    return {"KR": np.float32(out[0]), "R_MIN": np.float32(out[1]), "INV_2RMIN": np.float32(out[2])}


def g(u) -> np.float32:
    return np.float32(_load().orc_g(C.c_float(float(np.float32(u)))))


def kappa3(P, Q, S):
    ln = (C.c_float * 3)()
    a = [C.c_float(float(np.float32(v))) for v in (P[0], P[1], Q[0], Q[1], S[0], S[1])]
    k = _load().orc_kappa3(*a, ln)
    return np.float32(k), np.array(ln[:], dtype=np.float32)


def _fa(v, n):
    a = np.ascontiguousarray(np.asarray(v, dtype=np.float32).ravel())
    assert a.shape[0] >= n, (a.shape, n)
    return a, a.ctypes.data_as(C.POINTER(C.c_float))


def md_test(a, b, endcap: bool, p: Params | None = None):
    """a, b = (x, y, z) of the lower / upper hit."""
    vals = (C.c_float * 8)()
    near = C.c_int(0)
    f = [C.c_float(float(np.float32(v))) for v in (*a[:3], *b[:3])]
    acc = _load().orc_md_test(C.byref(_params(p)), int(bool(endcap)), *f, vals, C.byref(near))
    v = np.array(vals[:], dtype=np.float32)
    names = ("crs", "lim", "rv", "rl") if endcap else ("dd", "dot", "crs", "lim", "zv", "zl", "ux", "uy")
    return bool(acc), bool(near.value), dict(zip(names, v))


def ls_test(mdA, eA: bool, mdB, eB: bool, p: Params | None = None):
    """md = (x, y, z, r, ux, uy)."""
    vals = (C.c_float * 8)()
    near = C.c_int(0)
    a, pa = _fa(mdA, 6)
    b, pb = _fa(mdB, 6)
    acc = _load().orc_ls_test(C.byref(_params(p)), pa, int(bool(eA)), pb, int(bool(eB)), vals, C.byref(near))
    names = ("kappa", "kv", "rho", "zv", "zl", "half", "dA", "dB")
    return bool(acc), bool(near.value), dict(zip(names, np.array(vals[:], dtype=np.float32)))


def t3_test(mdA, eA, mdB, eB, mdC, eC, p: Params | None = None):
    vals = (C.c_float * 4)()
    near = C.c_int(0)
    a, pa = _fa(mdA, 4)
    b, pb = _fa(mdB, 4)
    c, pc = _fa(mdC, 4)
    acc = _load().orc_t3_test(C.byref(_params(p)), pa, int(bool(eA)), pb, int(bool(eB)), pc, int(bool(eC)),
                              vals, C.byref(near))
    names = ("k3", "ratio", "zv", "tol")
    return bool(acc), bool(near.value), dict(zip(names, np.array(vals[:], dtype=np.float32)))


def t5_test(ki, ko, mdB, mdC, mdD, p: Params | None = None):
    vals = (C.c_float * 4)()
    near = C.c_int(0)
    b, pb = _fa(mdB, 2)
    c, pc = _fa(mdC, 2)
    d, pd = _fa(mdD, 2)
    acc = _load().orc_t5_test(C.byref(_params(p)), C.c_float(float(np.float32(ki))),
                              C.c_float(float(np.float32(ko))), pb, pc, pd, vals, C.byref(near))
    names = ("kb", "tol", "score", "s")
    return bool(acc), bool(near.value), dict(zip(names, np.array(vals[:4], dtype=np.float32)))


def t4_test(k1, k2, p: Params | None = None):
    """CUTS.md section 10: two T3 curvatures -> (accept, near, {d, tol, score})."""
    vals = (C.c_float * 4)()
    near = C.c_int(0)
    acc = _load().orc_t4_test(C.byref(_params(p)), C.c_float(float(np.float32(k1))), C.c_float(float(np.float32(k2))),
                              vals, C.byref(near))
    return bool(acc), bool(near.value), dict(zip(("d", "tol", "score"), np.array(vals[:3], dtype=np.float32)))


def pt_test(pls, mdA, eA, mdL, eL, kt, base_score=0.0, p: Params | None = None):
    """pls = (pt, q, x0, y0, z0, x1, y1, z1); kt = stored curvatures of the T3 (1) / T5 (2)."""
    vals = (C.c_float * 8)()
    near = C.c_int(0)
    s, ps = _fa(pls, 8)
    a, pa = _fa(mdA, 4)
    l, pl = _fa(mdL, 4)
    k, pk = _fa(kt, 1)
    acc = _load().orc_pt_test(C.byref(_params(p)), ps, pa, int(bool(eA)), pl, int(bool(eL)), pk, int(k.shape[0]),
                              C.c_float(float(np.float32(base_score))), vals, C.byref(near))
    names = ("kp", "gdot", "gcrs", "glim", "kx", "zqA", "zqL", "score")
    return bool(acc), bool(near.value), dict(zip(names, np.array(vals[:], dtype=np.float32)))


def dedup(md_hits, t3_md, t5_md, t5_score, pt3, pt3_score, pt5, pt5_score, n_pls):
    """CUTS.md section 8 on plain arrays; returns (keep5, keep3, keepT, linked) as bool arrays."""
    ip = C.POINTER(C.c_int)
    fp = C.POINTER(C.c_float)
    cp = C.POINTER(C.c_char)

    def i32(a, w):
        return np.ascontiguousarray(np.asarray(a, dtype=np.int32).reshape(-1, w))

    def f32(a):
        return np.ascontiguousarray(np.asarray(a, dtype=np.float32).ravel())

    md_hits, t3_md, t5_md, pt3, pt5 = i32(md_hits, 2), i32(t3_md, 3), i32(t5_md, 5), i32(pt3, 2), i32(pt5, 2)
    t5_score, pt3_score, pt5_score = f32(t5_score), f32(pt3_score), f32(pt5_score)
    assert len(t5_score) == len(t5_md) and len(pt3_score) == len(pt3) and len(pt5_score) == len(pt5)
    keep5 = np.zeros(len(pt5) + 1, dtype=np.uint8)
    keep3 = np.zeros(len(pt3) + 1, dtype=np.uint8)
    keepT = np.zeros(len(t5_md) + 1, dtype=np.uint8)
    linked = np.zeros(n_pls + 1, dtype=np.uint8)
    _load().orc_dedup(md_hits.ctypes.data_as(ip), t3_md.ctypes.data_as(ip), len(t3_md), t5_md.ctypes.data_as(ip),
                      len(t5_md), t5_score.ctypes.data_as(fp), pt3.ctypes.data_as(ip), len(pt3),
                      pt3_score.ctypes.data_as(fp), pt5.ctypes.data_as(ip), len(pt5), pt5_score.ctypes.data_as(fp),
                      int(n_pls), keep5.ctypes.data_as(cp), keep3.ctypes.data_as(cp), keepT.ctypes.data_as(cp),
                      linked.ctypes.data_as(cp))
    return keep5[:-1].astype(bool), keep3[:-1].astype(bool), keepT[:-1].astype(bool), linked[:-1].astype(bool)


def dedup_t4(md_hits, t3_md, t5_md, pt3, pt5, keep5, keep3, keepT, t4_md, t4_score):
    """CUTS.md section 10 rule 5; returns keep4 as a bool array."""
    ip = C.POINTER(C.c_int)
    fp = C.POINTER(C.c_float)
    cp = C.POINTER(C.c_char)

    def i32(a, w):
        return np.ascontiguousarray(np.asarray(a, dtype=np.int32).reshape(-1, w))

    md_hits, t3_md, t5_md, pt3, pt5, t4_md = i32(md_hits, 2), i32(t3_md, 3), i32(t5_md, 5), i32(pt3, 2), i32(pt5, 2), i32(t4_md, 4)
    t4_score = np.ascontiguousarray(np.asarray(t4_score, dtype=np.float32).ravel())
    k5, k3, kT = (np.ascontiguousarray(np.append(np.asarray(k, dtype=np.uint8), 0)) for k in (keep5, keep3, keepT))
    keep4 = np.zeros(len(t4_md) + 1, dtype=np.uint8)
    _load().orc_dedup_t4(md_hits.ctypes.data_as(ip), t3_md.ctypes.data_as(ip), t5_md.ctypes.data_as(ip), len(t5_md),
                         pt3.ctypes.data_as(ip), len(pt3), pt5.ctypes.data_as(ip), len(pt5), k5.ctypes.data_as(cp),
                         k3.ctypes.data_as(cp), kT.ctypes.data_as(cp), t4_md.ctypes.data_as(ip), len(t4_md),
                         t4_score.ctypes.data_as(fp), keep4.ctypes.data_as(cp))
    return keep4[:-1].astype(bool)


def run_event(subdet, conn_off, conn_tgt, x, y, z, sensor, pls: dict | None = None, params: Params | None = None):
    """Run the chain on one event; returns a dict of numpy arrays (indices local to this event)."""
    lib = _load()
    fp = C.POINTER(C.c_float)
    ip = C.POINTER(C.c_int)

    def f32(a):
        return np.ascontiguousarray(np.asarray(a, dtype=np.float32))

    def i32(a):
        return np.ascontiguousarray(np.asarray(a, dtype=np.int32))

    subdet, conn_off, conn_tgt, sensor = i32(subdet), i32(conn_off), i32(conn_tgt), i32(sensor)
    x, y, z = f32(x), f32(y), f32(z)
    n_pls = 0
    pl = {}
    if pls and len(pls.get("pt", ())) > 0:
        n_pls = len(pls["pt"])
        pl = {k: f32(pls[k]) for k in ("pt", "x0", "y0", "z0", "x1", "y1", "z1")}
        pl["q"] = i32(pls["q"])

    def pf(k):
        return pl[k].ctypes.data_as(fp) if n_pls else None

    h = lib.orc_run_event(
        C.byref(_params(params)), int(subdet.shape[0]), subdet.ctypes.data_as(ip), conn_off.ctypes.data_as(ip),
        conn_tgt.ctypes.data_as(ip), int(x.shape[0]), x.ctypes.data_as(fp), y.ctypes.data_as(fp),
        z.ctypes.data_as(fp), sensor.ctypes.data_as(ip), n_pls, pf("pt"),
        pl["q"].ctypes.data_as(ip) if n_pls else None, pf("x0"), pf("y0"), pf("z0"), pf("x1"), pf("y1"), pf("z1"))
    if not h:
        raise ValueError("oracle: invalid input (sensor id or connection map out of range)")
    try:
        raw_i, raw_f = {}, {}
        for k, name in enumerate(KINDS):
            n = lib.orc_count(h, k)
            ai = np.zeros((n, _KIND_W[k]), dtype=np.int32)
            if n:
                lib.orc_copy_i32(h, k, ai.ctypes.data_as(ip))
            raw_i[name] = ai
            af = np.zeros((n, _KIND_FW[k]), dtype=np.float32)
            if n and _KIND_FW[k]:
                lib.orc_copy_f32(h, k, af.ctypes.data_as(fp))
            raw_f[name] = af
        near = (C.c_longlong * N_STAGES)()
        nt = (C.c_longlong * N_STAGES)()
        lib.orc_counters(h, near, nt)
    finally:
        lib.orc_free_event(h)
    return {
        "md_hits": raw_i["md"][:, 0:2].copy(), "md_module": raw_i["md"][:, 2].copy(), "md_f": raw_f["md"],
        "ls_md": raw_i["ls"], "ls_kappa": raw_f["ls"][:, 0].copy(),
        "t3_ls": raw_i["t3"][:, 0:2].copy(), "t3_md": raw_i["t3"][:, 2:5].copy(), "t3_k": raw_f["t3"][:, 0].copy(),
        "t5_t3": raw_i["t5"][:, 0:2].copy(), "t5_md": raw_i["t5"][:, 2:7].copy(),
        "t5_score": raw_f["t5"][:, 0].copy(),
        "pt3": raw_i["pt3"], "pt3_score": raw_f["pt3"][:, 0].copy(),
        "pt5": raw_i["pt5"], "pt5_score": raw_f["pt5"][:, 0].copy(),
        "tc": raw_i["tc"],
        "t4_t3": raw_i["t4"][:, 0:2].copy(), "t4_md": raw_i["t4"][:, 2:6].copy(), "t4_score": raw_f["t4"][:, 0].copy(),
        "near": np.array(near[:], dtype=np.int64), "n_tests": np.array(nt[:], dtype=np.int64),
    }
