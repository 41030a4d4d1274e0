"""Test helpers: canonical (implementation-independent) form of a chain result.

Objects are identified by their tuples of INPUT hit indices (north_star: "bit-exact sets of object
index tuples"); object indices (md/ls/t3/t5 numbers) are implementation-local and never compared.
"""
from __future__ import annotations

import numpy as np


def _sort_rows(keys: np.ndarray, *payload):
    if keys.shape[0] == 0:
        return (keys,) + tuple(payload)
    order = np.lexsort(keys.T[::-1])
    return (keys[order],) + tuple(p[order] for p in payload)


def canon(res: dict) -> dict:
    """Sorted hit-index tuples per object kind, with the float payload aligned to that order."""
    mdh = np.asarray(res["md_hits"], dtype=np.int64).reshape(-1, 2)
    out = {}
    k, mod, mf = _sort_rows(mdh, np.asarray(res["md_module"]), np.asarray(res["md_f"], dtype=np.float32))
    out["md"], out["md_module"], out["md_f"] = k, mod, mf

    ls = np.asarray(res["ls_md"], dtype=np.int64).reshape(-1, 2)
    k, kap = _sort_rows(mdh[ls].reshape(-1, 4), np.asarray(res["ls_kappa"], dtype=np.float32))
    out["ls"], out["ls_kappa"] = k, kap

    t3 = np.asarray(res["t3_md"], dtype=np.int64).reshape(-1, 3)
    t3h = mdh[t3].reshape(-1, 6)
    k, k3 = _sort_rows(t3h, np.asarray(res["t3_k"], dtype=np.float32))
    out["t3"], out["t3_k"] = k, k3

    t5 = np.asarray(res["t5_md"], dtype=np.int64).reshape(-1, 5)
    t5h = mdh[t5].reshape(-1, 10)
    k, sc = _sort_rows(t5h, np.asarray(res["t5_score"], dtype=np.float32))
    out["t5"], out["t5_score"] = k, sc

    pt3 = np.asarray(res["pt3"], dtype=np.int64).reshape(-1, 2)
    k, sc = _sort_rows(np.concatenate([pt3[:, :1], t3h[pt3[:, 1]]], axis=1) if len(pt3) else np.zeros((0, 7), np.int64),
                       np.asarray(res["pt3_score"], dtype=np.float32))
    out["pt3"], out["pt3_score"] = k, sc

    pt5 = np.asarray(res["pt5"], dtype=np.int64).reshape(-1, 2)
    k, sc = _sort_rows(np.concatenate([pt5[:, :1], t5h[pt5[:, 1]]], axis=1) if len(pt5) else np.zeros((0, 11), np.int64),
                       np.asarray(res["pt5_score"], dtype=np.float32))
    out["pt5"], out["pt5_score"] = k, sc

    tc = np.asarray(res["tc"], dtype=np.int64).reshape(-1, 16)
    out["tc_order_types"] = tc[:, 0].copy()  # class order pT5, pT3, T5, pLS must be non-decreasing
    (out["tc"],) = _sort_rows(np.concatenate([tc[:, 0:2], tc[:, 4:16]], axis=1))
    # extension (CUTS.md section 10): T4 objects, empty unless stage-mask bit 6 is set
    t4 = np.asarray(res.get("t4_md", np.zeros((0, 4))), dtype=np.int64).reshape(-1, 4)
    k, sc = _sort_rows(mdh[t4].reshape(-1, 8) if len(t4) else np.zeros((0, 8), np.int64),
                       np.asarray(res.get("t4_score", np.zeros(0)), dtype=np.float32))
    out["t4"], out["t4_score"] = k, sc
    out["near"] = np.asarray(res["near"], dtype=np.int64)
    out["n_tests"] = np.asarray(res["n_tests"], dtype=np.int64)
    return out


def assert_same(a: dict, b: dict, what: str = ""):
    """Bit-exact equality of two canonical results (index tuples AND float payloads)."""
    for key in ("md", "md_module", "ls", "t3", "t5", "pt3", "pt5", "t4", "tc", "near", "n_tests"):
        assert a[key].shape == b[key].shape, f"{what}{key}: count {a[key].shape} vs {b[key].shape}"
        assert np.array_equal(a[key], b[key]), f"{what}{key}: tuples differ"
    for key in ("md_f", "ls_kappa", "t3_k", "t5_score", "pt3_score", "pt5_score", "t4_score"):
        fa, fb = np.ascontiguousarray(a[key]), np.ascontiguousarray(b[key])
        na, nb = np.isnan(fa), np.isnan(fb)  # a NaN has no defined bit pattern (x86 and sm_100 produce different ones)
        assert np.array_equal(na, nb), f"{what}{key}: NaN payloads in different places"
        x = np.where(na, 0, fa.view(np.int32))
        y = np.where(nb, 0, fb.view(np.int32))
        assert np.array_equal(x, y), f"{what}{key}: float payload not bit-identical"
    assert np.all(np.diff(a["tc_order_types"]) >= 0) and np.all(np.diff(b["tc_order_types"]) >= 0), "TC class order"


def exact_helix_points(pt, q, phi0, eta, z0, radii):
    """Noise-free prompt-helix points at the given transverse radii (float64), via lst_inputs.helix."""
    from lst_inputs.helix import Tracks

    trk = Tracks([0.0], [0.0], [z0], [phi0], [eta], [pt], [q])
    pts = []
    for r in radii:
        t = np.nanmin(trk.cyl_crossings(float(r), 1), axis=1)
        x, y, z = trk.pos(t)
        pts.append((x[0], y[0], z[0]))
    return np.array(pts), trk


def run_batch(lst, ctx, events, with_seeds: bool = True):
    """Concatenates lst_inputs Events into one batch, runs it on `ctx` and syncs; returns the summary."""
    from lst_inputs.events import concat_events

    b = concat_events(events)
    h, keep = lst.make_hits(b["x"], b["y"], b["z"], b["sensor"], b["hit_offsets"])
    s, keep = lst.make_pls(b["pls"] if with_seeds else None, b["pls_offsets"], keep)
    lst.lst_ctx_run(ctx, len(events), h, s)
    return lst.lst_ctx_sync(ctx)
