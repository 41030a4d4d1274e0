"""Efficiency, fake rate and duplicate rate of the track candidates against the synthetic truth, with
the definitions of PAPER.md:54-58 (section 3) and the axes of its Figs. 3-4:

* a simulated track matches a reconstructed one if MORE than 75 % of the hits of the reconstructed
  track come from it;
* efficiency = matched fraction of the selected simulated tracks, shown against the simulated pT and
  against r_vertex, the radial distance of the production vertex (Fig. 3);
* fake rate = fraction of reconstructed tracks matched to no simulated track; duplicate rate = fraction
  of reconstructed tracks matched to a simulated track that is matched to several reconstructed tracks;
  both against the RECONSTRUCTED pT (Fig. 4).

SURVEY.md section 8(f) item 1: the synthetic analogue of those figures in form, not in values (the CMS
sample is not available).  Pure numpy on the OUTPUT of the chain (the oracle's or the CUDA path's -- both
give the same dictionaries) and on the generator's truth labels; it holds none of the method's
arithmetic and lives with the generator whose labels it reads.
"""
from __future__ import annotations

import numpy as np

from .helix import KR

PT_EDGES = (0.8, 1.0, 1.5, 2.0, 3.0, 5.0, 10.0, np.inf)
RVTX_EDGES = (0.0, 0.5, 2.0, 5.0, 10.0, 15.0, 20.0)


def match_candidates(tc: np.ndarray, hit_truth: np.ndarray, pls_truth: np.ndarray | None = None) -> np.ndarray:
    """Simulated track matched to every track candidate (-1 = fake).  tc: [n, 16] rows
    (type, pls, t5, t3, hit_idx[12]); the two pixel hits of a candidate's seed count as hits of the
    seed's truth track (a pLS-only candidate is matched by its seed alone)."""
    tc = np.asarray(tc).reshape(-1, 16)
    out = np.full(tc.shape[0], -1, dtype=np.int64)
    hit_truth = np.asarray(hit_truth)
    for k, row in enumerate(tc):
        idx = row[4:16]
        labels = list(hit_truth[idx[idx >= 0]])
        if row[1] >= 0 and pls_truth is not None:
            labels += [int(pls_truth[row[1]])] * 2
        if not labels:
            continue
        vals, counts = np.unique(np.asarray(labels), return_counts=True)
        best = int(np.argmax(counts))
        if vals[best] >= 0 and counts[best] > 0.75 * len(labels):
            out[k] = int(vals[best])
    return out


def reconstructed_pt(result: dict, pls: dict | None) -> np.ndarray:
    """pT of every track candidate as the chain knows it: the seed's pT for pT5 / pT3 / pLS candidates;
    for a T5 without seed, R = pT KR with 1/R = mean |curvature| of its two T3s (north_star: R = pT/(0.3 B))."""
    tc = np.asarray(result["tc"]).reshape(-1, 16)
    out = np.full(tc.shape[0], np.nan)
    seeded = tc[:, 1] >= 0
    if seeded.any():
        out[seeded] = np.asarray(pls["pt"], dtype=np.float64)[tc[seeded, 1]]
    t5 = ~seeded & (tc[:, 2] >= 0)
    if t5.any():
        t3 = np.asarray(result["t5_t3"])[tc[t5, 2]]
        k = 0.5 * (np.abs(np.asarray(result["t3_k"], dtype=np.float64)[t3[:, 0]]) +
                   np.abs(np.asarray(result["t3_k"], dtype=np.float64)[t3[:, 1]]))
        out[t5] = 1.0 / (np.maximum(k, 1e-9) * KR)
    return out


def _binned(mask_num, mask_den, x, edges):
    out = []
    for lo, hi in zip(edges[:-1], edges[1:]):
        sel = mask_den & (x >= lo) & (x < hi)
        out.append([int(sel.sum()), float(mask_num[sel].mean()) if sel.any() else float("nan")])
    return out


def track_candidate_metrics(result: dict, ev, pt_min: float = 0.8, classes=(0, 1, 2, 3)) -> dict:
    """result: output dictionary of one event (oracle.run_event or lst_ctx_fetch_event / lst_run_event);
    ev: the lst_inputs Event it came from.  `classes` restricts the candidates (0 pT5, 1 pT3, 2 T5, 3 pLS)."""
    tc_all = np.asarray(result["tc"]).reshape(-1, 16)
    keep = np.isin(tc_all[:, 0], classes)
    res = dict(result, tc=tc_all[keep])
    tc = res["tc"]
    pls_truth = ev.pls["truth"] if ev.pls else None
    match = match_candidates(tc, ev.truth, pls_truth)
    pt, d0 = np.asarray(ev.trk["pt"]), np.asarray(ev.trk["d0"])
    n_reco_of = np.bincount(match[match >= 0], minlength=pt.shape[0])
    found = n_reco_of > 0
    above = pt > pt_min                    # LST's lower threshold
    prompt = above & (d0 <= 0.0)           # the stand-in for "from the hard-scattering vertex"
    matched = match >= 0
    dup = matched & (n_reco_of[np.where(matched, match, 0)] > 1)
    rpt = reconstructed_pt(res, ev.pls)
    n_tc = int(tc.shape[0])
    ones = np.ones(n_tc, dtype=bool)
    return {
        "n_sim_prompt": int(prompt.sum()), "n_sim_displaced": int((above & (d0 > 0.0)).sum()), "n_tc": n_tc,
        "n_tc_by_class": [int((tc[:, 0] == c).sum()) for c in range(4)],
        "efficiency": float(found[prompt].mean()) if prompt.any() else float("nan"),
        "efficiency_displaced": float(found[above & (d0 > 0.0)].mean()) if (above & (d0 > 0.0)).any() else float("nan"),
        "fake_rate": float((~matched).mean()) if n_tc else float("nan"),
        "duplicate_rate": float(dup.mean()) if n_tc else float("nan"),
        "pt_edges": list(PT_EDGES), "rvtx_edges": list(RVTX_EDGES),
        "efficiency_vs_pt": _binned(found, prompt, pt, PT_EDGES),            # Fig. 3 left: [n_sim, efficiency]
        "efficiency_vs_rvtx": _binned(found, above, d0, RVTX_EDGES),         # Fig. 3 right (r_vertex = d0 here)
        "fake_rate_vs_pt": _binned(~matched, ones, rpt, PT_EDGES),           # Fig. 4 left: [n_reco, rate]
        "duplicate_rate_vs_pt": _binned(dup, ones, rpt, PT_EDGES),           # Fig. 4 right
    }


def merge_metrics(ms: list) -> dict:
    """Event-weighted combination of per-event metric dictionaries (counts add, rates are re-weighted)."""
    out = {"n_events": len(ms)}
    for key in ("n_sim_prompt", "n_sim_displaced", "n_tc"):
        out[key] = int(sum(m[key] for m in ms))
    out["n_tc_by_class"] = [int(sum(m["n_tc_by_class"][c] for m in ms)) for c in range(4)]

    def wavg(vals, weights):
        v, w = np.asarray(vals, dtype=float), np.asarray(weights, dtype=float)
        ok = np.isfinite(v) & (w > 0)
        return float((v[ok] * w[ok]).sum() / w[ok].sum()) if ok.any() else float("nan")

    out["efficiency"] = wavg([m["efficiency"] for m in ms], [m["n_sim_prompt"] for m in ms])
    out["efficiency_displaced"] = wavg([m["efficiency_displaced"] for m in ms], [m["n_sim_displaced"] for m in ms])
    out["fake_rate"] = wavg([m["fake_rate"] for m in ms], [m["n_tc"] for m in ms])
    out["duplicate_rate"] = wavg([m["duplicate_rate"] for m in ms], [m["n_tc"] for m in ms])
    out["pt_edges"], out["rvtx_edges"] = ms[0]["pt_edges"], ms[0]["rvtx_edges"]
    for key in ("efficiency_vs_pt", "efficiency_vs_rvtx", "fake_rate_vs_pt", "duplicate_rate_vs_pt"):
        rows = []
        for b in range(len(ms[0][key])):
            n = sum(m[key][b][0] for m in ms)
            rows.append([int(n), wavg([m[key][b][1] for m in ms], [m[key][b][0] for m in ms])])
        out[key] = rows
    return out
