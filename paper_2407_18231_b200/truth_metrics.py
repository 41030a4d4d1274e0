"""Efficiency, fake rate and duplicate rate of the track candidates against the synthetic truth,
with the definitions of PAPER.md:54-58 (section 3): a simulated track matches a reconstructed one if
more than 75 % of the hits of the reconstructed track come from it; efficiency = matched fraction of
the selected simulated tracks; fake rate = fraction of reconstructed tracks matched to no simulated
track; duplicate rate = fraction of reconstructed tracks matched to a simulated track that is matched
to several reconstructed tracks.  SURVEY.md section 8(f) item 1: the synthetic analogue of the
paper's Figs. 3-4 in form, not in values (the CMS sample is not available).  Pure numpy on the
OUTPUT of the chain; it holds none of the method's arithmetic.
"""
from __future__ import annotations

import numpy as np

PT_EDGES = (0.8, 1.0, 1.5, 2.0, 3.0, 5.0, 10.0, np.inf)


def match_candidates(tc: np.ndarray, hit_truth: np.ndarray, pls_truth: np.ndarray | None = None) -> np.ndarray:
    """Simulated track matched to every track candidate (-1 = fake).  tc: [n, 16] rows
    (type, pls, t5, t3, hit_idx[12]); the two pixel hits of a candidate's seed count as hits of the
    seed's truth track (a pLS-only candidate is matched by its seed alone)."""
    tc = np.asarray(tc).reshape(-1, 16)
    out = np.full(tc.shape[0], -1, dtype=np.int64)
    for k, row in enumerate(tc):
        idx = row[4:16]
        labels = list(np.asarray(hit_truth)[idx[idx >= 0]])
        if row[1] >= 0 and pls_truth is not None:
            labels += [int(pls_truth[row[1]])] * 2
        if not labels:
            continue
        vals, counts = np.unique(np.asarray(labels), return_counts=True)
        best = int(np.argmax(counts))
        if vals[best] >= 0 and counts[best] > 0.75 * len(labels):
            out[k] = int(vals[best])
    return out


def track_candidate_metrics(tc, hit_truth, trk: dict, pls_truth=None, pt_min: float = 0.8, d0_max: float = 0.0) -> dict:
    """trk: truth parameters per simulated track ("pt", "d0", ...), as lst_inputs.Event.trk."""
    match = match_candidates(tc, hit_truth, pls_truth)
    pt, d0 = np.asarray(trk["pt"]), np.asarray(trk["d0"])
    selected = (pt > pt_min) & (d0 <= d0_max)  # prompt tracks above LST's threshold
    n_reco_of = np.bincount(match[match >= 0], minlength=pt.shape[0])
    found = n_reco_of > 0
    eff_vs_pt = []
    for lo, hi in zip(PT_EDGES[:-1], PT_EDGES[1:]):
        sel = selected & (pt >= lo) & (pt < hi)
        eff_vs_pt.append(float(found[sel].mean()) if sel.any() else float("nan"))
    matched = match >= 0
    dup = matched & (n_reco_of[np.where(matched, match, 0)] > 1)
    n_tc = int(match.shape[0])
    return {
        "n_sim_selected": int(selected.sum()), "n_tc": n_tc,
        "efficiency": float(found[selected].mean()) if selected.any() else float("nan"),
        "fake_rate": float((~matched).mean()) if n_tc else float("nan"),
        "duplicate_rate": float(dup.mean()) if n_tc else float("nan"),
        "pt_edges": list(PT_EDGES), "efficiency_vs_pt": eff_vs_pt,
    }
