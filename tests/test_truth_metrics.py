"""Synthetic-truth sanity of the track candidates with the paper's metric definitions and the
axes of its Figs. 3-4: not parity, a physics check that the stand-in cuts build tracks."""
import numpy as np

from lst_inputs import make_config_event, make_config_geometry
from lst_inputs.truth_metrics import match_candidates, merge_metrics, reconstructed_pt, track_candidate_metrics


def test_matching_rule_is_more_than_75_percent():
    truth = np.array([5, 5, 5, 5, 7, -1, 5, 5, 5, 5], dtype=np.int64)
    tc = -np.ones((3, 16), dtype=np.int64)
    tc[0, 0], tc[0, 4:14] = 2, np.arange(10)          # 8 of 10 hits from track 5 -> matched
    tc[1, 0], tc[1, 4:8] = 2, [0, 1, 2, 4]            # 3 of 4 = 75 %, not MORE than 75 % -> fake
    tc[2, 0], tc[2, 1] = 3, 0                          # pLS-only: matched by its seed
    assert match_candidates(tc, truth, pls_truth=np.array([9])).tolist() == [5, -1, 9]
    assert match_candidates(tc[2:], truth, pls_truth=np.array([-1])).tolist() == [-1]


def test_reconstructed_pt_of_each_class():
    res = {"tc": np.array([[0, 1, 0, -1] + [-1] * 12, [2, -1, 0, -1] + [-1] * 12, [3, 0, -1, -1] + [-1] * 12]),
           "t5_t3": np.array([[0, 1]]), "t3_k": np.array([0.01, -0.012], np.float32)}
    pt = reconstructed_pt(res, {"pt": np.array([3.0, 7.0], np.float32)})
    assert pt[0] == 7.0 and pt[2] == 3.0
    assert abs(pt[1] - 1.0 / (0.011 * 100.0 / (0.3 * 3.8))) < 1e-6   # R = 1 / mean|k| = pT * 87.72 cm


def test_c4_candidates_are_efficient_and_clean(oracle_mod):
    geom, off, tgt = make_config_geometry("C4")
    ev = make_config_event("C4")
    r = oracle_mod.run_event(geom.subdet, off, tgt, ev.x, ev.y, ev.z, ev.sensor, ev.pls)
    m = track_candidate_metrics(r, ev)
    assert m["n_sim_prompt"] == 500 and m["n_sim_displaced"] == 50 and m["n_tc"] == len(r["tc"])
    assert m["efficiency"] > 0.95                      # every prompt track above 0.8 GeV has a seed here
    assert m["fake_rate"] < 0.15                       # ~ the 10 % fake seeds, which come out as unlinked pLS
    assert m["duplicate_rate"] < 0.02                  # CUTS.md section 8 removes duplicates
    ot = track_candidate_metrics(r, ev, classes=(0, 1, 2))
    assert ot["efficiency"] > 0.75 and ot["fake_rate"] < 0.05  # candidates with outer-tracker hits only
    # Fig. 3 right in form: efficiency against r_vertex (= d0 of the displaced helices); the beam-line pointing
    # windows of the stand-in MD / LS cuts lose tracks beyond a few cm, T5-only candidates recover some
    # displaced tracks without a seed
    assert sum(n for n, _ in m["efficiency_vs_rvtx"]) == 550
    assert m["efficiency_vs_rvtx"][0][1] > 0.95 and m["efficiency_displaced"] > 0.15
    t5 = track_candidate_metrics(r, ev, classes=(2,))
    assert t5["n_tc"] >= 1 and t5["efficiency"] == 0.0 and t5["efficiency_displaced"] > 0.0
    # Fig. 4 in form: one row per reconstructed-pT bin, the counts add up to the candidates
    assert sum(n for n, _ in m["fake_rate_vs_pt"]) <= m["n_tc"]
    mm = merge_metrics([m, m])
    assert mm["n_tc"] == 2 * m["n_tc"] and abs(mm["efficiency"] - m["efficiency"]) < 1e-12
    assert mm["efficiency_vs_pt"][0][0] == 2 * m["efficiency_vs_pt"][0][0]
