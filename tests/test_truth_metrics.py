"""Synthetic-truth sanity of the track candidates with the paper's metric definitions:
not parity, a physics check that the stand-in cuts build tracks."""
import numpy as np

from lst_inputs import make_config_event, make_config_geometry
from paper_2407_18231_b200.truth_metrics import match_candidates, track_candidate_metrics


def test_matching_rule_is_more_than_75_percent():
    truth = np.array([5, 5, 5, 5, 7, -1, 5, 5, 5, 5], dtype=np.int64)
    tc = -np.ones((3, 16), dtype=np.int64)
    tc[0, 0], tc[0, 4:14] = 2, np.arange(10)          # 8 of 10 hits from track 5 -> matched
    tc[1, 0], tc[1, 4:8] = 2, [0, 1, 2, 4]            # 3 of 4 = 75 %, not MORE than 75 % -> fake
    tc[2, 0], tc[2, 1] = 3, 0                          # pLS-only: matched by its seed
    assert match_candidates(tc, truth, pls_truth=np.array([9])).tolist() == [5, -1, 9]
    assert match_candidates(tc[2:], truth, pls_truth=np.array([-1])).tolist() == [-1]


def test_c4_candidates_are_efficient_and_clean(oracle_mod):
    geom, off, tgt = make_config_geometry("C4")
    ev = make_config_event("C4")
    r = oracle_mod.run_event(geom.subdet, off, tgt, ev.x, ev.y, ev.z, ev.sensor, ev.pls)
    m = track_candidate_metrics(r["tc"], ev.truth, ev.trk, ev.pls["truth"])
    assert m["n_sim_selected"] == 500 and m["n_tc"] == len(r["tc"])
    assert m["efficiency"] > 0.95                      # every prompt track above 0.8 GeV has a seed here
    assert m["fake_rate"] < 0.15                       # ~ the 10 % fake seeds, which come out as unlinked pLS
    assert m["duplicate_rate"] < 0.02                  # CUTS.md section 8 removes duplicates
    ot = track_candidate_metrics(r["tc"][r["tc"][:, 0] < 3], ev.truth, ev.trk, ev.pls["truth"])
    assert ot["efficiency"] > 0.75 and ot["fake_rate"] < 0.05  # candidates with outer-tracker hits only
