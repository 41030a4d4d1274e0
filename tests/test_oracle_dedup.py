"""Pins of the oracle's duplicate removal / track-candidate selection (CUTS.md section 8).

Hand-made object lists with answers that follow from the written rule by hand (PAPER.md:31-34
class priority pT5 > pT3 > T5 > unlinked pLS; PAPER.md:56 duplicates), plus the rule's stated
consequence (survivors pairwise non-overlapping) checked on a real event.
"""
import numpy as np

from lst_inputs import make_config_event, make_config_geometry

E3 = np.zeros((0, 3), np.int32)
E5 = np.zeros((0, 5), np.int32)
E2 = np.zeros((0, 2), np.int32)
F0 = np.zeros(0, np.float32)


def _md_hits(n):
    # MD i = hits (2i, 2i+1)
    return np.arange(2 * n, dtype=np.int32).reshape(n, 2)


def test_t5_pair_sharing_three_mds_keeps_lower_score(oracle_mod):
    t5 = [[0, 1, 2, 3, 4], [0, 1, 2, 5, 6]]
    k5, k3, kT, linked = oracle_mod.dedup(_md_hits(7), E3, t5, [2.0, 1.0], E2, F0, E2, F0, 0)
    assert kT.tolist() == [False, True]
    # sharing only two MDs: both survive
    t5 = [[0, 1, 2, 3, 4], [0, 1, 7, 5, 6]]
    assert oracle_mod.dedup(_md_hits(8), E3, t5, [2.0, 1.0], E2, F0, E2, F0, 0)[2].tolist() == [True, True]


def test_shared_mds_counted_as_a_set_not_by_position(oracle_mod):
    # second T5 starts one layer later: MDs 1,2,3 are shared at different positions
    t5 = [[0, 1, 2, 3, 4], [1, 2, 3, 5, 6]]
    kT = oracle_mod.dedup(_md_hits(7), E3, t5, [1.0, 2.0], E2, F0, E2, F0, 0)[2]
    assert kT.tolist() == [True, False]


def test_removal_uses_the_unfiltered_set(oracle_mod):
    """Chain A < B < C in score, A~B and B~C overlap but A,C do not: B is removed by A and C by B,
    although B itself is removed (the rule quantifies over the UNFILTERED set)."""
    t5 = [[0, 1, 2, 3, 4], [2, 3, 4, 5, 6], [4, 5, 6, 7, 8]]
    kT = oracle_mod.dedup(_md_hits(9), E3, t5, [1.0, 2.0, 3.0], E2, F0, E2, F0, 0)[2]
    assert kT.tolist() == [True, False, False]


def test_equal_scores_fall_back_to_hit_key(oracle_mod):
    t5 = [[0, 1, 2, 5, 6], [0, 1, 2, 3, 4]]
    kT = oracle_mod.dedup(_md_hits(7), E3, t5, [0.5, 0.5], E2, F0, E2, F0, 0)[2]
    assert kT.tolist() == [False, True]  # (.., MD3 = hits 6,7) < (.., MD5 = hits 10,11)
    # the key is the HIT tuple, not the MD index: give MD 5 smaller hit numbers than MD 3
    mdh = _md_hits(7)
    mdh[5] = [0, 0]
    kT = oracle_mod.dedup(mdh, E3, t5, [0.5, 0.5], E2, F0, E2, F0, 0)[2]
    assert kT.tolist() == [True, False]


def test_pt5_same_seed_and_class_priority(oracle_mod):
    t5 = [[0, 1, 2, 3, 4], [10, 11, 12, 13, 14], [0, 1, 20, 21, 22]]
    t3 = [[0, 1, 30], [40, 41, 42], [12, 13, 43]]
    pt5 = [[7, 0], [7, 1]]            # two pT5 of seed 7: the better one (score 1.0) survives
    pt3 = [[7, 1], [3, 0], [4, 1], [5, 2]]
    k5, k3, kT, linked = oracle_mod.dedup(_md_hits(50), t3, t5, [0.1, 0.1, 0.1], pt3, [0.1, 0.1, 0.1, 0.1],
                                           pt5, [1.0, 2.0], 9)
    assert k5.tolist() == [True, False]
    # pT3 0: seed 7 already in a surviving pT5            -> removed
    # pT3 1: its T3 shares MDs 0,1 with the surviving pT5 -> removed
    # pT3 2: T3 (40,41,42) overlaps nothing               -> kept
    # pT3 3: T3 (12,13,43) overlaps only the REMOVED pT5  -> kept
    assert k3.tolist() == [False, False, True, True]
    # T5 0 is the surviving pT5's own T5 (shares 5), T5 2 shares MDs 0,1 with it -> removed;
    # T5 1 shares MDs 12,13 with the T3 of the surviving pT3 3 -> removed
    assert kT.tolist() == [False, False, False]
    assert np.nonzero(linked)[0].tolist() == [4, 5, 7]


def test_pt3_duplicates(oracle_mod):
    t3 = [[0, 1, 2], [0, 1, 3], [5, 6, 7]]
    pt3 = [[1, 0], [2, 1], [2, 2]]
    k5, k3, kT, linked = oracle_mod.dedup(_md_hits(8), t3, E5, F0, pt3, [3.0, 2.0, 1.0], E2, F0, 4)
    # pT3 0 shares 2 MDs with the better pT3 1; pT3 1 has the same seed as the better pT3 2
    assert k3.tolist() == [False, False, True]
    assert np.nonzero(linked)[0].tolist() == [2]


def test_survivors_do_not_overlap_on_c4(oracle_mod):
    geom, off, tgt = make_config_geometry("C4")
    ev = make_config_event("C4")
    r = oracle_mod.run_event(geom.subdet, off, tgt, ev.x, ev.y, ev.z, ev.sensor, ev.pls)
    k5, k3, kT, linked = oracle_mod.dedup(r["md_hits"], r["t3_md"], r["t5_md"], r["t5_score"], r["pt3"],
                                           r["pt3_score"], r["pt5"], r["pt5_score"], ev.n_pls)
    assert 0 < k5.sum() < len(k5) and 0 < k3.sum() < len(k3) and 0 < kT.sum() < len(kT)
    s5 = [(p, set(r["t5_md"][t])) for p, t in r["pt5"][k5]]
    s3 = [(p, set(r["t3_md"][t])) for p, t in r["pt3"][k3]]
    sT = [set(m) for m in r["t5_md"][kT]]
    for i in range(len(s5)):
        for j in range(i + 1, len(s5)):
            assert s5[i][0] != s5[j][0] and len(s5[i][1] & s5[j][1]) < 3
    for i in range(len(s3)):
        for j in range(i + 1, len(s3)):
            assert s3[i][0] != s3[j][0] and len(s3[i][1] & s3[j][1]) < 2
        assert all(s3[i][0] != p and len(s3[i][1] & m) < 2 for p, m in s5)
    for i in range(len(sT)):
        for j in range(i + 1, len(sT)):
            assert len(sT[i] & sT[j]) < 3
        assert all(len(sT[i] & m) < 2 for _, m in s5) and all(len(sT[i] & m) < 2 for _, m in s3)
    # the best-scoring pT5 can be removed by nothing
    assert k5[np.argmin(r["pt5_score"])]
    # TC list = survivors in class order + unlinked seeds
    tc = r["tc"]
    assert (tc[:, 0] == 0).sum() == k5.sum() and (tc[:, 0] == 1).sum() == k3.sum()
    assert (tc[:, 0] == 2).sum() == kT.sum() and (tc[:, 0] == 3).sum() == ev.n_pls - linked.sum()
