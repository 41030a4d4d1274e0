"""GPU parity at the thresholds: candidates placed ON a cut (within a few ulp), seeds in the pT band where
the curvature pre-filter of the seed linking has no slack, NaN / Inf coordinates, and the per-event
counters returned through the C ABI (CUTS.md section 0).

Natural events put a handful of candidates per million inside the near-threshold window, so the flags
are exercised here on purpose: for every cut of every stage one cut CONSTANT is tuned (it is an input:
lst_params) so that the cut value of a chosen candidate of a real event equals the threshold, then moved
by -2 ... +2 ulp.  The oracle (tests only) and the CUDA path get the same constants; objects and both
counters must agree, and near[stage] must be > 0.
"""
import numpy as np
import pytest

from lst_inputs import make_config_event, make_config_geometry

from .util import assert_same, canon, run_batch

pytestmark = pytest.mark.gpu

F = np.float32


@pytest.fixture(scope="module")
def lst():
    import torch

    assert torch.cuda.is_available()
    from paper_2407_18231_b200 import build

    build.build()
    import paper_2407_18231_b200 as m

    return m


def _ulps(x, k):
    x = F(x)
    for _ in range(abs(k)):
        x = np.nextafter(x, F(np.inf) if k > 0 else F(-np.inf), dtype=F)
    return float(x)


def _r_min():
    kr = F(100.0) / (F(0.3) * F(3.8))
    return F(0.8) * kr


def tuned_constants(O, geom, ev, base):
    """(stage, parameter, value) triples: `value` puts the named cut of one accepted object of `base`
    (the oracle's result with default constants) at its threshold.  Uses the oracle's single-candidate
    functions only to read the cut values of that object."""
    sub = geom.subdet
    mdf, mdm = base["md_f"], base["md_module"]
    out = []
    # MD (barrel): lim = (ra dd)(ra INV_2RMIN + MD_B_PHI_TOL); zl = Z0_MAX (rb - ra) + MD_Z_TOL ra
    k = int(np.nonzero(sub[mdm] == 0)[0][7])
    a, b = base["md_hits"][k]
    lo, hi = (ev.x[a], ev.y[a], ev.z[a]), (ev.x[b], ev.y[b], ev.z[b])
    v = O.md_test(lo, hi, False)[2]
    ra = float(np.hypot(F(lo[0]), F(lo[1])))
    rb = float(np.hypot(F(hi[0]), F(hi[1])))
    out.append((0, "md_b_phi_tol", abs(float(v["crs"])) / (ra * float(v["dd"])) - ra * (1.0 / (2.0 * float(_r_min())))))
    out.append((0, "md_z_tol", (float(v["zv"]) - 15.0 * (rb - ra)) / ra))
    # LS: kv <= LS_KAPPA_MAX; zl = Z0_MAX (rho - 1) + LS_Z_TOL; dA <= LS_DIR_TOL
    A, B = base["ls_md"][11]
    v = O.ls_test(mdf[A], sub[mdm[A]] != 0, mdf[B], sub[mdm[B]] != 0)[2]
    out.append((1, "ls_kappa_max", float(v["kv"])))
    if not (sub[mdm[A]] or sub[mdm[B]]):
        out.append((1, "ls_z_tol", float(v["zv"]) - 15.0 * (float(v["rho"]) - 1.0)))
        out.append((1, "ls_dir_tol", float(v["dA"])))
    # T3: kv = |k3| R_MIN <= T3_KAPPA_MAX; tol = T3_Z_TOL0 + T3_Z_TOL1 ratio
    t = base["t3_md"][5]
    e = [sub[mdm[m]] != 0 for m in t]
    v = O.t3_test(mdf[t[0]][:4], e[0], mdf[t[1]][:4], e[1], mdf[t[2]][:4], e[2])[2]
    out.append((2, "t3_kappa_max", float(F(abs(v["k3"])) * _r_min())))
    if not any(e):
        out.append((2, "t3_z_tol0", float(v["zv"]) - 0.6 * float(v["ratio"])))
    # T5: tol = T5_TOL0 + T5_TOL1 max(|ki|, |ko|) against |ki - kb|
    t1, t2 = base["t5_t3"][3]
    m = base["t5_md"][3]
    ki, ko = base["t3_k"][t1], base["t3_k"][t2]
    v = O.t5_test(ki, ko, mdf[m[1]][:2], mdf[m[2]][:2], mdf[m[3]][:2])[2]
    out.append((3, "t5_tol0", abs(float(ki) - float(v["kb"])) - 0.05 * max(abs(float(ki)), abs(float(ko)))))
    # pT3: gate, dp, r-z at A
    p, t = base["pt3"][9]
    pls = [ev.pls[k][p] for k in ("pt", "q", "x0", "y0", "z0", "x1", "y1", "z1")]
    m = base["t3_md"][t]
    eA, eL = sub[mdm[m[0]]] != 0, sub[mdm[m[2]]] != 0
    v = O.pt_test(pls, mdf[m[0]][:4], eA, mdf[m[2]][:4], eL, [base["t3_k"][t]])[2]
    lw = float(np.hypot(F(mdf[m[0]][0]) - F(pls[5]), F(mdf[m[0]][1]) - F(pls[6])))
    lv = float(np.hypot(F(pls[5]) - F(pls[2]), F(pls[6]) - F(pls[3])))
    out.append((4, "pt_gate_tol", float(v["gcrs"]) / (lv * lw) - lw * (1.0 / (2.0 * float(_r_min())))))
    out.append((4, "pt_k_tol0", abs(float(v["kx"]) - float(v["kp"])) - 0.1 * abs(float(v["kp"]))))
    if not eA:
        out.append((4, "pt_z_tol", float(v["zqA"])))
    # pT5: |kx - ko| against tolk
    p, t = base["pt5"][4]
    pls = [ev.pls[k][p] for k in ("pt", "q", "x0", "y0", "z0", "x1", "y1", "z1")]
    m = base["t5_md"][t]
    kt = [base["t3_k"][base["t5_t3"][t][0]], base["t3_k"][base["t5_t3"][t][1]]]
    v = O.pt_test(pls, mdf[m[0]][:4], sub[mdm[m[0]]] != 0, mdf[m[4]][:4], sub[mdm[m[4]]] != 0, kt, base["t5_score"][t])[2]
    out.append((5, "pt_k_tol0", abs(float(v["kx"]) - float(kt[1])) - 0.1 * abs(float(v["kp"]))))
    return out


def test_cut_constants_tuned_onto_candidates(lst, oracle_mod):
    O = oracle_mod
    geom, off, tgt = make_config_geometry("C4")
    ev = make_config_event("C4")
    base = O.run_event(geom.subdet, off, tgt, ev.x, ev.y, ev.z, ev.sensor, ev.pls)
    flagged = set()
    for stage, name, value in tuned_constants(O, geom, ev, base):
        decisions = []
        for du in (-2, -1, 0, 1, 2):
            val = _ulps(value, du)
            want = O.run_event(geom.subdet, off, tgt, ev.x, ev.y, ev.z, ev.sensor, ev.pls, O.default_params(**{name: val}))
            g = lst.lst_load_geometry(geom.module_table(), off, tgt, lst.lst_default_params(**{name: val}))
            try:
                got = lst.lst_run_event(g, ev.x, ev.y, ev.z, ev.sensor, ev.pls)
            finally:
                lst.lst_free(g)
            assert_same(canon(got), canon(want), f"{name} = {val!r} ({du:+d} ulp): ")
            assert want["near"][stage] >= 1, f"{name}: the tuned candidate is not flagged ({want['near']})"
            decisions.append(len(want[("md_hits", "ls_md", "t3_md", "t5_md", "pt3", "pt5")[stage]]))
        flagged.add(stage)
        assert decisions == sorted(decisions), f"{name}: counts not monotone in the constant: {decisions}"
    assert flagged == {0, 1, 2, 3, 4, 5}


def test_narrower_near_windows(lst, oracle_mod):
    """near_rel is an input (lst_params, CUTS.md section 0).  The kernels' pre-filters hand every candidate within
    1e-5 of a threshold to the exact cut, so any window up to that is counted exactly as the oracle counts it --
    here 0 (only v == t is flagged) and 2.5e-6, with a constant tuned onto a candidate and one ulp to either side;
    a wider window is refused (LST_ERR_ARG, include/lst.h)."""
    O = oracle_mod
    geom, off, tgt = make_config_geometry("C4")
    ev = make_config_event("C4")
    base = O.run_event(geom.subdet, off, tgt, ev.x, ev.y, ev.z, ev.sensor, ev.pls)
    seen = np.zeros((2, 7), np.int64)
    for stage, name, value in tuned_constants(O, geom, ev, base):
        for j, rel in enumerate((0.0, 2.5e-6)):
            for du in (-1, 0, 1):
                kw = {name: _ulps(value, du), "near_rel": rel}
                want = O.run_event(geom.subdet, off, tgt, ev.x, ev.y, ev.z, ev.sensor, ev.pls, O.default_params(**kw))
                g = lst.lst_load_geometry(geom.module_table(), off, tgt, lst.lst_default_params(**kw))
                try:
                    got = lst.lst_run_event(g, ev.x, ev.y, ev.z, ev.sensor, ev.pls)
                finally:
                    lst.lst_free(g)
                assert_same(canon(got), canon(want), f"near_rel = {rel}, {name} {du:+d} ulp: ")
                seen[j] += want["near"]
    assert np.all(seen[1][:6] > 0), seen          # the narrow window still flags the tuned candidates
    assert np.all(seen[0] <= seen[1]) and seen[0].sum() > 0, seen   # v == t exactly happens at 0 ulp
    with pytest.raises(lst.LstError) as e:
        lst.lst_load_geometry(geom.module_table(), off, tgt, lst.lst_default_params(near_rel=1e-4))
    assert e.value.status == lst.LST_ERR_ARG


def straight_dense_event(n_trk=90, seed=11):
    """Near-parallel straight tracks through a chain of five barrel modules (thousands of T3s / T5s whose
    circle through a seed has |kx| ~ 1e-6 ... 1e-5), with 40 seeds per track direction whose pT scans
    20.2 ... 20.6 GeV: |kp| - tolk passes through zero inside that band (CUTS.md section 7)."""
    rng = np.random.default_rng(seed)
    phi = np.arange(n_trk) * 0.0007 + 0.3
    z0, cot = rng.normal(0, 2, n_trk), rng.normal(0, 0.2, n_trk)
    xs, ys, zs, ss = [], [], [], []
    for m, r in enumerate((23.0, 36.0, 51.0, 68.0, 88.0)):
        for s, rr in enumerate((r, r + 0.26)):
            ph = phi + rng.normal(0, 0.003, n_trk) / rr
            xs.append(rr * np.cos(ph)); ys.append(rr * np.sin(ph))
            zs.append(z0 + cot * rr + rng.normal(0, 0.1, n_trk)); ss.append(np.full(n_trk, 2 * m + s))
    perm = rng.permutation(n_trk * 10)
    f = lambda a, t: np.concatenate(a).astype(t)[perm]
    k = np.repeat(np.arange(0, n_trk, 6), 30)
    pls = {"pt": rng.uniform(20.2, 20.6, k.size), "q": np.where(rng.random(k.size) < 0.5, 1, -1)}
    for name, r in (("0", 3.0), ("1", 7.0)):
        ph = phi[k] + rng.normal(0, 0.0005, k.size)
        pls["x" + name], pls["y" + name] = r * np.cos(ph), r * np.sin(ph)
        pls["z" + name] = z0[k] + cot[k] * r
    pls = {key: np.ascontiguousarray(v, dtype=np.int32 if key == "q" else np.float32) for key, v in pls.items()}
    table = np.array([[0, m + 1, 0, 0] for m in range(5)], np.int32)
    return table, np.array([0, 1, 2, 3, 4, 4], np.int32), np.array([1, 2, 3, 4], np.int32), \
        f(xs, np.float32), f(ys, np.float32), f(zs, np.float32), f(ss, np.int32), pls


def test_seeds_where_kp_equals_tolk(lst, oracle_mod):
    """Seeds of pT 20.2-20.6 GeV on straight candidates: |kp| - tolk ~ 0, so a candidate with |kx| just
    below it fails the curvature match NEAR its threshold.  The pre-filter's margin must be relative to
    tolk there (round 1 took it relative to |kp| - tolk and lost such candidates from near[4], near[5])."""
    table, off, tgt, x, y, z, s, pls = straight_dense_event()
    want = oracle_mod.run_event(table[:, 0].copy(), off, tgt, x, y, z, s, pls)
    assert want["near"][4] >= 3 and want["near"][5] >= 1, want["near"]
    g = lst.lst_load_geometry(table, off, tgt)
    try:
        got = lst.lst_run_event(g, x, y, z, s, pls)
    finally:
        lst.lst_free(g)
    assert_same(canon(got), canon(want), "pT 20.4 GeV seeds: ")


def test_nan_and_inf_coordinates(lst, oracle_mod):
    """CUTS.md section 0: a comparison with a NaN is false -> the candidate is rejected and never flagged.
    Hits and seeds with NaN / +-Inf coordinates must neither be accepted nor disturb their neighbours."""
    geom, off, tgt = make_config_geometry("C4")
    ev = make_config_event("C4")
    rng = np.random.default_rng(3)
    x, y, z = ev.x.copy(), ev.y.copy(), ev.z.copy()
    bad = rng.choice(ev.n_hits, 600, replace=False)
    for k, val in enumerate((np.nan, np.inf, -np.inf)):
        x[bad[k * 100:(k + 1) * 100]] = val
        z[bad[300 + k * 100:300 + (k + 1) * 100]] = val
    pls = {k: v.copy() for k, v in ev.pls.items()}
    pb = rng.choice(ev.n_pls, 40, replace=False)
    pls["pt"][pb[:10]] = np.nan
    pls["x1"][pb[10:20]] = np.inf
    pls["z0"][pb[20:30]] = -np.inf
    pls["pt"][pb[30:40]] = 0.0
    want = oracle_mod.run_event(geom.subdet, off, tgt, x, y, z, ev.sensor, pls)
    g = lst.lst_load_geometry(geom.module_table(), off, tgt)
    try:
        got = lst.lst_run_event(g, x, y, z, ev.sensor, pls)
    finally:
        lst.lst_free(g)
    assert len(want["t5_md"]) > 100 and len(want["pt3"]) > 100
    used = set(want["md_hits"].ravel().tolist())
    assert not (used & set(bad[:100].tolist()) | used & set(bad[300:400].tolist()))  # no object holds a NaN hit
    # (an upper hit at x = +Inf IS accepted by the cuts as written: Inf <= Inf holds; both sides must agree on that too)
    assert_same(canon(got), canon(want), "NaN / Inf inputs: ")


def test_per_event_counters_through_the_abi(lst, oracle_mod):
    """lst_ctx_fetch_event returns the counters of THAT event (include/lst.h); the batch summary holds their sums."""
    geom, off, tgt = make_config_geometry("C4")
    from lst_inputs.events import Event

    empty = Event(x=np.zeros(0, np.float32), y=np.zeros(0, np.float32), z=np.zeros(0, np.float32),
                  sensor=np.zeros(0, np.int32), truth=np.zeros(0, np.int32))
    evs = [make_config_event("C4"), empty, make_config_event("C2"), make_config_event("C1")]
    g = lst.lst_load_geometry(geom.module_table(), off, tgt)
    ctx = lst.lst_ctx_create(g, lst.lst_default_caps(max_events=4))
    try:
        summ = run_batch(lst, ctx, evs)
        near, tests = np.zeros(7, np.int64), np.zeros(7, np.int64)
        for i, ev in enumerate(evs):
            want = oracle_mod.run_event(geom.subdet, off, tgt, ev.x, ev.y, ev.z, ev.sensor, ev.pls)
            got = lst.lst_ctx_fetch_event(ctx, i)
            assert np.array_equal(got["n_tests"], want["n_tests"]), (i, got["n_tests"], want["n_tests"])
            assert np.array_equal(got["near"], want["near"]), (i, got["near"], want["near"])
            near += want["near"]
            tests += want["n_tests"]
        assert summ["near"] == near.tolist() and summ["n_tests"] == tests.tolist()
        assert tests[0] > 0 and tests[4] > 0
    finally:
        lst.lst_free(ctx)
        lst.lst_free(g)
    with pytest.raises(lst.LstError) as ei:   # include/lst.h: LST_MAX_MD
        g = lst.lst_load_geometry(geom.module_table(), off, tgt)
        try:
            lst.lst_ctx_create(g, lst.lst_default_caps(max_events=1, max_md=(1 << 27) + 1))
        finally:
            lst.lst_free(g)
    assert ei.value.status == lst.LST_ERR_ARG
