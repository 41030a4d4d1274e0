"""Audit of the approximate cut cascades (lst_ctx_audit, csrc/lst_audit.cuh).

MD, LS and the seed linking decide most candidates with cheaper arithmetic inside hand-derived error bands; the
parity tests show that this changes nothing on the events the oracle can afford (about 2e8 candidates per PU200
batch, half a second of 16 host threads).  A band that is too tight by a factor of two would lose about one
object per 1e9 candidates -- out of the oracle's reach.  The audit re-evaluates every candidate with the exact
cuts ON THE GPU (milliseconds per batch), so it can cover many more events:

  * first the audit's own numbers are pinned to the oracle on batches the oracle runs (candidates, accepted and
    near-threshold candidates per stage are the oracle's n_tests, object counts and near): the brute-force kernels
    count the right things and do not depend on the chain's pre-filters;
  * then >= 2e9 candidates of PU 50 ... 250, the strip-like workload, the skip-layer map and the dense and
    on-threshold events go through chain + audit: not one comparison may differ.
"""
import numpy as np
import pytest

from lst_inputs import c5_batch, make_config_event, make_config_geometry

from .util import run_batch

pytestmark = pytest.mark.gpu

KEYS = ("md_hits", "ls_md", "pt3", "pt5")
STAGE = (0, 1, 4, 5)  # MD, LS, pT3, pT5 in near[] / n_tests[]


@pytest.fixture(scope="module")
def lst():
    import torch

    assert torch.cuda.is_available()
    from paper_2407_18231_b200 import build

    build.build()
    import paper_2407_18231_b200 as m

    return m


def audited(lst, ctx, events, what):
    run_batch(lst, ctx, events)
    rep = lst.lst_ctx_audit(ctx)
    assert rep["mismatches"] == 0, f"{what}: a pre-filter decision differs from the exact cuts: {rep}"
    assert rep["hash_exact"] == rep["hash_chain"] and rep["accepted"] == rep["chain_objects"]
    assert rep["near"] == rep["chain_near"] and rep["candidates"] == rep["chain_candidates"]
    return rep


def test_audit_numbers_are_the_oracles(lst, oracle_mod):
    """Mixed batch (C4 with displaced tracks, an empty event, two PU100 events): every audit number against the oracle."""
    from lst_inputs.events import Event

    geom, off, tgt = make_config_geometry("C5")
    empty = Event(x=np.zeros(0, np.float32), y=np.zeros(0, np.float32), z=np.zeros(0, np.float32),
                  sensor=np.zeros(0, np.int32), truth=np.zeros(0, np.int32))
    evs = [make_config_event("C4"), empty] + c5_batch(pu=100, n_events=2, first=40)
    g = lst.lst_load_geometry(geom.module_table(), off, tgt)
    ctx = lst.lst_ctx_create(g, lst.lst_default_caps(max_events=len(evs)))
    try:
        rep = audited(lst, ctx, evs, "mixed batch")
        want = [oracle_mod.run_event(geom.subdet, off, tgt, ev.x, ev.y, ev.z, ev.sensor, ev.pls) for ev in evs]
        for s, (key, st) in enumerate(zip(KEYS, STAGE)):
            assert rep["accepted"][s] == sum(len(w[key]) for w in want), key
            assert rep["candidates"][s] == sum(int(w["n_tests"][st]) for w in want), key
            assert rep["near"][s] == sum(int(w["near"][st]) for w in want), key
            assert rep["candidates"][s] > 0 and rep["accepted"][s] > 0
    finally:
        lst.lst_free(ctx)
        lst.lst_free(g)


def test_two_billion_candidates_without_a_wrong_decision(lst):
    total = np.zeros(4, np.int64)
    near = np.zeros(4, np.int64)
    geom, off, tgt = make_config_geometry("C5")
    g = lst.lst_load_geometry(geom.module_table(), off, tgt)
    ctx = lst.lst_ctx_create(g, lst.lst_default_caps(max_events=16))
    try:
        plan = [(200, 2000 + 16 * b) for b in range(10)] + [(50, 3000), (100, 3100), (140, 3200), (250, 3300), (250, 3400)]
        for pu, first in plan:
            rep = audited(lst, ctx, c5_batch(pu=pu, n_events=16, first=first), f"C5 PU{pu} events {first}..")
            total += rep["candidates"]
            near += rep["near"]
    finally:
        lst.lst_free(ctx)
        lst.lst_free(g)
    # the strip-like workload (wider r-z windows: other parts of the bands are exercised)
    from lst_inputs.configs import C6_PARAMS

    geom, off, tgt = make_config_geometry("C6")
    g = lst.lst_load_geometry(geom.module_table(), off, tgt, lst.lst_default_params(**C6_PARAMS))
    ctx = lst.lst_ctx_create(g, lst.lst_default_caps(max_events=16))
    try:
        for first in (0, 16):
            rep = audited(lst, ctx, c5_batch(pu=200, n_events=16, first=first, config="C6"), f"C6 PU200 {first}..")
            total += rep["candidates"]
            near += rep["near"]
    finally:
        lst.lst_free(ctx)
        lst.lst_free(g)
    # skip-layer connection map, 15 % hit inefficiency, T4 on (rows of up to 63 targets)
    geom, off, tgt = make_config_geometry("C7")
    g = lst.lst_load_geometry(geom.module_table(), off, tgt, lst.lst_default_params(stage_mask=0x7F))
    ctx = lst.lst_ctx_create(g, lst.lst_default_caps(max_events=3))
    try:
        rep = audited(lst, ctx, [make_config_event("C7"), make_config_event("C4"), make_config_event("C2")], "C7")
        total += rep["candidates"]
    finally:
        lst.lst_free(ctx)
        lst.lst_free(g)
    print("audited candidates (MD, LS, pT3, pT5):", total.tolist(), "near-threshold among them:", near.tolist())
    assert total.sum() >= 2_000_000_000 and np.all(total > 0) and np.all(near > 0)


def test_dense_and_on_threshold_events(lst):
    """The corners of the other GPU tests: thousands of MDs per module, straight high-pT tracks with seeds whose
    |kp| sits on tolk, and cut constants tuned onto a candidate -- the audit must agree there too."""
    from .test_gpu_engine import dense_chain_event
    from .test_gpu_near import straight_dense_event

    for name, make, kws in (("dense chain", dense_chain_event, ({},)),
                            ("straight tracks, |kp| on tolk", straight_dense_event, ({}, {"near_rel": 0.0}))):
        table, off, tgt, x, y, z, s, pls = make()
        for kw in kws:
            g = lst.lst_load_geometry(table, off, tgt, lst.lst_default_params(**kw))
            ctx = lst.lst_ctx_create(g, lst.lst_default_caps(max_events=1))
            try:
                h, keep = lst.make_hits(x, y, z, s)
                sd, keep = lst.make_pls(pls, keep=keep)
                lst.lst_ctx_run(ctx, 1, h, sd)
                lst.lst_ctx_sync(ctx)
                rep = lst.lst_ctx_audit(ctx)
                assert rep["mismatches"] == 0, f"{name} {kw}: {rep}"
                assert rep["accepted"][0] > 400 and rep["candidates"][2] > 0 and rep["accepted"] == rep["chain_objects"]
            finally:
                lst.lst_free(ctx)
                lst.lst_free(g)
