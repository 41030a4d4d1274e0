"""SURVEY.md 8(f)1 on the CUDA path: the synthetic-truth metrics (Figs. 3-4 in form) computed
from the track candidates that come back through the C ABI equal those computed from the oracle's (the
candidate sets are bit-identical, so every rate and every bin must be), and pass the physics sanity bars."""
import numpy as np
import pytest

from lst_inputs import c5_batch, make_config_event, make_config_geometry
from lst_inputs.truth_metrics import merge_metrics, track_candidate_metrics

from .util import run_batch

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def lst():
    import torch

    assert torch.cuda.is_available()
    from paper_2407_18231_b200 import build

    build.build()
    import paper_2407_18231_b200 as m

    return m


def _same(a, b):
    assert a.keys() == b.keys()
    for k in a:
        assert np.array_equal(np.asarray(a[k], dtype=float), np.asarray(b[k], dtype=float), equal_nan=True), k


def test_c4_metrics_from_the_cuda_path(lst, oracle_mod):
    geom, off, tgt = make_config_geometry("C4")
    ev = make_config_event("C4")
    g = lst.lst_load_geometry(geom.module_table(), off, tgt)
    try:
        got = lst.lst_run_event(g, ev.x, ev.y, ev.z, ev.sensor, ev.pls)
    finally:
        lst.lst_free(g)
    want = oracle_mod.run_event(geom.subdet, off, tgt, ev.x, ev.y, ev.z, ev.sensor, ev.pls)
    for classes in ((0, 1, 2, 3), (0, 1, 2), (2,)):
        _same(track_candidate_metrics(got, ev, classes=classes), track_candidate_metrics(want, ev, classes=classes))
    m = track_candidate_metrics(got, ev)
    assert m["efficiency"] > 0.95 and m["fake_rate"] < 0.15 and m["duplicate_rate"] < 0.02


def test_pu200_batch_metrics_from_the_cuda_path(lst, oracle_mod):
    geom, off, tgt = make_config_geometry("C5")
    evs = c5_batch(pu=200, n_events=3)
    g = lst.lst_load_geometry(geom.module_table(), off, tgt)
    ctx = lst.lst_ctx_create(g, lst.lst_default_caps(max_events=3))
    try:
        run_batch(lst, ctx, evs)
        got = [track_candidate_metrics(lst.lst_ctx_fetch_event(ctx, i), ev) for i, ev in enumerate(evs)]
    finally:
        lst.lst_free(ctx)
        lst.lst_free(g)
    want = [track_candidate_metrics(oracle_mod.run_event(geom.subdet, off, tgt, ev.x, ev.y, ev.z, ev.sensor, ev.pls), ev)
            for ev in evs]
    for a, b in zip(got, want):
        _same(a, b)
    m = merge_metrics(got)
    assert m["n_events"] == 3 and m["n_sim_prompt"] > 2500
    assert m["efficiency"] > 0.9 and m["duplicate_rate"] < 0.02
    assert m["fake_rate"] < 0.2          # the 10 % fake seeds come out as unlinked pLS candidates
    assert all(n > 0 for n, _ in m["efficiency_vs_pt"])
