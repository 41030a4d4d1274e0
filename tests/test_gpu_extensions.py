"""GPU parity of the extensions of SURVEY.md 8(f)3 and 8(f)4 ("more objects"; "machine
learning methods"): skip-layer connection-map edges, the 4-MD object T4 with its selection rule and track-candidate
class (CUTS.md section 10), and the learned T5 selection (CUTS.md section 11), against the oracle, object by object."""
import numpy as np
import pytest

from lst_inputs import make_config_event, make_config_geometry
from lst_inputs.configs import C7_MASK
from lst_inputs.t5_mlp import T5_MLP, T5_MLP_SCALE, T5_MLP_THR

from .util import assert_same, canon, run_batch

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def lst():
    import torch

    assert torch.cuda.is_available()
    from paper_2407_18231_b200 import build

    build.build()
    import paper_2407_18231_b200 as m

    return m


def test_skip_layer_map_and_t4(lst, oracle_mod):
    """C7: 15 % hit inefficiency, connection map with skip-layer edges, stage mask 0x7f (T4 on)."""
    geom, off, tgt = make_config_geometry("C7")
    plain = make_config_geometry("C4")
    assert len(tgt) > 2 * len(plain[2]) and np.diff(off).max() > np.diff(plain[1]).max()
    ev = make_config_event("C7")
    want = oracle_mod.run_event(geom.subdet, off, tgt, ev.x, ev.y, ev.z, ev.sensor, ev.pls,
                                oracle_mod.default_params(stage_mask=C7_MASK))
    ref = oracle_mod.run_event(plain[0].subdet, plain[1], plain[2], ev.x, ev.y, ev.z, ev.sensor, ev.pls)
    assert len(want["t5_md"]) > 2 * len(ref["t5_md"])          # the skip edges recover T5s across a missing layer
    assert len(want["t4_md"]) > 500 and (want["tc"][:, 0] == 4).sum() >= 1 and want["n_tests"][6] > 0
    g = lst.lst_load_geometry(geom.module_table(), off, tgt, lst.lst_default_params(stage_mask=C7_MASK))
    try:
        got = lst.lst_run_event(g, ev.x, ev.y, ev.z, ev.sensor, ev.pls)
    finally:
        lst.lst_free(g)
    assert_same(canon(got), canon(want), "C7 (skip edges + T4): ")
    assert np.all(np.diff(got["tc"][:, 0]) >= 0)                 # class order pT5, pT3, T5, pLS, T4
    assert np.all(np.diff(got["t4_t3"][:, 0]) >= 0)              # T4s grouped by their first T3


def test_t4_in_a_batch_and_capacity(lst, oracle_mod):
    geom, off, tgt = make_config_geometry("C7")
    evs = [make_config_event("C7"), make_config_event("C4"), make_config_event("C2")]
    g = lst.lst_load_geometry(geom.module_table(), off, tgt, lst.lst_default_params(stage_mask=C7_MASK))
    ctx = lst.lst_ctx_create(g, lst.lst_default_caps(max_events=3))
    try:
        summ = run_batch(lst, ctx, evs)
        n_t4 = 0
        for i, ev in enumerate(evs):
            want = oracle_mod.run_event(geom.subdet, off, tgt, ev.x, ev.y, ev.z, ev.sensor, ev.pls,
                                        oracle_mod.default_params(stage_mask=C7_MASK))
            assert_same(canon(lst.lst_ctx_fetch_event(ctx, i)), canon(want), f"T4 batch event {i}: ")
            n_t4 += len(want["t4_md"])
        assert summ["n_t4"] == n_t4
    finally:
        lst.lst_free(ctx)
    ctx = lst.lst_ctx_create(g, lst.lst_default_caps(max_events=1, max_t4=20))
    try:
        h, keep = lst.make_hits(evs[0].x, evs[0].y, evs[0].z, evs[0].sensor)
        s, keep = lst.make_pls(evs[0].pls, keep=keep)
        lst.lst_ctx_run(ctx, 1, h, s)
        with pytest.raises(lst.LstError) as ei:
            lst.lst_ctx_sync(ctx)
        assert ei.value.status == lst.LST_ERR_CAPACITY
    finally:
        lst.lst_free(ctx)
        lst.lst_free(g)


@pytest.mark.parametrize("cfg,kw", [("C4", {}), ("C5", dict(pu=140, index=3, seeds=True))])
def test_learned_t5_selection(lst, oracle_mod, cfg, kw):
    """Stage-mask bit 7: the perceptron of CUTS.md section 11 with the committed weights replaces the T5 cuts."""
    geom, off, tgt = make_config_geometry(cfg)
    ev = make_config_event(cfg, **kw)
    kwargs = dict(stage_mask=0x3f | 128, t5_mlp=T5_MLP, t5_mlp_scale=T5_MLP_SCALE, t5_mlp_thr=T5_MLP_THR)
    want = oracle_mod.run_event(geom.subdet, off, tgt, ev.x, ev.y, ev.z, ev.sensor, ev.pls, oracle_mod.default_params(**kwargs))
    ref = oracle_mod.run_event(geom.subdet, off, tgt, ev.x, ev.y, ev.z, ev.sensor, ev.pls)
    assert len(want["t5_md"]) > 100 and not np.array_equal(canon(want)["t5"], canon(ref)["t5"])
    g = lst.lst_load_geometry(geom.module_table(), off, tgt, lst.lst_default_params(**kwargs))
    try:
        got = lst.lst_run_event(g, ev.x, ev.y, ev.z, ev.sensor, ev.pls)
    finally:
        lst.lst_free(g)
    assert_same(canon(got), canon(want), f"learned T5 selection on {cfg}: ")


def test_learned_t5_threshold_tuned_onto_a_candidate(lst, oracle_mod):
    """The perceptron's threshold moved onto the output s of one accepted T5 (+-2 ulp): near[T5] > 0 and equal."""
    geom, off, tgt = make_config_geometry("C4")
    ev = make_config_event("C4")
    base = dict(stage_mask=0x3f | 128, t5_mlp=T5_MLP, t5_mlp_scale=T5_MLP_SCALE)
    r = oracle_mod.run_event(geom.subdet, off, tgt, ev.x, ev.y, ev.z, ev.sensor, ev.pls,
                             oracle_mod.default_params(t5_mlp_thr=T5_MLP_THR, **base))
    t1, t2 = r["t5_t3"][7]
    m = r["t5_md"][7]
    s = oracle_mod.t5_test(r["t3_k"][t1], r["t3_k"][t2], r["md_f"][m[1]][:2], r["md_f"][m[2]][:2], r["md_f"][m[3]][:2],
                           oracle_mod.default_params(t5_mlp_thr=T5_MLP_THR, **base))[2]["s"]
    for du in (-2, -1, 0, 1, 2):
        thr = np.float32(s)
        for _ in range(abs(du)):
            thr = np.nextafter(thr, np.float32(np.inf if du > 0 else -np.inf), dtype=np.float32)
        want = oracle_mod.run_event(geom.subdet, off, tgt, ev.x, ev.y, ev.z, ev.sensor, ev.pls,
                                    oracle_mod.default_params(t5_mlp_thr=float(thr), **base))
        assert want["near"][3] >= 1
        g = lst.lst_load_geometry(geom.module_table(), off, tgt, lst.lst_default_params(t5_mlp_thr=float(thr), **base))
        try:
            got = lst.lst_run_event(g, ev.x, ev.y, ev.z, ev.sensor, ev.pls)
        finally:
            lst.lst_free(g)
        assert_same(canon(got), canon(want), f"T5_MLP_THR = s {du:+d} ulp: ")
