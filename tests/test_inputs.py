"""The seeded input generators (lst_inputs): shapes, determinism, and the BASELINE.json recipes."""
import numpy as np

from lst_inputs import build_connection_map, make_config_event, make_config_geometry, make_geometry
from lst_inputs.events import concat_events


def test_geometry_sizes_follow_the_configs():
    g = make_geometry("barrel_z60")
    assert g.barrel_nphi.tolist() == [15, 23, 33, 43, 56, 68]  # ceil(2 pi r / 10 cm)
    assert g.n_modules == 238 * 12 == 2856
    g = make_geometry("barrel_z120_endcap")
    assert g.n_modules == 238 * 24 + 10 * int(g.endcap_nphi.sum()) == 9512
    assert (g.subdet == 0).sum() == 5712 and (g.subdet == 1).sum() == 3800


def test_connection_map_is_valid_csr_and_layer_forward():
    for cfg in ("C1", "C3"):
        g, off, tgt = make_config_geometry(cfg)
        assert off[0] == 0 and off[-1] == len(tgt) and np.all(np.diff(off) >= 0)
        assert tgt.min() >= 0 and tgt.max() < g.n_modules
        src = np.repeat(np.arange(g.n_modules), np.diff(off))
        bb = (g.subdet[src] == 0) & (g.subdet[tgt] == 0)
        assert np.all(g.layer[tgt][bb] == g.layer[src][bb] + 1)  # barrel -> next barrel layer only
        ee = (g.subdet[src] == 1) & (g.subdet[tgt] == 1)
        assert np.all(g.side[tgt][ee] == g.side[src][ee]) and np.all(g.layer[tgt][ee] == g.layer[src][ee] + 1)
        assert not np.any((g.subdet[src] == 1) & (g.subdet[tgt] == 0))  # never endcap -> barrel
        for m in (0, g.n_modules // 2):
            row = tgt[off[m]:off[m + 1]]
            assert np.all(np.diff(row) > 0)  # sorted, unique


def test_connection_map_deterministic_without_cache():
    g = make_geometry("barrel_z60")
    a = build_connection_map(g, n_samples=20000, seed=5, cache=False)
    b = build_connection_map(g, n_samples=20000, seed=5, cache=False)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])


def test_events_are_seeded_and_shaped_like_the_configs():
    e1 = make_config_event("C1")
    e1b = make_config_event("C1")
    assert np.array_equal(e1.x, e1b.x) and np.array_equal(e1.sensor, e1b.sensor)
    assert e1.x.dtype == np.float32 and e1.sensor.dtype == np.int32
    assert 150 < e1.n_hits < 260 and np.all(e1.truth >= 0) and e1.n_pls == 0
    e2 = make_config_event("C2")
    assert 6000 < e2.n_hits < 7500 and (e2.truth < 0).sum() == 2000
    e4 = make_config_event("C4")
    assert 500 < e4.n_pls < 650 and (e4.pls["truth"] < 0).sum() > 30 and len(e4.trk["pt"]) == 550
    g, _, _ = make_config_geometry("C1")
    assert e2.sensor.min() >= 0 and e2.sensor.max() < g.n_sensors


def test_hits_lie_on_their_sensor_surfaces():
    g, _, _ = make_config_geometry("C3")
    ev = make_config_event("C3")
    assert 0.9e5 < ev.n_hits < 1.6e5
    m = ev.sensor // 2
    s = ev.sensor % 2
    r = np.hypot(ev.x.astype(np.float64), ev.y.astype(np.float64))
    bar = g.subdet[m] == 0
    from lst_inputs.geometry import BARREL_R, ENDCAP_Z
    assert np.allclose(r[bar], BARREL_R[g.layer[m[bar]] - 1] + 0.26 * s[bar], atol=1e-4)
    end = ~bar
    assert np.allclose(np.abs(ev.z[end]), ENDCAP_Z[g.layer[m[end]] - 1] + 0.4 * s[end], atol=1e-4)
    assert np.all(np.sign(ev.z[end]) == g.side[m[end]])


def test_concat_events_offsets():
    evs = [make_config_event("C5", pu=50, index=i, seeds=True) for i in range(3)]
    b = concat_events(evs)
    assert b["hit_offsets"].tolist() == np.concatenate([[0], np.cumsum([e.n_hits for e in evs])]).tolist()
    assert b["pls_offsets"][-1] == sum(e.n_pls for e in evs) == len(b["pls"]["pt"])
    assert len(b["x"]) == b["hit_offsets"][-1]


def test_strip_like_sensors_quantise_z_and_r():
    """SURVEY.md 8(f)2 / PAPER.md:23, Fig. 1: on the three outer barrel layers a hit sits on the centre of a 5 cm
    strip, on the outer endcap rings on the centre of one of two strip rows; the inner layers keep their resolution.
    Same tracks, same hit count and module assignment as the pixel-like event of the same seed."""
    from lst_inputs.configs import STRIP_PITCH
    from lst_inputs.geometry import ENDCAP_NRINGS, ENDCAP_RMAX, ENDCAP_RMIN

    geom, off, tgt = make_config_geometry("C6")
    a = make_config_event("C5", pu=50, index=1, seeds=True)
    b = make_config_event("C6", pu=50, index=1, seeds=True)
    assert a.n_hits == b.n_hits and np.array_equal(a.sensor, b.sensor) and np.array_equal(a.truth, b.truth)
    m = b.sensor // 2
    bar = geom.subdet[m] == 0
    outer = bar & (geom.layer[m] >= 4)
    zq = b.z[outer] / STRIP_PITCH - 0.5
    assert outer.sum() > 1000 and np.allclose(zq, np.round(zq), atol=1e-4)
    inner = bar & (geom.layer[m] <= 3)
    assert np.array_equal(b.z[inner], a.z[inner]) and np.array_equal(b.x[bar], a.x[bar])
    zi = b.z[inner] / STRIP_PITCH - 0.5
    assert np.mean(np.abs(zi - np.round(zi)) < 1e-3) < 0.01
    end = ~bar
    w = (ENDCAP_RMAX - ENDCAP_RMIN) / ENDCAP_NRINGS
    r = np.hypot(b.x[end].astype(np.float64), b.y[end].astype(np.float64))
    far = r > 62.0
    rq = (r[far] - ENDCAP_RMIN) / (0.5 * w) - 0.5
    assert far.sum() > 100 and np.allclose(rq, np.round(rq), atol=2e-3)
    assert np.abs(np.hypot(a.x[end], a.y[end]) - np.hypot(b.x[end], b.y[end])).max() < 0.5 * w + 1e-3


def test_extension_inputs():
    """the skip-layer connection map holds the plain one; the committed perceptron weights
    have the layout of CUTS.md section 11."""
    from lst_inputs.t5_mlp import T5_MLP, T5_MLP_SCALE, T5_MLP_THR

    assert len(T5_MLP) == 65 and T5_MLP_SCALE == 100.0 and T5_MLP_THR == 1.0 and np.all(np.isfinite(T5_MLP))
    g, off, tgt = make_config_geometry("C4")
    g7, off7, tgt7 = make_config_geometry("C7")
    assert g7.n_modules == g.n_modules and len(tgt7) > 2 * len(tgt)
    for m in (0, 500, 2000):
        assert set(tgt[off[m]:off[m + 1]]) <= set(tgt7[off7[m]:off7[m + 1]])
    src = np.repeat(np.arange(g7.n_modules), np.diff(off7))
    dl = g7.layer[tgt7] - g7.layer[src]
    assert set(np.unique(dl)) == {1, 2}        # next layer and the one after it
