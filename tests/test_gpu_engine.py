"""GPU parity, part 2: the MD / LS / seed-linking kernels at their edges (dense modules, stash and
stage overflows, capacities), and the full benchmark configuration (16 PU200 events in one launch sequence, default capacities)."""
import numpy as np
import pytest

from lst_inputs import c5_batch, make_config_event, make_config_geometry

from .util import assert_same, canon, run_batch

pytestmark = pytest.mark.gpu

R_LAYER = (23.0, 36.0, 51.0, 68.0, 88.0)


@pytest.fixture(scope="module")
def lst():
    import torch

    assert torch.cuda.is_available()
    from paper_2407_18231_b200 import build

    build.build()
    import paper_2407_18231_b200 as m

    return m


def dense_chain_event(n_trk=150, dphi=0.0005, seed=5):
    """Five barrel modules in a chain, n_trk near-parallel straight tracks through all of them: every
    module holds n_trk^2 hit pairs, thousands of MDs share a module (upper hits with more MDs than the
    stash holds), and every MD has hundreds of LS candidates (more LSs per warp pass than the stage holds) -- the opposite corner from the sparse PU200 modules."""
    rng = np.random.default_rng(seed)
    phi = np.arange(n_trk) * dphi + 0.3
    z0, cot = rng.normal(0, 2, n_trk), rng.normal(0, 0.2, n_trk)
    xs, ys, zs, ss = [], [], [], []
    for m, r in enumerate(R_LAYER):
        for s, rr in enumerate((r, r + 0.26)):
            ph = phi + rng.normal(0, 0.003, n_trk) / rr
            xs.append(rr * np.cos(ph))
            ys.append(rr * np.sin(ph))
            zs.append(z0 + cot * rr + rng.normal(0, 0.15, n_trk))
            ss.append(np.full(n_trk, 2 * m + s))
    perm = rng.permutation(n_trk * 10)
    f = lambda a, t: np.concatenate(a).astype(t)[perm]
    table = np.array([[0, m + 1, 0, 0] for m in range(5)], np.int32)
    # seeds on every 5th track (straight: very high pT): each sees hundreds of T3s / T5s behind one anchor
    k = np.arange(0, n_trk, 5)
    pls = {"pt": np.full(k.size, 200.0), "q": np.where(k % 2 == 0, 1, -1)}
    for name, r in (("0", 3.0), ("1", 7.0)):
        pls["x" + name], pls["y" + name] = r * np.cos(phi[k]), r * np.sin(phi[k])
        pls["z" + name] = z0[k] + cot[k] * r
    pls = {key: np.ascontiguousarray(v, dtype=np.int32 if key == "q" else np.float32) for key, v in pls.items()}
    return table, np.array([0, 1, 2, 3, 4, 4], np.int32), np.array([1, 2, 3, 4], np.int32), \
        f(xs, np.float32), f(ys, np.float32), f(zs, np.float32), f(ss, np.int32), pls


def test_dense_modules_span_many_chunks(lst, oracle_mod):
    table, off, tgt, x, y, z, s, pls = dense_chain_event()
    g = lst.lst_load_geometry(table, off, tgt)
    try:
        got = lst.lst_run_event(g, x, y, z, s, pls)
    finally:
        lst.lst_free(g)
    want = oracle_mod.run_event(table[:, 0].copy(), off, tgt, x, y, z, s, pls)
    assert want["n_tests"][0] == 5 * 150 * 150 and len(want["ls_md"]) > 10_000 and len(want["t5_md"]) > 5_000
    assert len(want["pt3"]) > 100 and len(want["pt5"]) > 100  # anchors with more candidates than a warp list holds
    assert_same(canon(got), canon(want), "dense chain: ")
    # storage order (what the begin-offset arrays rely on): MDs grouped by module, LSs by inner MD,
    # T3s by first LS, T5s by first T3
    for key, col in (("md_module", None), ("ls_md", 0), ("t3_ls", 0), ("t5_t3", 0)):
        v = got[key] if col is None else got[key][:, col]
        assert np.all(np.diff(v) >= 0), key


@pytest.mark.parametrize("cap", ["max_md", "max_ls", "max_t3", "max_t5", "max_pt3", "max_pt5", "max_tc"])
def test_every_object_capacity_overflow_is_an_error(lst, cap):
    geom, off, tgt = make_config_geometry("C4")
    ev = make_config_event("C4")
    g = lst.lst_load_geometry(geom.module_table(), off, tgt)
    ctx = lst.lst_ctx_create(g, lst.lst_default_caps(max_events=1, **{cap: 20}))
    try:
        h, keep = lst.make_hits(ev.x, ev.y, ev.z, ev.sensor)
        s, keep = lst.make_pls(ev.pls, keep=keep)
        lst.lst_ctx_run(ctx, 1, h, s)
        with pytest.raises(lst.LstError) as ei:
            lst.lst_ctx_sync(ctx)
        assert ei.value.status == lst.LST_ERR_CAPACITY
    finally:
        lst.lst_free(ctx)
        lst.lst_free(g)


def test_hits_on_one_sensor_only(lst, oracle_mod):
    """No module has a hit pair: zero candidate pairs in every stage, every seed comes out unlinked."""
    geom, off, tgt = make_config_geometry("C4")
    ev = make_config_event("C4")
    low = (ev.sensor % 2) == 0
    x, y, z, s = ev.x[low], ev.y[low], ev.z[low], ev.sensor[low]
    g = lst.lst_load_geometry(geom.module_table(), off, tgt)
    try:
        got = lst.lst_run_event(g, x, y, z, s, ev.pls)
    finally:
        lst.lst_free(g)
    want = oracle_mod.run_event(geom.subdet, off, tgt, x, y, z, s, ev.pls)
    assert len(want["md_hits"]) == 0 and len(want["tc"]) == ev.n_pls
    assert_same(canon(got), canon(want), "lower sensors only: ")


def test_many_sensors_span_several_ingest_rounds(lst, oracle_mod):
    """A module table of 8 copies of C4's (45,696 sensors): the ingest kernels keep at most 40,960 sensor counters
    in shared memory and take the sensors in rounds.  Event 0 sits in the first copy, event 1 in the last, event
    2 is spread over all of them (module copy = hit index mod 8: no hit pair survives, which is a result too)."""
    import dataclasses

    geom, off, tgt = make_config_geometry("C4")
    n_mod, copies = geom.n_modules, 8
    table = np.tile(geom.module_table(), (copies, 1))
    subdet = np.tile(geom.subdet, copies)
    deg = np.diff(off)
    off_big = np.concatenate([[0], np.cumsum(np.tile(deg, copies))]).astype(np.int32)
    tgt_big = np.concatenate([tgt + k * n_mod for k in range(copies)]).astype(np.int32)
    ev = make_config_event("C4")
    shifts = [np.zeros(ev.n_hits, np.int32), np.full(ev.n_hits, (copies - 1) * 2 * n_mod, np.int32),
              (np.arange(ev.n_hits, dtype=np.int32) % copies) * 2 * n_mod]
    evs = [dataclasses.replace(ev, sensor=(ev.sensor + sh).astype(np.int32)) for sh in shifts]
    g = lst.lst_load_geometry(table, off_big, tgt_big)
    ctx = lst.lst_ctx_create(g, lst.lst_default_caps(max_events=3))
    # a second, small geometry created afterwards and alive at the same time: per-function launch limits
    # (shared memory of the ingest) must not depend on which context was created last
    g_small = lst.lst_load_geometry(geom.module_table(), off, tgt)
    ctx_small = lst.lst_ctx_create(g_small, lst.lst_default_caps(max_events=1))
    try:
        run_batch(lst, ctx_small, [ev])
        want_small = canon(oracle_mod.run_event(geom.subdet, off, tgt, ev.x, ev.y, ev.z, ev.sensor, ev.pls))
        assert_same(canon(lst.lst_ctx_fetch_event(ctx_small, 0)), want_small, "C4 next to 8 x C4: ")
        run_batch(lst, ctx, evs)
        for i, e in enumerate(evs):
            want = oracle_mod.run_event(subdet, off_big, tgt_big, e.x, e.y, e.z, e.sensor, e.pls)
            assert_same(canon(lst.lst_ctx_fetch_event(ctx, i)), canon(want), f"8 x C4 modules, event {i}: ")
    finally:
        lst.lst_free(ctx_small)
        lst.lst_free(g_small)
        lst.lst_free(ctx)
        lst.lst_free(g)


def test_benchmark_configuration(lst, oracle_mod):
    """BASELINE.json config 5 as bench.py times it: 16 PU200 events (seeds on) in one launch sequence
    on a non-default stream, default capacities, device-resident inputs, two batches back to back on
    the same context.  Every event of the last batch is compared with the oracle, object by object."""
    import torch

    geom, off, tgt = make_config_geometry("C5")
    g = lst.lst_load_geometry(geom.module_table(), off, tgt)
    stream = torch.cuda.Stream()
    ctx = lst.lst_ctx_create(g, lst.lst_default_caps(max_events=16), stream.cuda_stream)
    try:
        from lst_inputs.events import concat_events

        batches = [c5_batch(pu=200, n_events=16, first=0), c5_batch(pu=200, n_events=16, first=16)]
        keepalive = []
        for evs in batches:
            b = concat_events(evs)
            dev = {k: torch.from_numpy(b[k]).cuda() for k in ("x", "y", "z", "sensor")}
            pls = {k: torch.from_numpy(v).cuda() for k, v in b["pls"].items()}
            h, keep = lst.make_hits(dev["x"], dev["y"], dev["z"], dev["sensor"], b["hit_offsets"])
            s, keep = lst.make_pls(pls, b["pls_offsets"], keep)
            keepalive.append((dev, pls, keep))
            torch.cuda.synchronize()
            lst.lst_ctx_run(ctx, 16, h, s)
        summ = lst.lst_ctx_sync(ctx)
        assert summ["n_events"] == 16 and summ["n_hits"] > 16 * 100_000
        tot = np.zeros(7, np.int64)
        tests = np.zeros(7, np.int64)
        near = np.zeros(7, np.int64)
        for i, ev in enumerate(batches[1]):
            want = oracle_mod.run_event(geom.subdet, off, tgt, ev.x, ev.y, ev.z, ev.sensor, ev.pls)
            got = lst.lst_ctx_fetch_event(ctx, i)
            assert_same(canon(got), canon(want), f"bench config, event {i}: ")
            tot += [len(want[k]) for k in ("md_hits", "ls_md", "t3_md", "t5_md", "pt3", "pt5", "tc")]
            tests += want["n_tests"]
            near += want["near"]
        assert [summ["n_" + k] for k in ("md", "ls", "t3", "t5", "pt3", "pt5", "tc")] == tot.tolist()
        assert summ["n_tests"] == tests.tolist() and summ["near"] == near.tolist()
        assert np.all(near <= 1e-4 * tests), "near-threshold candidates above 0.01 % of the stage's candidates (CUTS.md section 0, DESIGN.md N2)"
    finally:
        lst.lst_free(ctx)
        lst.lst_free(g)


def test_randomised_batches(lst, oracle_mod):
    """Many small and odd-sized batches (1-5 events, 1-400 tracks, with and without noise, seeds and
    displaced tracks) on one reused context: every event equals the oracle's.  (compute-sanitizer is
    not available on the GPU pool; this is the race / bounds shake-out.)"""
    from lst_inputs.events import EventSpec, generate_event

    geom, off, tgt = make_config_geometry("C4")
    g = lst.lst_load_geometry(geom.module_table(), off, tgt)
    ctx = lst.lst_ctx_create(g, lst.lst_default_caps(max_events=5))
    rng = np.random.default_rng(2407)
    try:
        for rep in range(8):
            evs = []
            for k in range(int(rng.integers(1, 6))):
                spec = EventSpec(n_tracks=int(rng.integers(1, 400)), pt_dist=("loguniform", 0.8, 20.0), eta_max=1.0,
                                 noise=("count", int(rng.integers(0, 3000))) if rng.random() < 0.7 else None,
                                 inefficiency=0.05 * float(rng.random()), seeds=bool(rng.random() < 0.8),
                                 n_displaced=int(rng.integers(0, 30)))
                evs.append(generate_event(geom, spec, 10_000 + 100 * rep + k))
            if all(e.n_pls == 0 for e in evs):
                evs[0] = make_config_event("C4")
            run_batch(lst, ctx, evs)
            for i, ev in enumerate(evs):
                want = oracle_mod.run_event(geom.subdet, off, tgt, ev.x, ev.y, ev.z, ev.sensor, ev.pls)
                got = lst.lst_ctx_fetch_event(ctx, i)
                assert_same(canon(got), canon(want), f"random batch {rep}, event {i}: ")
    finally:
        lst.lst_free(ctx)
        lst.lst_free(g)


def test_blocks_per_sm_changes_no_result(lst, oracle_mod):
    """lst_ctx_set_blocks_per_sm (include/lst.h): every kernel is a ticket / grid-stride loop, so the grid size
    changes who shares the SMs, never a result.  One context, grids of 1, 2, 3 and 8 blocks per SM in turn
    (the captured launch sequence is rebuilt each time); out-of-range values are argument errors."""
    geom, off, tgt = make_config_geometry("C4")
    g = lst.lst_load_geometry(geom.module_table(), off, tgt)
    ctx = lst.lst_ctx_create(g, lst.lst_default_caps(max_events=3))
    try:
        evs = [make_config_event("C4"), make_config_event("C2"), make_config_event("C4")]
        want = [canon(oracle_mod.run_event(geom.subdet, off, tgt, ev.x, ev.y, ev.z, ev.sensor, ev.pls)) for ev in evs]
        for blocks in (1, 2, 3, 8, 0, 1):
            lst.lst_ctx_set_blocks_per_sm(ctx, blocks)
            for rep in range(2):  # the second run replays the captured graph
                run_batch(lst, ctx, evs)
                for i in range(len(evs)):
                    assert_same(canon(lst.lst_ctx_fetch_event(ctx, i)), want[i], f"{blocks} blocks per SM, event {i}: ")
        for bad in (-1, 9):
            with pytest.raises(lst.LstError):
                lst.lst_ctx_set_blocks_per_sm(ctx, bad)
    finally:
        lst.lst_free(ctx)
        lst.lst_free(g)


def test_contexts_in_flight_share_the_sms(lst, oracle_mod):
    """The configuration of the bench's timed region: several contexts on streams of their own, every kernel at 2
    (then 1) blocks per SM, all batches launched before any is awaited, three rounds back to back -- kernels of
    different batches co-reside on the SMs (and k_ls_place's wait for its scan tiles runs next to other kernels).
    Every event of every batch of every round equals the oracle's."""
    import torch

    geom, off, tgt = make_config_geometry("C5")
    n_ctx, n_ev = 6, 3
    batches = [[make_config_event("C5", pu=50, index=100 + n_ev * c + i, seeds=True) for i in range(n_ev)] for c in range(n_ctx)]
    want = [[canon(oracle_mod.run_event(geom.subdet, off, tgt, ev.x, ev.y, ev.z, ev.sensor, ev.pls)) for ev in b] for b in batches]
    from lst_inputs.events import concat_events

    g = lst.lst_load_geometry(geom.module_table(), off, tgt)
    streams = [torch.cuda.Stream() for _ in range(n_ctx)]
    ctxs = [lst.lst_ctx_create(g, lst.lst_default_caps(max_events=n_ev), st.cuda_stream) for st in streams]
    try:
        inputs = []
        for b in batches:
            cb = concat_events(b)
            h, keep = lst.make_hits(cb["x"], cb["y"], cb["z"], cb["sensor"], cb["hit_offsets"])
            s, keep = lst.make_pls(cb["pls"], cb["pls_offsets"], keep)
            inputs.append((h, s, keep))
        for blocks in (2, 1):
            for c in ctxs:
                lst.lst_ctx_set_blocks_per_sm(c, blocks)
            for rnd in range(3):
                for c in range(n_ctx):  # context c runs batch (c + rnd) mod n_ctx: every workspace sees every batch
                    b = (c + rnd) % n_ctx
                    lst.lst_ctx_run(ctxs[c], n_ev, inputs[b][0], inputs[b][1])
                for c in range(n_ctx):
                    b = (c + rnd) % n_ctx
                    lst.lst_ctx_sync(ctxs[c])
                    for i in range(n_ev):
                        assert_same(canon(lst.lst_ctx_fetch_event(ctxs[c], i)), want[b][i],
                                    f"{blocks} blocks per SM, round {rnd}, context {c}, event {i}: ")
    finally:
        for c in ctxs:
            lst.lst_free(c)
        lst.lst_free(g)


def test_more_pu200_batches_at_small_grids(lst, oracle_mod):
    """Two more batches of 16 PU200 events (event numbers 48-63 and 80-95) on one context at 2 and 1 blocks per SM,
    each run twice (the second replays the graph on a used workspace): every event equals the oracle's.  These
    are the batches on which a dropped variant of k_rule3 failed (profiles/r02_iterations.md, section 6)."""
    from concurrent.futures import ThreadPoolExecutor

    geom, off, tgt = make_config_geometry("C5")
    g = lst.lst_load_geometry(geom.module_table(), off, tgt)
    ctx = lst.lst_ctx_create(g, lst.lst_default_caps(max_events=16))
    try:
        for first in (48, 80):
            evs = [make_config_event("C5", pu=200, index=first + i, seeds=True) for i in range(16)]
            with ThreadPoolExecutor(16) as ex:  # ctypes releases the GIL: one oracle call per core
                want = list(ex.map(lambda ev: canon(oracle_mod.run_event(geom.subdet, off, tgt, ev.x, ev.y, ev.z,
                                                                         ev.sensor, ev.pls)), evs))
            for blocks in (2, 1):
                lst.lst_ctx_set_blocks_per_sm(ctx, blocks)
                for rep in range(2):
                    run_batch(lst, ctx, evs)
                    for i in range(16):
                        assert_same(canon(lst.lst_ctx_fetch_event(ctx, i)), want[i],
                                    f"events {first}+, {blocks} blocks per SM, rep {rep}, event {i}: ")
    finally:
        lst.lst_free(ctx)
        lst.lst_free(g)


def test_many_small_events_in_one_batch(lst, oracle_mod):
    """40 events per launch sequence (more events than any table is sized for by default)."""
    geom, off, tgt = make_config_geometry("C4")
    from lst_inputs.events import EventSpec, generate_event

    evs = [generate_event(geom, EventSpec(n_tracks=30 + 5 * (k % 7), pt_dist=("loguniform", 0.8, 10.0), eta_max=1.0,
                                          noise=("count", 100), seeds=True), 5000 + k) for k in range(40)]
    g = lst.lst_load_geometry(geom.module_table(), off, tgt)
    ctx = lst.lst_ctx_create(g, lst.lst_default_caps(max_events=40))
    try:
        summ = run_batch(lst, ctx, evs)
        assert summ["n_events"] == 40
        n_tc = 0
        for i, ev in enumerate(evs):
            want = oracle_mod.run_event(geom.subdet, off, tgt, ev.x, ev.y, ev.z, ev.sensor, ev.pls)
            got = lst.lst_ctx_fetch_event(ctx, i)
            assert_same(canon(got), canon(want), f"40-event batch, event {i}: ")
            n_tc += len(want["tc"])
        assert summ["n_tc"] == n_tc
    finally:
        lst.lst_free(ctx)
        lst.lst_free(g)


def test_pu250_events(lst, oracle_mod):
    """The densest point of the BASELINE.json sweep (8,750 tracks per event)."""
    geom, off, tgt = make_config_geometry("C5")
    evs = c5_batch(pu=250, n_events=2)
    g = lst.lst_load_geometry(geom.module_table(), off, tgt)
    ctx = lst.lst_ctx_create(g, lst.lst_default_caps(max_events=2))
    try:
        run_batch(lst, ctx, evs)
        for i, ev in enumerate(evs):
            want = oracle_mod.run_event(geom.subdet, off, tgt, ev.x, ev.y, ev.z, ev.sensor, ev.pls)
            got = lst.lst_ctx_fetch_event(ctx, i)
            assert_same(canon(got), canon(want), f"PU250 event {i}: ")
    finally:
        lst.lst_free(ctx)
        lst.lst_free(g)
