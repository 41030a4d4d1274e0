"""Soak test of the benchmark's timed configuration, with every result checked.

bench.py's timed loop keeps eight contexts in flight on eight streams, each replaying its CUDA graph on one of six
rotating batches of 16 PU200 events, every kernel limited to 2 (or 1) resident blocks per SM so that kernels of
different batches share the SMs -- and it checks no result.  The parity tests check results but run a context for
two or three rounds.  A stale read of the workspace (a flag outside the region that is cleared per batch) or a race
between co-resident kernels would show up only after several rounds of several contexts, so this test runs that
exact configuration for 300 steps per variant (2 and 1 blocks per SM; inputs resident on the device, and pinned
host buffers with uint16 sensor ids, as bench.py's end-to-end leg) and, at every retire, compares with the oracle's
values for the batch that context just ran:
  * the batch summary: every object count, near[] and n_tests[] (sums of the oracle's per-event values);
  * the fetched track candidates of the whole batch as a set of rows (event, class, seed, 12 hit indices) --
    object indices inside a row (t5, t3) are implementation-local and left out, as in tests/util.canon.
The oracle runs once per batch (96 events, one thread per event).
"""
from concurrent.futures import ThreadPoolExecutor

import numpy as np
import pytest

from lst_inputs import make_config_event, make_config_geometry
from lst_inputs.events import concat_events

pytestmark = pytest.mark.gpu

E, S, NB, STEPS = 16, 8, 6, 300   # bench.py defaults: --events, --streams, --batches; steps per variant
COUNTS = ("n_md", "n_ls", "n_t3", "n_t5", "n_pt3", "n_pt5", "n_tc")


@pytest.fixture(scope="module")
def lst():
    import torch

    assert torch.cuda.is_available()
    from paper_2407_18231_b200 import build

    build.build()
    import paper_2407_18231_b200 as m

    return m


def tc_rows(tc, offsets):
    """Sorted rows (event, class, seed, hit indices) of a batch's track candidates."""
    tc = np.asarray(tc, dtype=np.int64).reshape(-1, 16)
    ev = np.repeat(np.arange(len(offsets) - 1), np.diff(offsets))
    rows = np.concatenate([ev[:, None], tc[:, 0:2], tc[:, 4:16]], axis=1)
    return rows[np.lexsort(rows.T[::-1])]


@pytest.fixture(scope="module")
def workload(oracle_mod):
    """Six batches of 16 PU200 events (event numbers 0..95, as bench.py on rank 0) and the oracle's result for each."""
    geom, off, tgt = make_config_geometry("C5")
    batches, expect = [], []
    with ThreadPoolExecutor(16) as ex:  # ctypes releases the GIL inside the oracle's C call
        for b in range(NB):
            evs = [make_config_event("C5", pu=200, index=b * E + i, seeds=True) for i in range(E)]
            res = list(ex.map(lambda ev: oracle_mod.run_event(geom.subdet, off, tgt, ev.x, ev.y, ev.z, ev.sensor, ev.pls), evs))
            keys = ("md_hits", "ls_md", "t3_md", "t5_md", "pt3", "pt5", "tc")
            want = {c: int(sum(len(r[k]) for r in res)) for c, k in zip(COUNTS, keys)}
            want["near"] = np.sum([r["near"] for r in res], axis=0).astype(np.int64).tolist()
            want["n_tests"] = np.sum([r["n_tests"] for r in res], axis=0).astype(np.int64).tolist()
            tc_off = np.concatenate([[0], np.cumsum([len(r["tc"]) for r in res])])
            want["tc"] = tc_rows(np.concatenate([r["tc"] for r in res]), tc_off)
            batches.append(concat_events(evs))
            expect.append(want)
    return geom, off, tgt, batches, expect


def soak(lst, workload, blocks_per_sm, host_inputs):
    import torch

    geom, off, tgt, batches, expect = workload
    g = lst.lst_load_geometry(geom.module_table(), off, tgt)
    caps = lst.lst_default_caps(max_events=E)
    streams = [torch.cuda.Stream() for _ in range(S)]
    ctxs = [lst.lst_ctx_create(g, caps, st.cuda_stream) for st in streams]
    try:
        for c in ctxs:
            lst.lst_ctx_set_blocks_per_sm(c, blocks_per_sm)
        f_hit, f_pls = ("x", "y", "z", "sensor"), ("pt", "x0", "y0", "z0", "x1", "y1", "z1", "q")
        inputs = []
        for b in batches:
            pin = {k: torch.from_numpy(np.ascontiguousarray(b[k])).pin_memory() for k in f_hit}
            pin_p = {k: torch.from_numpy(np.ascontiguousarray(b["pls"][k])).pin_memory() for k in f_pls}
            if host_inputs:
                pin["sensor"] = torch.from_numpy(np.ascontiguousarray(b["sensor"].astype(np.uint16))).pin_memory()
                h, keep = lst.make_hits(*(pin[k].numpy() for k in f_hit), b["hit_offsets"])
                s, keep = lst.make_pls({k: v.numpy() for k, v in pin_p.items()}, b["pls_offsets"], keep)
                inputs.append((h, s, keep, pin, pin_p))
            else:
                d = {k: v.cuda() for k, v in pin.items()}
                d_p = {k: v.cuda() for k, v in pin_p.items()}
                h, keep = lst.make_hits(d["x"], d["y"], d["z"], d["sensor"], b["hit_offsets"])
                s, keep = lst.make_pls(d_p, b["pls_offsets"], keep)
                inputs.append((h, s, keep, d, d_p))
        torch.cuda.synchronize()
        tc_pin = [torch.empty((caps.max_tc, 16), dtype=torch.int32).pin_memory().numpy() for _ in range(S)]
        running = [None] * S   # batch number a context has in flight
        checked = 0

        def retire(c, step):
            nonlocal checked
            want = expect[running[c]]
            where = f"blocks/SM {blocks_per_sm}, {'host' if host_inputs else 'device'} inputs, step {step}, " \
                    f"context {c}, batch {running[c]}: "
            summ = lst.lst_ctx_sync(ctxs[c])
            for k in COUNTS:
                assert summ[k] == want[k], where + f"{k} {summ[k]} != {want[k]}"
            assert summ["near"] == want["near"], where + f"near {summ['near']} != {want['near']}"
            assert summ["n_tests"] == want["n_tests"], where + "n_tests"
            tc, tc_off = lst.lst_ctx_fetch_tc(ctxs[c], tc_pin[c], E)
            assert np.array_equal(tc_rows(tc, tc_off), want["tc"]), where + "track candidates differ"
            running[c] = None
            checked += 1

        for i in range(STEPS):  # the loop of bench.py's pipelined()
            c = i % S
            if running[c] is not None:
                retire(c, i)
            h, s = inputs[i % NB][0], inputs[i % NB][1]
            lst.lst_ctx_run(ctxs[c], E, h, s)
            running[c] = i % NB
        for c in range(S):
            if running[c] is not None:
                retire(c, STEPS)
        torch.cuda.synchronize()
        assert checked == STEPS
    finally:
        for c in ctxs:
            lst.lst_free(c)
        lst.lst_free(g)


@pytest.mark.parametrize("host_inputs", [False, True], ids=["device_inputs", "pinned_host_inputs"])
@pytest.mark.parametrize("blocks_per_sm", [2, 1])
def test_timed_configuration_300_steps_every_result_checked(lst, workload, blocks_per_sm, host_inputs):
    soak(lst, workload, blocks_per_sm, host_inputs)
