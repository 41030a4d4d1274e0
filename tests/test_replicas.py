"""Multi-rank host logic (replicas only, no data-path collective) on CPU with gloo, world_size 2."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2407_18231_b200 import replicas


def test_event_indices_partition_the_events():
    world, nb, e = 4, 3, 16
    seen = []
    for r in range(world):
        batches = replicas.event_indices(r, world, nb, e)
        assert len(batches) == nb and all(len(b) == e for b in batches)
        assert batches == replicas.event_indices(r, world, nb, e)  # deterministic
        seen += [i for b in batches for i in b]
    assert sorted(seen) == list(range(world * nb * e))  # disjoint and complete
    with pytest.raises(ValueError):
        replicas.event_indices(4, 4, 1, 1)


def test_reductions_without_a_process_group_are_identities():
    assert replicas.max_over_ranks([1.5, 2.0]) == [1.5, 2.0]
    assert replicas.sum_over_ranks([3]) == [3.0]
    replicas.barrier()


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        mine = replicas.event_indices(rank, world, 2, 4)
        # every rank generates its own first event: different seeds -> different events
        from lst_inputs import make_config_event

        ev = make_config_event("C5", pu=50, index=mine[0][0])
        replicas.barrier()
        ms = replicas.max_over_ranks([10.0 + rank, 5.0 - rank])
        tot = replicas.sum_over_ranks([ev.n_hits, len(mine) * len(mine[0])])
        out.put((rank, mine, ev.n_hits, ms, tot))
    finally:
        dist.destroy_process_group()


def test_two_ranks_gloo():
    world = 2
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, m0, h0, ms0, t0), (r1, m1, h1, ms1, t1) = res
    assert not set(sum(m0, [])) & set(sum(m1, []))  # the ranks take different events
    assert h0 != h1  # and therefore see different inputs
    assert ms0 == ms1 == [11.0, 5.0]  # max over ranks, the same on every rank
    assert t0 == t1 == [float(h0 + h1), 16.0]  # whole-job totals
