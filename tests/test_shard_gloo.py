"""N > 1 path on CPU: world_size-2 gloo run of the sharding logic bench.py uses under torchrun."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1711_06571_b200 import shard, synth


def test_track_range_partitions():
    for n in (0, 1, 7, 1000, 1_000_003):
        for world in (1, 2, 3, 8):
            r = [shard.track_range(n, k, world) for k in range(world)]
            assert r[0][0] == 0 and r[-1][1] == n
            assert all(r[k][1] == r[k + 1][0] for k in range(world - 1))
            sizes = [e - b for b, e in r]
            assert max(sizes) - min(sizes) <= 1


def test_assign_events_balances_seed_counts():
    rng = np.random.default_rng(5)
    counts = rng.integers(9_000, 12_001, size=64)
    for world in (1, 2, 4, 8):
        a = shard.assign_events(counts, world)
        assert sorted(e for v in a for e in v) == list(range(64))
        load = [int(counts[v].sum()) for v in a]
        assert max(load) - min(load) <= counts.max()
    assert shard.assign_events([], 2) == [[], []]


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close()
    return p


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # weak scaling as in bench.py: every rank generates its own shard (event = rank) of the same size
        fi = synth.fit_inputs(0, n=256, event=rank)
        bi = synth.build_inputs(3, n_events=2, tracks=50, event0=rank * 1000)
        # strong split of one common track list
        b, e = shard.track_range(1001, rank, world)
        # timing reduction: the max over ranks is what every rank reports
        ms = shard.max_over_ranks(10.0 + rank)
        total = shard.sum_over_ranks(float(fi.n))
        # every rank computes the same event table
        table = shard.assign_events([bi.n_seeds + 3 * k for k in range(6)], world)
        # strong scaling of a build as bench.py does it: the rank generates exactly the events the table deals to it
        mine = shard.assign_events([50.0] * 5, world)[rank]
        sb = synth.build_inputs(3, events=mine, tracks=50)
        gathered = [None] * world
        dist.all_gather_object(gathered, dict(rank=rank, ms=ms, total=total, range=(b, e), table=table,
                                              par0=float(fi.par[3, 0]), hit0=float(bi.hit_x[0]),
                                              strong_events=[int(v) for v in sb.event_ids], strong_n_events=sb.n_events,
                                              strong_first_hits=[float(sb.hit_x[sb.seg_off[k * sb.geom.n_layers]]) for k in range(sb.n_events)]))
        if rank == 0:
            q.put(gathered)
    finally:
        dist.destroy_process_group()


def test_world_size_2_gloo():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.SimpleQueue()
    procs = [ctx.Process(target=_worker, args=(r, world, _free_port() if r < 0 else PORT, q)) for r in range(world)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    g = q.get()
    assert [x["rank"] for x in g] == [0, 1]
    assert all(x["ms"] == 11.0 for x in g)                    # max over ranks
    assert all(x["total"] == 512.0 for x in g)                # whole-job units = sum over ranks
    assert g[0]["range"] == (0, 501) and g[1]["range"] == (501, 1001)
    assert g[0]["table"] == g[1]["table"]
    assert g[0]["par0"] != g[1]["par0"] and g[0]["hit0"] != g[1]["hit0"]   # ranks work on different events
    # strong-scaled build: the ranks' events partition 0..4 -- no event is built twice, none is left out
    ev = [x["strong_events"] for x in g]
    assert sorted(ev[0] + ev[1]) == [0, 1, 2, 3, 4] and not set(ev[0]) & set(ev[1])
    assert [x["strong_n_events"] for x in g] == [len(ev[0]), len(ev[1])]
    # and an event's content depends on its global id only, not on the rank or its place in the call
    ref = synth.build_inputs(3, n_events=5, tracks=50)
    first = [float(ref.hit_x[ref.seg_off[k * ref.geom.n_layers]]) for k in range(5)]
    for x in g:
        assert x["strong_first_hits"] == [first[e] for e in x["strong_events"]]


PORT = _free_port()
