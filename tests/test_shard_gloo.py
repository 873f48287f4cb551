"""Multi-GPU host logic on CPU: event sharding and the gather of per-event results over a
world_size-2 gloo group.  Events are independent, so sharded results must equal the unsharded ones;
the per-rank compute in this CPU test is the oracle (the product has no CPU path)."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_event_ranges_partition_the_batch():
    from paper_2412_14966_b200 import shard
    from synth import events
    data = events.generate(events.config(1, 3000))
    off = data["offsets"]
    E, T = off.size - 1, int(off[-1])
    for world in (1, 2, 3, 8, 64):
        r = [shard.event_range(off, k, world) for k in range(world)]
        assert r[0][0] == 0 and r[-1][1] == E
        assert all(r[k][1] == r[k + 1][0] for k in range(world - 1))            # disjoint, ordered, complete
        trk = np.array([off[b] - off[a] for a, b in r])
        assert trk.sum() == T
        assert np.abs(trk - T / world).max() <= 2 * np.diff(off).max()            # balanced to within an event
    # more ranks than events, empty batch
    tiny = events.slice_events(data, 0, 3)
    r = [shard.event_range(tiny["offsets"], k, 8) for k in range(8)]
    assert sum(b - a for a, b in r) == 3 and all(b >= a for a, b in r)
    assert shard.event_range(np.zeros(1, np.int32), 0, 2) == (0, 0)
    s = shard.slice_batch(data, 10, 20)
    assert s["offsets"][0] == 0 and s["offsets"][-1] == off[20] - off[10]
    assert np.array_equal(s["x"], data["x"][off[10]:off[20]])


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    from oracle import pvref
    from paper_2412_14966_b200 import shard
    from synth import events
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    try:
        data = events.generate(events.config(1, 600))
        e0, e1 = shard.event_range(data["offsets"], rank, world)
        mine = shard.slice_batch(data, e0, e1)
        pvref.build()
        res = pvref.find(mine, pvref.default_params(), n_threads=1)
        n_vtx = shard.gather_per_event(res["n_vtx"])
        pos = shard.gather_per_event(res["vtx_pos"])
        trk_per_rank = shard.gather_per_event(np.array([mine["offsets"][-1]], np.int64))
        if rank == 0:
            q.put((n_vtx, pos, trk_per_rank))
    finally:
        dist.destroy_process_group()


def test_sharded_equals_unsharded_over_gloo():
    import torch.multiprocessing as mp
    from oracle import pvref
    from synth import events
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    world = 2
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    n_vtx, pos, trk = q.get(timeout=240)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    data = events.generate(events.config(1, 600))
    pvref.build()
    ref = pvref.find(data, pvref.default_params(), n_threads=1)
    assert np.array_equal(n_vtx, ref["n_vtx"])
    m = np.arange(pos.shape[1])[None, :] < ref["n_vtx"][:, None]
    assert np.array_equal(pos[m], ref["vtx_pos"][m])
    assert trk.sum() == data["offsets"][-1] and abs(int(trk[0]) - int(trk[1])) < 600
