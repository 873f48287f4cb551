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


def test_bench_gpus_n_spawns_n_ranks_over_shard():
    """`python bench.py --gpus N` (no torchrun around it) re-executes itself under torch.distributed.run with one rank
    per GPU, refuses to start when the box has fewer devices, and every rank takes shard.event_range of ONE batch of
    N x E events."""
    import subprocess
    import bench
    from synth import events
    cmd = bench.spawn_command(4, ["--gpus", "4", "--steps", "3"], 29517)
    assert cmd[0] == sys.executable and cmd[1:3] == ["-m", "torch.distributed.run"]
    assert "--nnodes=1" in cmd and "--nproc-per-node=4" in cmd
    assert cmd[cmd.index("--master-addr") + 1] == "127.0.0.1" and cmd[cmd.index("--master-port") + 1] == "29517"
    assert cmd[-5].endswith("bench.py") and cmd[-4:] == ["--gpus", "4", "--steps", "3"]
    import torch
    if not torch.cuda.is_available():
        r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "3"],
                           capture_output=True, text=True, timeout=300)
        assert r.returncode != 0 and "needs 2 CUDA devices" in (r.stderr + r.stdout)
    # the batches of a 3-rank job: drawn independently by every rank, together exactly the 3 x E events
    E, world = 400, 3
    import dataclasses
    whole = events.generate(dataclasses.replace(events.config(1, E), n_events=world * E))
    counts = np.diff(whole["offsets"]).astype(np.int64)
    parts = []
    for rank in range(world):
        seen = {}

        def gather(mine, rank=rank, seen=seen):
            assert np.array_equal(mine, counts[rank * E:(rank + 1) * E])          # the rank drew its nominal range
            seen["called"] = True
            return counts
        d, m, (e0, e1), T = bench.gen_batch(1, E, rank, world, gather)
        assert seen["called"] and m.n_events == world * E and T == whole["offsets"][-1]
        parts.append((e0, e1, d))
    assert parts[0][0] == 0 and parts[-1][1] == world * E
    assert all(parts[k][1] == parts[k + 1][0] for k in range(world - 1))
    for k in events.FIELDS:
        assert np.array_equal(np.concatenate([d[k] for _a, _b, d in parts]), whole[k]), k
    trk = [int(d["offsets"][-1]) for _a, _b, d in parts]
    assert max(trk) - min(trk) <= 2 * counts.max()                                # equal track counts per GPU
    d1, m1, rng1, T1 = bench.gen_batch(1, E)
    assert rng1 == (0, E) and np.array_equal(d1["x"], whole["x"][:whole["offsets"][E]])
