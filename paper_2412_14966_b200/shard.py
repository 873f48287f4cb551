"""Multi-GPU host logic: events are independent, so a batch is sharded over ranks by contiguous event
ranges of about equal track count, every rank runs pv_find on its slice, and nothing is exchanged on the data
path.  Only the small per-event results are gathered when a caller wants them in one place.
Pure index arithmetic: no method arithmetic here."""
from __future__ import annotations

from typing import Dict, Tuple

import numpy as np

FIELDS = ("x", "y", "z", "tx", "ty", "var_x", "var_y", "var_tx", "var_ty")


def event_range(offsets: np.ndarray, rank: int, world: int) -> Tuple[int, int]:
    """[e0, e1) of `rank`: boundaries at the events whose first track is the first at or beyond rank * T / world, so
    the ranges are disjoint, ordered, cover every event, and hold about T / world tracks each.  (pv_find_host places
    its chunk boundaries the same way, at targets that follow its ramped chunk weights instead of k / world.)"""
    offsets = np.asarray(offsets)
    E = int(offsets.size - 1)
    if world < 1 or not 0 <= rank < world:
        raise ValueError("need 0 <= rank < world")
    if E <= 0:
        return 0, 0
    T = int(offsets[-1])

    def bound(k: int) -> int:
        if k <= 0:
            return 0
        if k >= world:
            return E
        return int(min(np.searchsorted(offsets[:E], (T * k) // world, side="left"), E))

    e0, e1 = bound(rank), bound(rank + 1)
    return e0, max(e0, e1)


def slice_batch(data: Dict[str, np.ndarray], e0: int, e1: int) -> Dict[str, np.ndarray]:
    """The events [e0, e1) as a batch of their own (offsets rebased to 0)."""
    off = np.asarray(data["offsets"])
    t0, t1 = int(off[e0]), int(off[e1])
    out = {k: np.ascontiguousarray(data[k][t0:t1]) for k in FIELDS}
    out["offsets"] = (off[e0:e1 + 1] - off[e0]).astype(np.int32)
    return out


def gather_per_event(local: np.ndarray, group=None) -> np.ndarray:
    """Concatenate a per-event array over the ranks in rank order (torch.distributed all_gather of ragged
    pieces: sizes first, then padded payloads).  Works with gloo (CPU tensors) and nccl (device tensors)."""
    import torch
    import torch.distributed as dist
    world = dist.get_world_size(group)
    t = torch.as_tensor(np.ascontiguousarray(local))
    dev = torch.device("cuda", torch.cuda.current_device()) if dist.get_backend(group) == "nccl" else torch.device("cpu")
    t = t.to(dev)
    n = torch.tensor([t.shape[0]], dtype=torch.int64, device=dev)
    sizes = [torch.zeros_like(n) for _ in range(world)]
    dist.all_gather(sizes, n, group=group)
    sizes = [int(s.item()) for s in sizes]
    cap = max(sizes + [1])
    pad = torch.zeros((cap,) + tuple(t.shape[1:]), dtype=t.dtype, device=dev)
    pad[: t.shape[0]] = t
    parts = [torch.zeros_like(pad) for _ in range(world)]
    dist.all_gather(parts, pad, group=group)
    return torch.cat([p[:s] for p, s in zip(parts, sizes)], dim=0).cpu().numpy()
