"""Multi-GPU sharding of the VELO path: events are independent units
(§3, the farm processes an event stream), so ranks reconstruct disjoint contiguous
event ranges with the replicated geometry and parameters. There is NO data-path collective. The
only exchange, needed just when one global track numbering is wanted, is an all-gather of two
integers per rank (n_tracks, n_track_hits) followed by a local offset add.

Host logic only (no method arithmetic): it is covered by the world_size-2 `gloo` test in
tests/test_sharding.py and used by bench.py for N > 1.
"""
from __future__ import annotations

import numpy as np


def event_range(rank: int, world: int, n_events: int) -> tuple[int, int]:
    """Strong scaling: the contiguous, balanced range [e0, e1) of a fixed batch that `rank` owns."""
    if not (0 <= rank < world):
        raise ValueError("rank outside the world")
    return n_events * rank // world, n_events * (rank + 1) // world


def weak_event_range(rank: int, events_per_rank: int) -> tuple[int, int]:
    """Weak scaling (bench.py): every rank owns `events_per_rank` events of the generator's
    stream; event e depends only on (seed, e), so the ranks' workloads are disjoint."""
    return rank * events_per_rank, (rank + 1) * events_per_rank


def slice_events(d: dict, e0: int, e1: int) -> dict:
    """The inputs of events [e0, e1) of a batch, with offsets rebased to the slice."""
    off = np.asarray(d["event_offsets"]).astype(np.int64)
    h0, h1 = int(off[e0]), int(off[e1])
    return {"x": d["x"][h0:h1], "y": d["y"][h0:h1], "z": d["z"][h0:h1], "module": d["module"][h0:h1],
            "event_offsets": (off[e0:e1 + 1] - h0).astype(np.uint32), "n_events": e1 - e0, "n_hits": h1 - h0,
            "first_hit": h0, "first_event": e0}


def global_bases(n_tracks: int, n_track_hits: int, group=None) -> dict:
    """All-gather of (n_tracks, n_track_hits): this rank's base in the global track and track-hit
    numbering, and the totals. Works on any initialised torch.distributed backend (nccl tensors on
    the current CUDA device, gloo tensors on the CPU)."""
    import torch
    import torch.distributed as dist
    if not dist.is_available() or not dist.is_initialized():
        return {"track_base": 0, "track_hit_base": 0, "total_tracks": n_tracks, "total_track_hits": n_track_hits}
    dev = torch.device("cuda", torch.cuda.current_device()) if dist.get_backend(group) == "nccl" else torch.device("cpu")
    mine = torch.tensor([n_tracks, n_track_hits], dtype=torch.int64, device=dev)
    world = dist.get_world_size(group)
    parts = [torch.zeros_like(mine) for _ in range(world)]
    dist.all_gather(parts, mine, group=group)
    counts = torch.stack(parts).cpu().numpy()
    rank = dist.get_rank(group)
    return {"track_base": int(counts[:rank, 0].sum()), "track_hit_base": int(counts[:rank, 1].sum()),
            "total_tracks": int(counts[:, 0].sum()), "total_track_hits": int(counts[:, 1].sum())}


def to_global(res: dict, sl: dict, bases: dict) -> dict:
    """A rank's result (offsets local to its slice) renumbered into the batch-global numbering:
    track_hits become absolute hit indices of the whole batch, the offset arrays start at the
    rank's bases (first element dropped by the caller when concatenating)."""
    out = dict(res)
    out["track_hits"] = np.asarray(res["track_hits"]).astype(np.uint32) + np.uint32(sl["first_hit"])
    out["event_track_offsets"] = np.asarray(res["event_track_offsets"]).astype(np.uint32) + np.uint32(bases["track_base"])
    out["track_hit_offsets"] = np.asarray(res["track_hit_offsets"]).astype(np.uint32) + np.uint32(bases["track_hit_base"])
    return out
