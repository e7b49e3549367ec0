"""Host logic of multi-GPU event sharding.

Events are independent and the RNG is keyed by the global event index, so a batch shards by contiguous
event ranges with no collective inside the chain.  What is left for the host:

  * balanced_event_ranges : split [0, n_events) into `world` contiguous ranges of ~equal particle count
  * shard_arrays          : the CSR slice of one range (offsets rebased to 0); its event_base is e0
  * exchange_totals       : ONE all-gather of three int64 per rank (tracks, towers, eflow totals) ->
                            this rank's bases in the global output CSR
  * rebase_outputs        : shift a shard's output offsets by those bases and its particle indices
                            (trk_src, efl_src of track entries) by the shard's first particle
  * concat_outputs        : stitch rebased shards into the single-call result

No detector arithmetic lives here.  numpy only; torch.distributed is touched only by exchange_totals.
"""
from __future__ import annotations

import numpy as np

EVENT_ARRAYS = ("pid", "charge", "px", "py", "pz", "E", "vx", "vy", "vz")
PD_CLS_MUON = 2  # eflow classes 0..2 are track entries (src = particle index); 3, 4 are neutrals (src = tower id)


def balanced_event_ranges(offsets, world: int):
    """Contiguous event ranges [(e0, e1)] * world whose particle counts are as equal as whole events allow."""
    offsets = np.asarray(offsets, dtype=np.int64)
    ne = int(offsets.shape[0] - 1)
    if world < 1:
        raise ValueError("world must be >= 1")
    total = int(offsets[-1])
    cuts = [0]
    for r in range(1, world):
        target = (total * r) // world
        # first event boundary at or after the target, never before the previous cut
        e = int(np.searchsorted(offsets, target, side="left"))
        cuts.append(min(max(e, cuts[-1]), ne))
    cuts.append(ne)
    return [(cuts[r], cuts[r + 1]) for r in range(world)]


def shard_arrays(ev, e0: int, e1: int) -> dict:
    """CSR slice of events [e0, e1) as a dict of numpy arrays (offsets start at 0) + first_particle."""
    offsets = np.asarray(ev.offsets, dtype=np.int64)
    a, b = int(offsets[e0]), int(offsets[e1])
    out = {"offsets": offsets[e0:e1 + 1] - a, "first_particle": a, "event_base": int(e0)}
    for k in EVENT_ARRAYS:
        out[k] = np.ascontiguousarray(getattr(ev, k)[a:b])
    return out


def exchange_totals(totals, rank: int, world: int, dist=None, device=None):
    """All-gather (n_tracks, n_towers, n_eflow) of every rank; return (bases of this rank [3], all totals [world, 3])."""
    mine = np.asarray(totals, dtype=np.int64).reshape(3)
    if world == 1 or dist is None:
        return np.zeros(3, dtype=np.int64), mine.reshape(1, 3)
    import torch

    t = torch.from_numpy(mine.copy())
    if device is not None:
        t = t.to(device)
    gathered = [torch.zeros_like(t) for _ in range(world)]
    dist.all_gather(gathered, t)
    allt = np.stack([g.cpu().numpy() for g in gathered]).astype(np.int64)
    return allt[:rank].sum(axis=0), allt


def rebase_outputs(res: dict, bases, first_particle: int) -> dict:
    """Shift a shard's result (dict of trk_*/tow_*/efl_* numpy arrays) into the global numbering."""
    out = dict(res)
    for prefix, base in zip(("trk", "tow", "efl"), bases):
        out[prefix + "_offsets"] = np.asarray(res[prefix + "_offsets"], dtype=np.int64) + int(base)
    out["trk_src"] = np.asarray(res["trk_src"], dtype=np.int32) + np.int32(first_particle)
    src = np.asarray(res["efl_src"], dtype=np.int32).copy()
    is_track = np.asarray(res["efl_cls"]) <= PD_CLS_MUON
    src[is_track] += np.int32(first_particle)
    out["efl_src"] = src
    return out


def concat_outputs(shards) -> dict:
    """Concatenate rebased shard results (in rank order) into one result."""
    out = {}
    keys = [k for k in shards[0] if k.startswith(("trk_", "tow_", "efl_"))]
    for k in keys:
        if k.endswith("_offsets"):
            out[k] = np.concatenate([shards[0][k]] + [s[k][1:] for s in shards[1:]])
        else:
            out[k] = np.concatenate([s[k] for s in shards])
    return out
