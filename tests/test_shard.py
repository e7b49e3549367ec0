"""Host logic of multi-GPU event sharding (paper_2606_26089_b200/shard.py), on CPU.

The N > 1 path has no data-path collective: each rank simulates a contiguous event range with its own
event_base, then ONE all-gather of three int64 per rank rebases the output CSR.  Here two `gloo` ranks
run that protocol with the oracle standing in for the per-rank simulate call (test infrastructure; the
sharding code under test is the product's), and the stitched result must equal the single-call result
bit for bit -- which also pins reading A27 (event index = event_base + index in call)."""
import importlib
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
wl = importlib.import_module("workloads.generate")

from paper_2606_26089_b200 import shard  # noqa: E402


def test_balanced_ranges_cover_and_balance():
    rng = np.random.default_rng(0)
    counts = rng.poisson(60, size=1000)
    offsets = np.concatenate([[0], np.cumsum(counts)]).astype(np.int64)
    for world in (1, 2, 3, 8):
        ranges = shard.balanced_event_ranges(offsets, world)
        assert ranges[0][0] == 0 and ranges[-1][1] == 1000
        assert all(a[1] == b[0] for a, b in zip(ranges, ranges[1:]))
        sizes = [int(offsets[e1] - offsets[e0]) for e0, e1 in ranges]
        assert max(sizes) - min(sizes) <= 2 * counts.max()
    # degenerate: fewer events than ranks, empty events, zero events
    assert shard.balanced_event_ranges(np.array([0, 5]), 4)[-1][1] == 1
    assert shard.balanced_event_ranges(np.array([0]), 2) == [(0, 0), (0, 0)]
    r = shard.balanced_event_ranges(np.array([0, 0, 0, 7, 7]), 2)
    assert r[0][0] == 0 and r[-1][1] == 4 and r[0][1] == r[1][0]


def test_rebase_and_concat_roundtrip_without_dist():
    from oracle import pdo

    ev = wl.generate(0, 50)
    card = pdo.Card("cms_like")
    full = pdo.simulate(card, ev, 7, debug=False)
    ranges = shard.balanced_event_ranges(ev.offsets, 3)
    parts, totals = [], []
    for e0, e1 in ranges:
        sh = shard.shard_arrays(ev, e0, e1)
        res = pdo.simulate(card, wl.slice_events(ev, e0, e1), 7, event_base=sh["event_base"], debug=False)
        parts.append((res, sh["first_particle"]))
        totals.append([int(res[p + "_offsets"][-1]) for p in ("trk", "tow", "efl")])
    bases = np.concatenate([[np.zeros(3, dtype=np.int64)], np.cumsum(np.array(totals), axis=0)[:-1]])
    merged = shard.concat_outputs([shard.rebase_outputs(r, b, fp) for (r, fp), b in zip(parts, bases)])
    for k, v in merged.items():
        assert np.array_equal(v, full[k]), k


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    if ROOT not in sys.path:
        sys.path.insert(0, ROOT)
    import torch.distributed as dist

    from oracle import pdo

    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ev = wl.generate(3, 400)
        e0, e1 = shard.balanced_event_ranges(ev.offsets, world)[rank]
        sh = shard.shard_arrays(ev, e0, e1)
        res = pdo.simulate(pdo.Card("atlas_like"), wl.slice_events(ev, e0, e1), 4, event_base=sh["event_base"], debug=False)
        totals = [int(res[p + "_offsets"][-1]) for p in ("trk", "tow", "efl")]
        bases, allt = shard.exchange_totals(totals, rank, world, dist)
        reb = shard.rebase_outputs(res, bases, sh["first_particle"])
        gathered = [None] * world
        dist.all_gather_object(gathered, reb)
        if rank == 0:
            q.put((shard.concat_outputs(gathered), allt))
    finally:
        dist.destroy_process_group()


def test_world_size_2_gloo_sharding_matches_single_call():
    import torch.multiprocessing as mp

    from oracle import pdo

    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    merged, allt = q.get(timeout=180)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    ev = wl.generate(3, 400)
    full = pdo.simulate(pdo.Card("atlas_like"), ev, 4, debug=False)
    assert allt.shape == (2, 3) and int(allt[:, 0].sum()) == int(full["trk_offsets"][-1])
    for k, v in merged.items():
        assert np.array_equal(v, full[k]), k
