"""-m gpu: one step of the chain captured in a CUDA graph.  After pd_card_upload the step allocates nothing and is made of stream
operations only (a memset of the workspace head and three kernel launches), so it can be captured once and replayed: the
launch-bound small batches (cfg0: 60,000 particles) then pay one graph launch instead of four operations.  The replayed
step must write bit for bit what the plain call writes, also after the inputs behind the same pointers have changed."""
import importlib

import numpy as np
import pytest

wl = importlib.import_module("workloads.generate")

pytestmark = pytest.mark.gpu


def test_a_step_captured_in_a_cuda_graph_replays_bit_for_bit():
    import torch

    import paper_2606_26089_b200 as pd

    card = pd.Card("cms_like")
    ev_a = wl.generate(0, 1000)
    # other events behind the same pointers: the same particle count and event sizes, momenta mirrored in z
    ev_b = wl.Events(offsets=ev_a.offsets, **{k: (-getattr(ev_a, k) if k in ("pz", "vz") else getattr(ev_a, k))
                                              for k in ("pid", "charge", "px", "py", "pz", "E", "vx", "vy", "vz")})
    pd.card_upload(card)
    # plain calls: the expected outputs for both batches
    want = []
    for ev in (ev_a, ev_b):
        dev = pd.DeviceEvents(ev)
        out = pd.DeviceOutputs(card, dev.n_events, dev.n_particles)
        pd.simulate(card, dev, out, 5)
        want.append(out.to_numpy())
    # capture with batch A resident
    side = torch.cuda.Stream()
    dev = pd.DeviceEvents(ev_a)
    out = pd.DeviceOutputs(card, dev.n_events, dev.n_particles)
    with torch.cuda.stream(side):
        pd.simulate(card, dev, out, 5)                            # warm-up on the capturing stream (kernel attributes, first launches)
    side.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=side):
        pd.simulate(card, dev, out, 5)
    for t in list(out.trk.values()) + list(out.tow.values()) + list(out.efl.values()):
        t.zero_()
    graph.replay()
    torch.cuda.synchronize()
    got = out.to_numpy()
    assert pd.last_status(out) == 0
    for k, v in want[0].items():
        assert got[k].tobytes() == v.tobytes(), k
    # the graph holds pointers and sizes, not data: batch B of the same shape behind the same pointers
    for k, t in dev.t.items():
        t.copy_(torch.from_numpy(np.ascontiguousarray(getattr(ev_b, k))))
    graph.replay()
    torch.cuda.synchronize()
    got = out.to_numpy()
    assert not np.array_equal(want[0]["tow_tower"], want[1]["tow_tower"])
    for k, v in want[1].items():
        assert got[k].tobytes() == v.tobytes(), k
    # replaying is cheaper than launching for a launch-bound batch (reported, not asserted: timing on a shared box)
    def timed(fn, reps=200):
        fn()
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(reps):
            fn()
        b.record()
        torch.cuda.synchronize()
        return a.elapsed_time(b) / reps

    t_plain = timed(lambda: pd.simulate(card, dev, out, 5))
    t_graph = timed(graph.replay)
    print("cfg0 step: %.4f ms by four stream operations, %.4f ms by one graph launch" % (t_plain, t_graph))
