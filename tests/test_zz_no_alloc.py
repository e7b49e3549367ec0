"""-m gpu: pd_truth_features_static, the entry point that allocates nothing (include/pd.h): the [n_events][3] accumulators of
pd_truth_features in a fixed device array inside the library instead of a caller's workspace.  Checked against the
existing path (pd_truth_features with a workspace) on two calls in a row -- the second on a smaller, different batch, so
that anything the first call left in the shared array would show -- within the tolerance of
tests/test_gpu_truth_features.py (and, since both paths run the same exact fixed-point sums, bit for bit); against the
oracle; at the limit and beyond it; and that a call leaves the amount of free device memory as it found it.

Collected last on purpose (the suite runs with pytest -x); passes alone in a fresh process and after the other tests."""
import importlib

import numpy as np
import pytest

wl = importlib.import_module("workloads.generate")

pytestmark = pytest.mark.gpu

KEYS = ("ht", "met_x", "met_y", "met")


def _check(g, o):
    """the tolerance of tests/test_gpu_truth_features.py"""
    ht = o["ht"]
    assert np.all(np.abs(g["ht"] - ht) <= np.maximum(1e-5 * ht, 1e-6))
    for k in ("met_x", "met_y", "met"):
        assert np.all(np.abs(g[k] - o[k]) <= 1e-6 * ht + 1e-6), k


def _existing(pd, dev, skip):
    feat = pd.DeviceFeatures(dev.n_events, 1)
    pd.truth_features(dev, feat, skip)
    r = feat.to_numpy(0)
    return {k: r[k] for k in KEYS}


def _static(pd, dev, skip):
    import torch

    feat = pd.DeviceFeatures(dev.n_events, 1)
    for k in KEYS:
        feat.ev[k].fill_(float("nan"))  # every output must be written by the call
    pd.truth_features_static(dev, feat, skip)
    torch.cuda.synchronize()
    r = feat.to_numpy(0)
    return {k: r[k] for k in KEYS}


def test_two_calls_in_a_row_match_the_existing_path():
    import paper_2606_26089_b200 as pd
    from oracle import pdo

    # first a batch of many events with large sums, then a smaller one of other events: stale accumulators would show
    batches = [(wl.generate(1, 2000), True), (wl.generate(0, 700), False), (wl.generate(3, 5000), True)]
    for ev, skip in batches:
        dev = pd.DeviceEvents(ev)
        want = _existing(pd, dev, skip)
        got = _static(pd, dev, skip)
        _check(got, want)
        for k in KEYS:
            assert got[k].tobytes() == want[k].tobytes(), k  # the same exact sums
        _check(got, pdo.truth_features(ev, skip))
    # the same batch twice in a row gives the same answer twice
    dev = pd.DeviceEvents(batches[0][0])
    a, b = _static(pd, dev, True), _static(pd, dev, True)
    assert all(a[k].tobytes() == b[k].tobytes() for k in KEYS)


def test_limit_and_beyond():
    import paper_2606_26089_b200 as pd

    n_max = pd.binding.TRUTH_STATIC_MAX_EVENTS
    assert n_max == 262144

    def sparse_events(n_events):
        # a few particles in the first, a middle and the last event; every other event empty
        sizes = np.zeros(n_events, dtype=np.int64)
        sizes[[0, n_events // 2, n_events - 1]] = (3, 2, 4)
        off = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int64)
        n = int(off[-1])
        f = np.arange(1, n + 1, dtype=np.float32)
        z = np.zeros(n, dtype=np.float32)
        return wl.Events(offsets=off, pid=np.full(n, 211, np.int32), charge=np.zeros(n, np.int8), px=f, py=-2 * f, pz=z, E=3 * f,
                         vx=z, vy=z, vz=z)

    # exactly the maximum: accepted, and equal to the existing path
    dev = pd.DeviceEvents(sparse_events(n_max))
    want, got = _existing(pd, dev, True), _static(pd, dev, True)
    _check(got, want)
    assert got["ht"][0] > 0 and got["ht"][n_max - 1] > 0 and not got["ht"][1:n_max // 2].any()
    # one more: refused with PD_EWORKSPACE, nothing launched, nothing written
    dev = pd.DeviceEvents(sparse_events(n_max + 1))
    feat = pd.DeviceFeatures(dev.n_events, 1)
    feat.ev["ht"].fill_(-1.0)
    with pytest.raises(pd.PdError) as e:
        pd.truth_features_static(dev, feat, True)
    assert e.value.code == pd.binding.PD_EWORKSPACE
    assert "too small" in pd.binding.lib().pd_strerror(e.value.code).decode()
    assert bool((feat.ev["ht"] == -1.0).all())
    # an empty batch is the set-up call: PD_OK, nothing else
    pd.truth_features_static(pd.DeviceEvents(wl.from_lists([])), pd.DeviceFeatures(0, 1), True)


def test_a_call_allocates_no_device_memory():
    import torch

    import paper_2606_26089_b200 as pd

    dev = pd.DeviceEvents(wl.generate(0, 1000))
    feat = pd.DeviceFeatures(dev.n_events, 1)
    pd.truth_features_static(dev, feat, True)  # set-up: symbol address, module load, first launches
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        pd.truth_features_static(dev, feat, True)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0, (free0, free1)
