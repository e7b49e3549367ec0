"""-m gpu: pd_truth_features (H_T and E_T^miss over the truth collection; Table 2, readings T1, T2 of
DESIGN.md section 15) through the C ABI against the fp64 oracle, event by event, on seeded synthetic inputs.

Tolerances (as for the PFlow-side features): H_T is an exact fixed-point sum of fp32 pT values
(each sqrt(px^2 + py^2) rounded to fp32: 1e-7 relative) -> 1e-5 relative / 1e-6 absolute; the components of E_T^miss
are exact sums of the fp32 inputs, so they agree to the rounding of the fp32 OUTPUT, whose scale is set by the terms,
not by the possibly cancelling result: |g - o| <= 1e-6 H_T + 1e-6."""
import importlib

import numpy as np
import pytest

wl = importlib.import_module("workloads.generate")

pytestmark = pytest.mark.gpu


def _run_gpu(ev, skip=True):
    import paper_2606_26089_b200 as pd

    dev = pd.DeviceEvents(ev)
    feat = pd.DeviceFeatures(dev.n_events, 1)
    pd.truth_features(dev, feat, skip)
    assert pd.last_launch_count() == (0 if dev.n_events == 0 else (2 if dev.n_particles > 0 else 1))
    r = feat.to_numpy(0)
    return {k: r[k] for k in ("ht", "met_x", "met_y", "met")}


def _check(g, o):
    ht = o["ht"]
    assert np.all(np.abs(g["ht"] - ht) <= np.maximum(1e-5 * ht, 1e-6))
    for k in ("met_x", "met_y", "met"):
        assert np.all(np.abs(g[k] - o[k]) <= 1e-6 * ht + 1e-6), k


@pytest.mark.parametrize("cfg,n_events", [(0, 3000), (1, 400), (2, 30), (3, 20000), (4, 20000)])
def test_truth_features_of_the_workloads(cfg, n_events):
    from oracle import pdo

    ev = wl.generate(cfg, n_events)
    for skip in (True, False):
        _check(_run_gpu(ev, skip), pdo.truth_features(ev, skip))


def _random_events(seed, sizes, nu_frac=0.1):
    rng = np.random.default_rng(seed)
    offsets = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int64)
    n = int(offsets[-1])
    pid = rng.choice([211, -211, 22, 130, 11, -13, 12, -14, 16, -16], n,
                     p=[(1 - nu_frac) / 6] * 6 + [nu_frac / 4] * 4).astype(np.int32)
    pt = 0.05 * 4000 ** rng.random(n)
    phi = rng.uniform(-np.pi, np.pi, n)
    z = np.zeros(n, dtype=np.float32)
    return wl.Events(offsets=offsets, pid=pid, charge=np.zeros(n, np.int8), px=(pt * np.cos(phi)).astype(np.float32),
                     py=(pt * np.sin(phi)).astype(np.float32), pz=z, E=pt.astype(np.float32), vx=z, vy=z, vz=z)


def test_ragged_events_tile_boundaries_and_edge_cases():
    from oracle import pdo

    # events that end exactly on, one before and one after the 2,048-particle tile boundaries; empty events; one
    # event spanning several tiles; a tile with fewer than 8 events (segments cut into pieces) and tiles with many
    sizes = [0, 2048, 0, 0, 2047, 1, 2049, 4095, 1, 0, 7000, 3, 5, 0, 1, 1, 1] + [7] * 900 + [0] * 5000 + [1] * 3000 + [12345]
    ev = _random_events(3, sizes)
    for skip in (True, False):
        _check(_run_gpu(ev, skip), pdo.truth_features(ev, skip))
    # more empty events inside one tile than the on-chip offset cache holds (offsets then read from global memory)
    ev = _random_events(4, [5] + [0] * 6000 + [9] + [0] * 3000 + [2])
    _check(_run_gpu(ev), pdo.truth_features(ev))
    # neutrinos only: everything is 0 with the default, H_T > 0 without
    ev = _random_events(5, [10, 20], nu_frac=1.0)
    g = _run_gpu(ev)
    assert np.all(g["ht"] == 0) and np.all(g["met"] == 0) and np.all(_run_gpu(ev, False)["ht"] > 0)
    # events without particles; zero events
    g = _run_gpu(_random_events(6, [0, 0, 0]))
    assert g["ht"].tolist() == [0, 0, 0] and g["met"].tolist() == [0, 0, 0]
    assert _run_gpu(_random_events(7, []))["ht"].shape == (0,)


def test_batches_of_huge_events_take_the_register_path():
    """batches whose events average 2,048 particles or more run the kernel variant with the register path (tiles that lie in one or
    two events); its sums are the same exact fixed-point sums: against the oracle, and bit for bit against the other variant, which
    the same events get when enough empty events are appended to bring the average down"""
    from oracle import pdo

    # boundaries exactly on, one before and one after a tile edge; runs of tiny and empty events between huge ones (those tiles take
    # the staged path inside the same kernel); a last event that ends mid-tile
    sizes = [5000, 0, 0, 3, 7000, 1, 2, 2, 6000, 4096, 2048, 2047, 2049, 10000, 0, 12288, 4095, 1, 20000, 6001] + [3000] * 7 + [9000, 0, 0]
    assert sum(sizes) >= 2048 * len(sizes)
    ev = _random_events(21, sizes)
    for skip in (True, False):
        g = _run_gpu(ev, skip)
        _check(g, pdo.truth_features(ev, skip))
        padded = _random_events(21, sizes + [0] * 100)  # the same particles (same seed and sizes first), average below 2,048
        assert padded.px[: ev.n_particles].tobytes() == ev.px.tobytes()
        h = _run_gpu(padded, skip)
        for k in g:
            assert h[k][: len(sizes)].tobytes() == g[k].tobytes(), k
    # one event only; two events split inside a tile; a batch that ends exactly on a tile edge
    for sz in ([30000], [3000, 3100], [2048, 2048, 4096]):
        ev = _random_events(22, sz)
        _check(_run_gpu(ev), pdo.truth_features(ev))


def test_bitwise_reproducible_and_independent_of_batching():
    ev = _random_events(9, np.random.default_rng(2).poisson(300, 4000))
    a, b = _run_gpu(ev), _run_gpu(ev)
    for k in a:
        assert a[k].tobytes() == b[k].tobytes(), k
    cut = 1234
    h1, h2 = _run_gpu(wl.slice_events(ev, 0, cut)), _run_gpu(wl.slice_events(ev, cut, 4000))
    for k in a:
        assert np.concatenate([h1[k], h2[k]]).tobytes() == a[k].tobytes(), k
