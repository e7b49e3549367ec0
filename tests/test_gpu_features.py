"""-m gpu: pd_event_features (H_T, E_T^miss, lepton isolation Eq. 1) through the C ABI
against the fp64 oracle, element by element.  The input collections come from the ORACLE's own chain output and
from seeded synthetic generators -- never from the CUDA chain.

Tolerances: H_T and the isolation sums are exact fixed-point sums of fp32 terms, compared
at the north-star 1e-5 relative / 1e-6 absolute; the components of E_T^miss are sums of products pT cos(phi)
each rounded to fp32 (relative 2^-23, plus a 1e-7 cosine error), so their absolute error scales with H_T, not
with the (possibly cancelling) result: |g - o| <= 1e-6 H_T + 1e-6.  A cone decision within 1e-6 of its edge may go
either way (north_star): the oracle reports the pT at stake per lepton (iso_amb) and it is added to the bound."""
import importlib

import numpy as np
import pytest

wl = importlib.import_module("workloads.generate")

pytestmark = pytest.mark.gpu


def _run_gpu(offsets, cls, pt, eta, phi, dr_max=0.4, fsr_dr=0.0):
    import paper_2606_26089_b200 as pd

    obj = pd.DeviceObjects(offsets, cls, pt, eta, phi)
    feat = pd.DeviceFeatures(obj.n_events, obj.n_objects)
    pd.event_features(obj, feat, dr_max, fsr_dr)
    assert pd.last_launch_count() == (1 if obj.n_events > 0 else 0)
    return feat.to_numpy(obj.n_objects)


def _check(g, o, pt):
    ht = o["ht"]
    assert np.all(np.abs(g["ht"] - ht) <= np.maximum(1e-5 * ht, 1e-6))
    for k in ("met_x", "met_y", "met"):
        assert np.all(np.abs(g[k] - o[k]) <= 1e-6 * ht + 1e-6), k
    amb = o["iso_amb"]
    for k in ("iso_charged", "iso_neutral", "iso_photon"):
        assert np.all(np.abs(g[k] - o[k]) <= np.maximum(1e-5 * np.abs(o[k]), 1e-6) + amb * (1 + 1e-5)), k
    ptd = np.asarray(pt, dtype=np.float64)
    assert np.all(np.abs(g["r_iso"] - o["r_iso"]) <= np.maximum(1e-5 * np.abs(o["r_iso"]), 1e-6) + amb / np.maximum(ptd, 1e-30) * (1 + 1e-5))
    return int((amb > 0).sum())


@pytest.mark.parametrize("cfg,n_events", [(0, 600), (1, 200), (2, 12), (3, 2000), (4, 2000)])
def test_features_of_oracle_eflow(cfg, n_events):
    from oracle import pdo

    ev = wl.generate(cfg, n_events)
    o = pdo.simulate(pdo.Card(wl.config_card(cfg)), ev, wl.CONFIGS[cfg]["seed"], debug=False)
    off, cls = o["efl_offsets"], o["efl_cls"]
    pt, eta, phi = (o["efl_" + k].astype(np.float32) for k in ("pt", "eta", "phi"))
    for dr_max, fsr in ((0.4, 0.0), (0.3, 0.05)):
        ref = pdo.event_features(off, cls, pt, eta, phi, dr_max, fsr)
        got = _run_gpu(off, cls, pt, eta, phi, dr_max, fsr)
        n_amb = _check(got, ref, pt)
        lep = (cls == 1) | (cls == 2)
        assert lep.sum() > 0 and np.all(got["r_iso"][~lep] == 0)
    print("cfg%d: %d objects, %d leptons, %d near-edge" % (cfg, len(cls), int(lep.sum()), n_amb))


def _random_objects(seed, sizes, eta_max=1.5, lepton_frac=0.2):
    rng = np.random.default_rng(seed)
    offsets = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int64)
    n = int(offsets[-1])
    rest = (1 - lepton_frac) / 3
    cls = rng.choice([0, 1, 2, 3, 4], n, p=[rest, lepton_frac / 2, lepton_frac / 2, rest, rest]).astype(np.int8)
    pt = (0.2 * 2000 ** rng.random(n)).astype(np.float32)
    eta = rng.uniform(-eta_max, eta_max, n).astype(np.float32)
    phi = rng.uniform(-np.pi, np.pi, n).astype(np.float32)
    return offsets, cls, pt, eta, phi


def test_dense_random_collections_and_edge_cases():
    from oracle import pdo

    # ragged: empty events, single objects, a few hundred, and one event larger than the kernel's on-chip cache
    sizes = [0, 1, 0, 2, 33, 0, 257, 1, 5000, 64, 0, 0, 31, 32, 900, 3456, 3457, 0]
    args = _random_objects(5, sizes)
    for dr_max, fsr in ((0.4, 0.0), (0.4, 0.1), (0.0, 0.0), (10.0, 0.0)):
        _check(_run_gpu(*args, dr_max, fsr), pdo.event_features(*args, dr_max, fsr), args[2])
    # single big events per run (eta-strip pre-selection), wide eta range incl. beyond the strips' span, cones
    # narrower and wider than the minimum strip width
    args = _random_objects(7, [2500, 3000, 3072, 600, 2900], eta_max=7.0, lepton_frac=0.05)
    for dr_max, fsr in ((0.4, 0.0), (0.2, 0.05), (1.0, 0.0), (0.375, 0.0), (0.0, 0.0)):
        _check(_run_gpu(*args, dr_max, fsr), pdo.event_features(*args, dr_max, fsr), args[2])
    # many small events (several runs per chunk, several chunks per CTA)
    args = _random_objects(6, np.random.default_rng(1).poisson(30, 20000))
    _check(_run_gpu(*args), pdo.event_features(*args), args[2])
    # phi exactly at +-pi, identical directions (dR = 0), leptons only, no leptons at all
    off = np.array([0, 4, 7, 9], dtype=np.int64)
    cls = np.array([1, 4, 0, 3, 2, 2, 2, 0, 4], dtype=np.int8)
    pt = np.array([10, 1, 2, 3, 5, 6, 7, 1, 1], dtype=np.float32)
    eta = np.array([0, 0, 0.1, -0.1, 1, 1, 1.2, 0, 0], dtype=np.float32)
    phi = np.array([np.pi, -np.pi, 3.1, -3.1, 0, 0, 0, 0, 0], dtype=np.float32)
    g, o = _run_gpu(off, cls, pt, eta, phi), pdo.event_features(off, cls, pt, eta, phi)
    _check(g, o, pt)
    assert np.allclose(g["iso_charged"][:1], [2.0]) and np.allclose(g["iso_photon"][:1], [1.0]) and np.allclose(g["iso_neutral"][:1], [3.0])
    assert np.allclose(g["iso_charged"][4:7], [13.0, 12.0, 11.0]) and np.all(g["r_iso"][7:] == 0)
    # zero events
    z = _run_gpu(np.zeros(1, dtype=np.int64), np.zeros(0, np.int8), np.zeros(0, np.float32), np.zeros(0, np.float32), np.zeros(0, np.float32))
    assert z["ht"].shape == (0,)


def test_bitwise_reproducible_and_independent_of_batching():
    args = _random_objects(9, np.random.default_rng(2).poisson(120, 3000))
    a, b = _run_gpu(*args), _run_gpu(*args)
    for k in a:
        assert a[k].tobytes() == b[k].tobytes(), k
    off, cls, pt, eta, phi = args
    cut, m = 1234, int(off[1234])
    h1 = _run_gpu(off[: cut + 1], cls[:m], pt[:m], eta[:m], phi[:m])
    h2 = _run_gpu(off[cut:] - m, cls[m:], pt[m:], eta[m:], phi[m:])
    for k in a:
        assert np.concatenate([h1[k], h2[k]]).tobytes() == a[k].tobytes(), k
