"""-m gpu: a seeded random sweep over what the parity tests cover one at a time -- the three cards, the five workloads, random
subsets of the card options of DESIGN.md section 17 (K1 eta-dependent calorimeter resolutions, K2 significance cut, K3 smeared
tower positions, K4 eta-dependent track resolutions, K5 weighted EFlow, K6 a grid of its own for the HCAL), a reversed field, a
huge event among the small ones (big-tile path), the events-per-tile option -- each draw compared with the oracle through
tests/parity.py (integers exact, floats 1e-5 / 1e-6, near-edge overrides counted and bounded)."""
import importlib
import random

import numpy as np
import pytest

wl = importlib.import_module("workloads.generate")

pytestmark = pytest.mark.gpu


def _draw(rng, b, base):
    kw = {}
    if rng.random() < 0.5:
        kw["ecal_res_eta"] = [(0.0, 0.8, 0.005, 0.05, 0.2), (0.8, 1.6, 0.01, 0.1, 0.3), (2.0, 3.0, 0.03, 0.2, 0.0)]
        kw["hcal_res_eta"] = [(0.0, 1.3, 0.04, 1.0, 0.0), (1.3, 3.0, 0.06, 1.3, 0.5)]
    if rng.random() < 0.5:
        kw["ecal_nsigma"], kw["hcal_nsigma"] = rng.choice([0.5, 1.0, 2.0]), rng.choice([0.5, 1.2])
    if rng.random() < 0.5:
        kw["smear_tower_center"] = 1
    if rng.random() < 0.5:
        kw["track_res_eta"] = [(0.0, 0.9, 0.015, 2e-4), (0.9, 1.4, 0.05, 0.0, 2), (0.9, 1.4, 0.02, 3e-4), (1.7, "inf", 0.04, 1e-3)]
    if rng.random() < 0.5:
        kw["eflow_weighted"] = 1
    if rng.random() < 0.5:
        step = rng.choice([2, 3])
        he = [float(x) for x in np.asarray(b.edges)[::step]]
        if he[-1] != float(b.edges[-1]):
            he.append(float(b.edges[-1]))
        kw["hcal_edges"] = he
        kw["hcal_nphi"] = [max(1, int(b.nphi[min(i * step, len(b.nphi) - 1)]) // step) for i in range(len(he) - 1)]
    if rng.random() < 0.3:
        kw["bz"] = -float(b.bz)
    return kw


@pytest.mark.parametrize("seed", [3, 17])
def test_random_cards_workloads_and_options(seed, tmp_path):
    import cards
    from gpu_util import run_gpu
    from oracle import pdo
    from parity import compare

    rng = random.Random(seed)
    for it in range(16):
        base = rng.choice(["cms_like", "atlas_like", "aleph_like"])
        cfg = {"cms_like": rng.choice([0, 1, 2]), "atlas_like": 3, "aleph_like": 4}[base]
        ne = {0: rng.randint(50, 1500), 1: rng.randint(20, 300), 2: rng.randint(2, 12), 3: rng.randint(100, 3000), 4: rng.randint(100, 3000)}[cfg]
        b = pdo.Card(base)
        kw = _draw(rng, b, base)
        path = cards.variant(tmp_path / ("c%d.card" % it), b.edges, b.nphi, base=base, **kw)
        ev = wl.generate(cfg, ne)
        if rng.random() < 0.3:  # a huge event in the middle: its tile takes the big-tile path
            big = wl.generate(2, 3)
            big = wl.Events(offsets=np.array([0, big.n_particles], dtype=np.int64),
                            **{k: getattr(big, k) for k in ("pid", "charge", "px", "py", "pz", "E", "vx", "vy", "vz")})
            ev = wl.concat_events([wl.slice_events(ev, 0, ne // 2), big, wl.slice_events(ev, ne // 2, ne)])
        call_seed = rng.randint(0, 2**40)
        tile_events = rng.choice([0, 0, 1, 7])
        gpu = run_gpu(path, ev, call_seed, tile_events=tile_events)
        assert gpu["status_word"] == 0
        rep = compare(path, ev, call_seed, gpu)
        what = (seed, it, base, cfg, ne, sorted(kw), tile_events)
        assert rep["unexcused"] == 0, (what, rep["problems"][:5])
        assert rep["overridden_particles"] <= max(3, 5e-4 * rep["n_particles"]), (what, rep["overridden_particles"])
