"""-m gpu: parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (non-debug kernel,
the whole config in one pd_simulate call).

The oracle cannot run 4e7 particles in seconds, so the check is on SAMPLED events: windows of consecutive
events at the start, in the middle and at the end of the batch.  Events are independent and the RNG is keyed
by the global event index (reading A27), so
  (1) the window is re-run on the GPU alone with event_base = its first event and debug outputs on, and must
      reproduce the full-size run's records of those events BIT FOR BIT (different tile plan, different kernel
      template, same numbers), and
  (2) that window run is compared with the fp64 oracle element by element (tests/parity.py).
On top of that, properties that hold at any size are checked over the whole output: CSR offsets monotone and
consistent, tracks in particle order, towers in ascending id per event, EFlow = tracks ++ photons ++ neutral
hadrons with every neutral above its threshold, tower energies consistent.
"""
import importlib

import numpy as np
import pytest

wl = importlib.import_module("workloads.generate")

pytestmark = pytest.mark.gpu

WINDOWS = {2: 3, 3: 300, 4: 300}  # events per sampled window


def _slice_outputs(full, prefix, e0, e1):
    off = full[prefix + "_offsets"]
    a, b = int(off[e0]), int(off[e1])
    out = {prefix + "_offsets": off[e0:e1 + 1] - off[e0]}
    for k, v in full.items():
        if k.startswith(prefix + "_") and not k.endswith("offsets"):
            out[k] = v[a:b]
    return out


@pytest.mark.parametrize("cfg", [2, 3, 4])  # 4: the sparse (two-level bitmap) tiling
def test_full_size_sampled_parity_and_invariants(cfg):
    import paper_2606_26089_b200 as pd
    from gpu_util import run_gpu
    from parity import compare

    ev = wl.generate(cfg, None)
    seed = wl.CONFIGS[cfg]["seed"]
    card_name = wl.config_card(cfg)
    ne, n = ev.n_events, ev.n_particles
    full = run_gpu(card_name, ev, seed, debug=False)  # exactly what bench.py launches
    assert full["status_word"] == 0 and full["launches"] >= 1

    # ---- properties over the whole output
    for prefix in ("trk", "tow", "efl"):
        off = full[prefix + "_offsets"]
        assert off.shape[0] == ne + 1 and off[0] == 0 and np.all(np.diff(off) >= 0)
    n_trk, n_tow, n_efl = (int(full[p + "_offsets"][-1]) for p in ("trk", "tow", "efl"))
    assert 0 < n_trk <= n and 0 < n_tow <= n and n_trk < n_efl <= 2 * n
    # tracks: particle order, each inside its event
    src = full["trk_src"].astype(np.int64)
    assert np.all(np.diff(src) > 0)
    trk_ev = np.repeat(np.arange(ne), np.diff(full["trk_offsets"]))
    assert np.all(src >= ev.offsets[trk_ev]) and np.all(src < ev.offsets[trk_ev + 1])
    assert np.all(ev.charge[src] != 0) and np.array_equal(full["trk_pid"], ev.pid[src])
    assert np.all(full["trk_pt"] > 0) and np.all(np.isfinite(full["trk_E"]))
    # towers: ascending id inside an event, components above threshold or zero, E = Eem + Ehad
    tow_ev = np.repeat(np.arange(ne), np.diff(full["tow_offsets"]))
    key = tow_ev.astype(np.int64) * (1 << 20) + full["tow_tower"]
    assert np.all(np.diff(key) > 0)
    assert full["tow_tower"].min() >= 0 and full["tow_tower"].max() < pd.Card(card_name).n_towers
    em, had = full["tow_Eem"], full["tow_Ehad"]
    assert np.all((em == 0) | (em > 0.5)) and np.all((had == 0) | (had > 1.0)) and np.all(em + had > 0)
    assert np.array_equal(full["tow_E"], em + had)
    # eflow: per event tracks, then photons (4), then neutral hadrons (3); neutrals above threshold
    cls = full["efl_cls"]
    efl_ev = np.repeat(np.arange(ne), np.diff(full["efl_offsets"]))
    rank = np.where(cls <= 2, 0, np.where(cls == 4, 1, 2))
    assert np.all(np.diff(efl_ev.astype(np.int64) * 4 + rank) >= 0)
    assert int((cls <= 2).sum()) == n_trk
    assert np.all(full["efl_E"][cls == 4] > 0.5) and np.all(full["efl_E"][cls == 3] > 1.0)
    assert np.array_equal(np.diff(full["efl_offsets"]) - np.diff(full["trk_offsets"]) >= 0, np.ones(ne, dtype=bool))

    # ---- sampled windows: bitwise against a stand-alone GPU run, then against the oracle
    w = WINDOWS[cfg]
    flagged = overridden = 0
    for e0 in (0, ne // 2, ne - w):
        e1 = e0 + w
        sub = wl.slice_events(ev, e0, e1)
        win = run_gpu(card_name, sub, seed, event_base=e0, debug=True)
        assert win["status_word"] == 0
        p_base = int(ev.offsets[e0])
        for prefix in ("trk", "tow", "efl"):
            ref = _slice_outputs(full, prefix, e0, e1)
            for k, v in ref.items():
                got = win[k]
                if k == "trk_src":
                    v = v - p_base  # particle indices are per call
                elif k == "efl_src":
                    v = np.where(ref["efl_cls"] <= 2, v - p_base, v)
                assert got.tobytes() == np.ascontiguousarray(v).astype(got.dtype).tobytes(), (cfg, e0, k)
        rep = compare(card_name, sub, seed, win, event_base=e0)
        assert rep["unexcused"] == 0, rep["problems"][:10]
        flagged += rep["flagged_particles"]
        overridden += rep["overridden_particles"]
    print("cfg%d full size: %d particles, %d tracks, %d towers, %d eflow; sampled windows near-edge flagged %d, overridden %d"
          % (cfg, n, n_trk, n_tow, n_efl, flagged, overridden))
