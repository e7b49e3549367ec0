"""Pins of the oracle's truth-level event features (Table 2 "H_T, E_T^miss values for Truth and PFlow
collections"; readings T1, T2 of DESIGN.md section 15): closed forms, a hand-worked event, momentum balance (the
visible recoil equals the neutrinos' transverse momentum), a numpy re-derivation on the synthetic workloads, and
agreement with the PFlow-side definition (pdo_event_features) on the same objects given as (pT, phi)."""
import importlib
import math

import numpy as np
import pytest

from oracle import pdo

wl = importlib.import_module("workloads.generate")


def _ev(events):
    return wl.from_lists(events)


def test_closed_forms_and_worked_event():
    P = wl.particle
    ev = _ev([
        [P(211, 1, 10.0, 0.3, 0.0)],                                       # one particle: MET = pT, opposite to it
        [P(211, 1, 5.0, 0.1, 1.0), P(-211, -1, 5.0, -2.0, 1.0 - math.pi)],  # back to back: MET 0, H_T 10
        [],                                                                 # empty event
        [P(22, 0, 3.0, 0.0, 0.0), P(22, 0, 4.0, 1.0, math.pi / 2)],         # 3-4-5 triangle
        [P(11, -1, 20.0, 0.5, 0.3), P(-12, 0, 7.0, 1.5, 2.0), P(14, 0, 2.0, 0.0, -1.0), P(16, 0, 1.0, 0.0, 0.5)],
    ])
    r = pdo.truth_features(ev)
    assert r["ht"] == pytest.approx([10, 10, 0, 7, 20], abs=1e-5)
    assert r["met"] == pytest.approx([10, 0, 0, 5, 20], abs=1e-5)
    assert (r["met_x"][0], r["met_y"][0]) == pytest.approx((-10, 0), abs=1e-6)
    assert (r["met_x"][3], r["met_y"][3]) == pytest.approx((-3, -4), abs=1e-6)
    assert (r["met_x"][4], r["met_y"][4]) == pytest.approx((-20 * math.cos(0.3), -20 * math.sin(0.3)), abs=1e-5)
    # T2 off: neutrinos count like everything else
    a = pdo.truth_features(ev, skip_neutrinos=False)
    assert a["ht"][4] == pytest.approx(30, abs=1e-5) and np.array_equal(a["ht"][:4], r["ht"][:4])


def test_visible_recoil_balances_the_neutrinos():
    rng = np.random.default_rng(8)
    events = []
    for _ in range(50):
        n = int(rng.integers(3, 40))
        parts = []
        for _ in range(n):
            pid = int(rng.choice([211, -211, 22, 130, 11, -13, 12, -14, 16]))
            parts.append(wl.particle(pid, 0 if abs(pid) in (22, 130, 12, 14, 16) else int(np.sign(pid)), float(rng.uniform(0.2, 50)),
                                     float(rng.uniform(-3, 3)), float(rng.uniform(-math.pi, math.pi))))
        # close the event: one more visible particle that balances the transverse momentum
        sx, sy = sum(p[2] for p in parts), sum(p[3] for p in parts)
        parts.append(wl.particle(211, 1, math.hypot(sx, sy), 0.0, math.atan2(-sy, -sx)))
        events.append(parts)
    ev = _ev(events)
    r = pdo.truth_features(ev)
    nu = np.isin(np.abs(ev.pid), (12, 14, 16))
    e_of = np.repeat(np.arange(ev.n_events), np.diff(ev.offsets))
    nx = np.bincount(e_of, weights=np.where(nu, ev.px, 0).astype(np.float64), minlength=ev.n_events)
    ny = np.bincount(e_of, weights=np.where(nu, ev.py, 0).astype(np.float64), minlength=ev.n_events)
    # total transverse momentum is zero (to fp32 rounding of the inputs), so -sum(visible) = sum(neutrinos)
    assert np.allclose(r["met_x"], nx, atol=2e-4) and np.allclose(r["met_y"], ny, atol=2e-4)
    assert np.all(pdo.truth_features(ev, skip_neutrinos=False)["met"] < 2e-4)


@pytest.mark.parametrize("cfg", [0, 3, 4])
def test_numpy_rederivation_and_pflow_side_definition(cfg):
    ev = wl.generate(cfg, 300)
    r = pdo.truth_features(ev)
    vis = ~np.isin(np.abs(ev.pid), (12, 14, 16))
    e_of = np.repeat(np.arange(ev.n_events), np.diff(ev.offsets))
    px, py = ev.px.astype(np.float64), ev.py.astype(np.float64)
    assert np.allclose(r["ht"], np.bincount(e_of[vis], weights=np.hypot(px, py)[vis], minlength=ev.n_events), rtol=1e-13)
    assert np.allclose(r["met_x"], -np.bincount(e_of[vis], weights=px[vis], minlength=ev.n_events), rtol=1e-12, atol=1e-12)
    assert np.allclose(r["met"], np.hypot(r["met_x"], r["met_y"]), rtol=1e-14)
    assert np.all(r["met"] <= r["ht"] * (1 + 1e-12))
    # the same objects handed to the PFlow-side routine as (pT, phi): same H_T and E_T^miss (F1, F2 of section 10)
    pt, phi = np.hypot(px, py).astype(np.float32), np.arctan2(py, px).astype(np.float32)
    a = pdo.truth_features(ev, skip_neutrinos=False)
    f = pdo.event_features(ev.offsets, np.zeros(len(pt), np.int8), pt, np.zeros(len(pt), np.float32), phi)
    assert np.allclose(f["ht"], a["ht"], rtol=1e-6) and np.allclose(f["met"], a["met"], atol=1e-5 * a["ht"].max())
    # batching: events are independent
    b = pdo.truth_features(wl.slice_events(ev, 100, 300))
    assert np.array_equal(b["ht"], r["ht"][100:]) and np.array_equal(b["met"], r["met"][100:])
