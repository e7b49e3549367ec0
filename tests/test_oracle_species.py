"""Pins of the per-species efficiency and track resolution (readings J1-J3; PAPER.md L653
"the efficiency with which CMS tracks charged hadrons ... CMSChargedHadronTrackingEfficiency", L655 "charged hadron
tracking, electron momentum smearing"): row semantics case by case, acceptance frequencies and smearing widths per
species on large samples, and that cards naming no species behave exactly as before.  CPU only."""
import importlib

import numpy as np

import cards
from oracle import pdo

wl = importlib.import_module("workloads.generate")

# (pt_lo, pt_hi, |eta|_lo, |eta|_hi, eps, species): electrons 0.9 / 0.5, muons 1.0 everywhere, hadrons the common rows
EFF = [(5.0, "inf", 0.0, 2.5, 0.9, 1), (0.5, 5.0, 0.0, 2.5, 0.5, 1), (0.1, "inf", 0.0, 2.4, 1.0, 2),
       (1.0, "inf", 0.0, 1.5, 0.97), (1.0, "inf", 1.5, 2.5, 0.85, 0), (0.1, 1.0, 0.0, 2.5, 0.70, 3)]
RES = {1: (0.03, 0.0), 2: (0.0, 2e-4)}   # electrons 3 % flat, muons b pT only; hadrons: the common (0.01, 1.5e-4)


def _card(tmp_path):
    b = pdo.Card("cms_like")
    return pdo.Card(cards.variant(tmp_path / "species.card", b.edges, b.nphi, eff=EFF, track_res_species=RES))


def test_row_semantics_per_species(tmp_path):
    c = _card(tmp_path)
    f = np.float32
    cases = [  # (pt, eta, species) -> (eps, row)
        ((10.0, 0.3, 1), (f(0.9), 0)), ((2.0, 0.3, 1), (f(0.5), 1)), ((5.0, 0.3, 1), (f(0.5), 1)),   # pt_hi inclusive
        ((0.3, 0.3, 1), (f(0.70), None)),    # no electron row: falls to ... the hadron-only row does not apply
        ((10.0, 0.3, 2), (f(1.0), 2)), ((0.3, 2.3, 2), (f(1.0), 2)), ((3.0, 2.45, 2), (f(0.85), 4)),  # muon beyond 2.4: common row
        ((10.0, 0.3, 3), (f(0.97), 3)), ((10.0, 2.0, 3), (f(0.85), 4)), ((0.5, 1.0, 3), (f(0.70), 5)),
        ((0.5, 1.0, 2), (f(1.0), 2)), ((0.05, 0.0, 3), (0.0, -1)), ((10.0, 2.6, 1), (0.0, -1)),
    ]
    for (pt, eta, sp), (eps, row) in cases:
        got = c.efficiency(pt, eta, 0.0, sp)
        if row is None:   # an electron of 0.3 GeV: rows 0, 1 (electron) fail on pT, row 5 is hadron-only -> nothing
            assert got == (0.0, -1)
        else:
            assert got == (float(eps), row), (pt, eta, sp, got)
    # the species-less entry point is the charged-hadron case, and a card without species is unchanged
    assert c.efficiency(10.0, 0.3) == c.efficiency(10.0, 0.3, 0.0, 3)
    b = pdo.Card("cms_like")
    for sp in (1, 2, 3):
        for pt, eta in ((10.0, 0.3), (0.5, 2.0), (3.0, 1.7), (0.05, 0.0)):
            assert b.efficiency(pt, eta, 0.0, sp) == b.efficiency(pt, eta)


def _sample(n_events=4000):
    ev = wl.generate(0, n_events)
    # make the lepton share large enough to measure: a third electrons, a third muons among the charged
    rng = np.random.default_rng(3)
    pid = ev.pid.copy()
    ch = ev.charge != 0
    r = rng.random(len(pid))
    pid[ch & (r < 1 / 3)] = 11
    pid[ch & (r >= 1 / 3) & (r < 2 / 3)] = 13
    return wl.Events(offsets=ev.offsets, **{k: (pid if k == "pid" else getattr(ev, k)) for k in ("pid", "charge", "px", "py", "pz", "E", "vx", "vy", "vz")})


def test_frequencies_and_widths_per_species(tmp_path):
    c = _card(tmp_path)
    ev = _sample()
    o = pdo.simulate(c, ev, 5)
    pt = np.hypot(ev.px.astype(np.float64), ev.py)
    aeta = np.abs(np.arcsinh(ev.pz / pt))
    acc = o["dbg_accepted"].astype(bool)
    alive = (o["dbg_status"] & 3) != 0
    ap = np.abs(ev.pid)
    sel = {
        "electron high": (ap == 11) & (pt > 5.2) & (aeta < 2.4), "electron low": (ap == 11) & (pt > 0.6) & (pt < 4.8) & (aeta < 2.4),
        "muon": (ap == 13) & (pt > 0.12) & (aeta < 2.3), "hadron central": (ap == 211) & (pt > 1.1) & (aeta < 1.4),
        "hadron soft": (ap == 211) & (pt > 0.12) & (pt < 0.95) & (aeta < 2.4),
    }
    want = {"electron high": 0.9, "electron low": 0.5, "muon": 1.0, "hadron central": 0.97, "hadron soft": 0.70}
    for k, m in sel.items():
        m = m & alive & (ev.charge != 0)
        n, p = int(m.sum()), want[k]
        assert n > 1500, (k, n)
        assert abs(acc[m].mean() - p) <= 4 * np.sqrt(max(p * (1 - p), 1e-9) / n) + 1e-12, (k, acc[m].mean())
    # smearing widths: std of pT'/pT = sqrt(a^2 + (b pT)^2) of the species (log-normal with that relative std)
    src = o["trk_src"]
    ratio = o["trk_pt"] / pt[src]
    tp, tpid = pt[src], np.abs(ev.pid[src])
    e = (tpid == 11)
    assert abs(ratio[e].std() - 0.03) < 0.03 * 4 / np.sqrt(2 * e.sum()) and abs(ratio[e].mean() - 1) < 4 * 0.03 / np.sqrt(e.sum())
    mu = (tpid == 13) & (tp > 50) & (tp < 100)
    z = (ratio[mu] - 1) / (2e-4 * tp[mu])
    assert mu.sum() > 300 and abs(z.std() - 1) < 4 / np.sqrt(2 * mu.sum())
    had = (tpid == 211) & (tp < 20)
    assert abs(ratio[had].std() - 0.01) < 0.01 * (4 / np.sqrt(2 * had.sum()) + 0.02)


def test_species_card_is_still_a_valid_chain(tmp_path):
    """The chain invariants hold with a per-species card (energy bookkeeping does not depend on the track tables)."""
    c = _card(tmp_path)
    ev = _sample(300)
    a, b = pdo.simulate(c, ev, 9), pdo.simulate(c, ev, 9)
    assert all(a[k].tobytes() == b[k].tobytes() for k in a)
    ref = pdo.simulate(pdo.Card("cms_like"), ev, 9)
    # same propagation and towers' true energies; different track lists
    assert np.array_equal(a["dbg_tower"], ref["dbg_tower"]) and np.array_equal(a["dtw_Eem_true"], ref["dtw_Eem_true"])
    assert int(a["trk_offsets"][-1]) != int(ref["trk_offsets"][-1])
