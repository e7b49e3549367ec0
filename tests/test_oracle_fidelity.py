"""Pins of the oracle's higher-card-fidelity steps (readings K1-K3 of DESIGN.md section 17):
eta-dependent calorimeter resolutions, the significance cut, tower positions smeared inside the cell.
Closed forms, limiting cases that reduce to the plain card, and statistics -- no formula of the oracle is retyped."""
import importlib
import math

import numpy as np
import pytest
import scipy.stats

import cards
from oracle import pdo

wl = importlib.import_module("workloads.generate")
P = wl.particle


def _photons(etas, E=40.0, n_events=1):
    """n_events identical events of photons from the origin, one per eta, all at phi = 0.3: each alone in its tower."""
    ev = [[P(22, 0, E / math.cosh(eta), eta, 0.3, 0.0) for eta in etas] for _ in range(n_events)]
    return wl.from_lists(ev)


def test_eta_rows_pick_the_row_of_the_tower_centre(tmp_path):
    b = pdo.Card("cms_like")
    # K1: rows that repeat the common line change nothing, bit for bit
    same = cards.variant(tmp_path / "same.card", b.edges, b.nphi, ecal_res_eta=[(0.0, 1.5, 0.007, 0.07, 0.35), (1.5, 9.0, 0.007, 0.07, 0.35)],
                         hcal_res_eta=[(0.0, 9.0, 0.05, 1.5, 0.0)])
    ev = wl.generate(0, 60)
    ref, got = pdo.simulate(b, ev, 3), pdo.simulate(pdo.Card(same), ev, 3)
    for k in ref:
        assert got[k].tobytes() == ref[k].tobytes(), k
    # a row with zero resolution for |eta_c| in [0.5, 1.5): towers there come out UNSMEARED (E' = E exactly: reading A21,
    # s <= 0), towers elsewhere are smeared; the interval is half open and is tested on the tower CENTRE, not on the hit
    path = cards.variant(tmp_path / "rows.card", b.edges, b.nphi, ecal_res_eta=[(0.5, 1.5, 0.0, 0.0, 0.0)], ecal_thr=0.0)
    # 0.087-wide bins: 0.51 lies in [0.435, 0.522), centre 0.4785 (outside the row although the hit is inside); 1.49 lies in
    # [1.479, 1.566), centre 1.5225 (outside although the hit is inside)
    etas = [0.02, 0.51, 0.53, 0.9, 1.45, 1.49, -0.7, -1.6, 2.5]
    ev = _photons(etas)
    o = pdo.simulate(pdo.Card(path), ev, 5)
    assert len(o["tow_tower"]) == len(etas)
    n_in = 0
    for k, eta in enumerate(etas):
        i = int(np.searchsorted(b.edges, np.float32(eta), side="right") - 1)
        centre = 0.5 * (float(b.edges[i]) + float(b.edges[i + 1]))
        sel = np.nonzero(np.abs(o["tow_eta"] - centre) < 1e-9)[0]
        assert sel.size == 1
        inside = 0.5 <= abs(centre) < 1.5
        n_in += inside
        assert (float(o["tow_E"][sel[0]]) == float(ev.E[k])) == inside, (eta, centre)
    assert n_in == 4


def test_eta_rows_give_the_rows_resolution(tmp_path):
    """Sample standard deviation of E'/E over many events = sigma_row(E)/E, row by row (4 sigma of the estimator)."""
    b = pdo.Card("cms_like")
    rows = [(0.0, 1.0, 0.10, 0.0, 0.0), (1.0, 2.0, 0.0, 0.632455532, 0.0), (2.0, 9.0, 0.0, 0.0, 4.0)]  # 10 %, 0.632/sqrt(E), 4 GeV
    path = cards.variant(tmp_path / "res.card", b.edges, b.nphi, hcal_res_eta=rows, hcal=(0.5, 0.0, 0.0), hcal_thr=0.0)
    n_ev, E = 4000, 40.0
    ev = wl.from_lists([[P(130, 0, E / math.cosh(eta), eta, 0.3, 0.0) for eta in (0.3, 1.5, 2.4)] for _ in range(n_ev)])
    o = pdo.simulate(pdo.Card(path), ev, 11)
    for k, eta in enumerate((0.3, 1.5, 2.4)):
        i = int(np.searchsorted(b.edges, np.float32(eta), side="right") - 1)
        centre = 0.5 * (float(b.edges[i]) + float(b.edges[i + 1]))
        sel = np.abs(o["tow_eta"] - centre) < 1e-9
        Ein = float(ev.E[k])
        ratio = o["tow_Ehad"][sel] / Ein
        assert ratio.shape[0] == n_ev
        rel = (0.10, 0.632455532 / math.sqrt(Ein), 4.0 / Ein)[k]  # C; S / sqrt(E); N / E
        assert abs(ratio.mean() - 1.0) < 4.0 * rel / math.sqrt(n_ev)
        assert abs(ratio.std() - rel) < 4.0 * rel / math.sqrt(2.0 * n_ev), (k, ratio.std(), rel)


def test_significance_cut_closed_forms(tmp_path):
    b = pdo.Card("cms_like")
    ev = wl.generate(0, 80)
    # sigma = 0.5 E': E' > n 0.5 E' <=> n < 2 -- just below keeps every HCAL component the plain card keeps, just above none
    for nsig, keeps in ((1.9, True), (2.1, False)):
        path = cards.variant(tmp_path / ("s%g.card" % nsig), b.edges, b.nphi, hcal=(0.5, 0.0, 0.0), hcal_nsigma=nsig)
        plain = cards.variant(tmp_path / ("p%g.card" % nsig), b.edges, b.nphi, hcal=(0.5, 0.0, 0.0))
        o, ref = pdo.simulate(pdo.Card(path), ev, 7), pdo.simulate(pdo.Card(plain), ev, 7)
        if keeps:
            for k in ref:
                assert o[k].tobytes() == ref[k].tobytes(), k
        else:
            assert (o["tow_Ehad"] == 0).all() and not (o["efl_cls"] == 3).any()
            assert np.array_equal(o["tow_Eem"], ref["tow_Eem"][ref["tow_Eem"] > 0])  # the ECAL side is untouched
    # sigma = S sqrt(E'): E' > n S sqrt(E') <=> E' > n^2 S^2 = 2.25 GeV for n = 3, S = 0.5 -- an energy threshold
    path = cards.variant(tmp_path / "sq.card", b.edges, b.nphi, hcal=(0.0, 0.5, 0.0), hcal_nsigma=3.0, hcal_thr=1.0)
    as_thr = cards.variant(tmp_path / "thr.card", b.edges, b.nphi, hcal=(0.0, 0.5, 0.0), hcal_thr=2.25)
    o, ref = pdo.simulate(pdo.Card(path), ev, 9), pdo.simulate(pdo.Card(as_thr), ev, 9)
    assert np.array_equal(o["tow_tower"], ref["tow_tower"]) and o["tow_Ehad"].tobytes() == ref["tow_Ehad"].tobytes()
    had = o["tow_Ehad"]
    assert (had[had > 0] > 2.25).all() and (o["tow_Ehad"] > 0).sum() < (pdo.simulate(pdo.Card(
        cards.variant(tmp_path / "no.card", b.edges, b.nphi, hcal=(0.0, 0.5, 0.0))), ev, 9)["tow_Ehad"] > 0).sum()
    # the neutral-hadron threshold itself stays hcal_thr = 1.0 (the cut acts on the tower component, reading K2)
    nh = o["efl_E"][o["efl_cls"] == 3]
    assert nh.size > 0 and nh.min() > 1.0


@pytest.mark.parametrize("name", ["cms_like", "aleph_like"])
def test_tower_positions_uniform_inside_the_cell(name, tmp_path):
    b = pdo.Card(name)
    path = cards.variant(tmp_path / "c.card", b.edges, b.nphi, base=name, smear_tower_center=1)
    card = pdo.Card(path)
    cfg = 0 if name == "cms_like" else 4
    ev = wl.generate(cfg, 400)
    o, ref = pdo.simulate(card, ev, 21), pdo.simulate(b, ev, 21)
    # K3 moves the reported position only: same towers, same energies, same neutrals
    for k in ("tow_tower", "tow_E", "tow_Eem", "tow_Ehad", "efl_cls", "efl_src", "efl_E", "trk_pt"):
        assert o[k].tobytes() == ref[k].tobytes(), k
    edges = np.asarray(b.edges, dtype=np.float64)
    nphi = np.asarray(b.nphi)
    off = np.concatenate([[0], np.cumsum(nphi)])
    i = np.searchsorted(off, o["tow_tower"], side="right") - 1
    j = o["tow_tower"] - off[i]
    coord = o["tow_eta"] if name == "cms_like" else 2.0 * np.arctan(np.exp(-o["tow_eta"]))
    u1 = (coord - edges[i]) / (edges[i + 1] - edges[i])
    u2 = (o["tow_phi"] + math.pi) / (2.0 * math.pi / nphi[i]) - j
    assert (u1 >= -1e-9).all() and (u1 < 1 + 1e-9).all() and (u2 >= -1e-9).all() and (u2 < 1 + 1e-9).all()
    assert scipy.stats.kstest(np.clip(u1, 0, 1), "uniform").pvalue > 1e-4
    assert scipy.stats.kstest(np.clip(u2, 0, 1), "uniform").pvalue > 1e-4
    assert abs(np.corrcoef(u1, u2)[0, 1]) < 4.0 / math.sqrt(u1.size)
    # ET and the neutrals' pT follow the reported position: pT = E / cosh(eta)
    assert np.allclose(o["tow_ET"], o["tow_E"] / np.cosh(o["tow_eta"]), rtol=1e-12)
    neu = o["efl_cls"] >= 3
    assert np.allclose(o["efl_pt"][neu], o["efl_E"][neu] / np.cosh(o["efl_eta"][neu]), rtol=1e-12)
    # one draw per (seed, event, tower): the Tower and its neutrals sit at the same point; another seed moves it
    tow_ev = np.repeat(np.arange(400), np.diff(o["tow_offsets"]))
    efl_ev = np.repeat(np.arange(400), np.diff(o["efl_offsets"]))
    pos = {(int(e), int(t)): (float(a), float(p)) for e, t, a, p in zip(tow_ev, o["tow_tower"], o["tow_eta"], o["tow_phi"])}
    n_checked = 0
    for e, t, a, p, c in zip(efl_ev, o["efl_src"], o["efl_eta"], o["efl_phi"], o["efl_cls"]):
        if c >= 3 and (int(e), int(t)) in pos:
            assert pos[(int(e), int(t))] == (float(a), float(p))
            n_checked += 1
    assert n_checked > 100
    other = pdo.simulate(card, ev, 22)
    assert not np.array_equal(other["tow_eta"][:50], o["tow_eta"][:50])
    # the library entry point gives the same position, and the centre when the card does not smear
    e0, t0 = int(tow_ev[5]), int(o["tow_tower"][5])
    assert pdo.tower_position(card, 21, e0, t0) == (float(o["tow_eta"][5]), float(o["tow_phi"][5]))
    assert pdo.tower_position(b, 21, e0, t0) == b.tower_centre(t0)


def _tracks(pid, q, etas, pt=20.0, n_events=1, mass=0.13957039):
    """n_events identical events of charged particles from the origin, one per eta, spread in phi"""
    return wl.from_lists([[P(pid, q, pt, eta, 0.1 + 0.3 * k, mass) for k, eta in enumerate(etas)] for _ in range(n_events)])


def test_track_resolution_rows_by_eta_and_species(tmp_path):
    """Reading K4: eta-dependent track resolution rows (first match in file order, optional species, half-open |eta| range of the
    TRUE momentum), falling back to the species' / the card's track_res line (J2)."""
    b = pdo.Card("cms_like")
    eff = [(0.1, "inf", 0.0, 2.5, 1.0)]
    # rows that repeat the common line change nothing, bit for bit
    same = cards.variant(tmp_path / "same.card", b.edges, b.nphi, track_res_eta=[(0.0, 1.0, 0.01, 1.5e-4), (1.0, 9.0, 0.01, 1.5e-4, 3)])
    ev = wl.generate(0, 60)
    ref, got = pdo.simulate(b, ev, 3), pdo.simulate(pdo.Card(same), ev, 3)
    for k in ref:
        assert got[k].tobytes() == ref[k].tobytes(), k
    # the selection function: first match wins, species rows apply to their species only, the range is [lo, hi)
    rows = [(0.5, 1.5, 0.0, 0.0), (1.0, 2.0, 0.07, 0.0, 2), (0.0, 9.0, 0.03, 2e-4, 1)]
    path = cards.variant(tmp_path / "rows.card", b.edges, b.nphi, eff=eff, track_res=(0.02, 1e-4), track_res_eta=rows)
    c = pdo.Card(path)
    f32 = lambda x: float(np.float32(x))  # noqa: E731
    mom = lambda eta, pt=10.0: (pt, 0.0, pt * math.sinh(eta))  # noqa: E731
    assert c.track_resolution(3, *mom(0.7)) == (0, 0.0, 0.0)                     # hadron inside row 0
    assert c.track_resolution(3, *mom(-1.2)) == (0, 0.0, 0.0)                    # |eta|: both signs
    assert c.track_resolution(2, *mom(1.2)) == (0, 0.0, 0.0)                     # row 0 precedes the muon row
    assert c.track_resolution(2, *mom(1.7)) == (1, f32(0.07), 0.0)               # muon row
    assert c.track_resolution(3, *mom(1.7)) == (-1, f32(0.02), f32(1e-4))        # no row for a hadron there: the common line
    assert c.track_resolution(1, *mom(1.7)) == (2, f32(0.03), f32(2e-4))         # electron row (any eta)
    assert c.track_resolution(1, *mom(0.7))[0] == 0                              # ... but row 0 comes first
    lo, hi = f32(0.5), f32(1.5)
    assert c.track_resolution(3, *mom(lo * (1 + 1e-9)))[0] == 0 and c.track_resolution(3, *mom(lo * (1 - 1e-9)))[0] == -1
    assert c.track_resolution(3, *mom(hi * (1 - 1e-9)))[0] == 0 and c.track_resolution(3, *mom(hi * (1 + 1e-9)))[0] == -1
    # through the chain: tracks in the zero-resolution row come out with pT' = pT exactly, the others are smeared
    etas = [0.2, 0.45, 0.55, 1.0, 1.45, 1.55, -0.8, -2.0]
    ev = _tracks(211, 1, etas)
    o = pdo.simulate(c, ev, 5)
    assert list(o["trk_src"]) == list(range(len(etas)))
    pt_true = np.hypot(ev.px.astype(np.float64), ev.py.astype(np.float64))
    for k, eta in enumerate(etas):
        assert (float(o["trk_pt"][k]) == pt_true[k]) == (0.5 <= abs(eta) < 1.5), eta


def test_track_resolution_rows_give_the_rows_width(tmp_path):
    """Sample std of pT'/pT over many events = the row's sigma_rel (a for b = 0; b pT for a = 0), row by row and by species."""
    b = pdo.Card("cms_like")
    rows = [(0.0, 1.0, 0.05, 0.0), (1.0, 2.0, 0.0, 1e-3), (2.0, 9.0, 0.12, 0.0, 2)]
    path = cards.variant(tmp_path / "w.card", b.edges, b.nphi, eff=[(0.1, "inf", 0.0, 2.5, 1.0)], track_res=(0.01, 0.0), track_res_eta=rows)
    n_ev, pt = 4000, 30.0
    for pid, mass, want in ((211, 0.13957039, (0.05, 1e-3 * pt, 0.01)), (13, 0.1056584, (0.05, 1e-3 * pt, 0.12))):
        ev = _tracks(pid, 1, (0.4, 1.5, 2.3), pt=pt, n_events=n_ev, mass=mass)
        o = pdo.simulate(pdo.Card(path), ev, 17)
        assert o["trk_src"].shape[0] == 3 * n_ev
        ratio = (o["trk_pt"] / np.hypot(ev.px.astype(np.float64), ev.py.astype(np.float64))[o["trk_src"]]).reshape(n_ev, 3)
        for k in range(3):
            assert abs(ratio[:, k].mean() - 1.0) < 4.0 * want[k] / math.sqrt(n_ev)
            assert abs(ratio[:, k].std() - want[k]) < 4.0 * want[k] / math.sqrt(2.0 * n_ev), (pid, k, ratio[:, k].std(), want[k])


def test_weighted_eflow_limits_and_closed_forms(tmp_path):
    """Reading K5 (card key eflow_weighted): the EFlow entries of the tracks of a tower component whose neutral is not emitted are
    rescaled to the inverse-variance weighted mean of the track and the calorimeter measurement.  Pinned on the textbook
    properties of that mean and on limits in which the result has a closed form -- not on the formula."""
    # the weight function: equal variances -> arithmetic mean; a perfect side wins; nothing to combine -> 1
    assert pdo.eflow_weight(10.0, 4.0, 14.0, 2.0) == pytest.approx(1.2, rel=1e-15)     # (10 + 14) / 2 over 10
    assert pdo.eflow_weight(10.0, 1.0, 14.0, 3.0) == pytest.approx((10 * 9 + 14 * 1) / 10.0 / 10.0, rel=1e-15)  # weights 9 : 1
    assert pdo.eflow_weight(10.0, 0.0, 12.0, 1.0) == 1.0 and pdo.eflow_weight(10.0, 4.0, 12.0, 0.0) == pytest.approx(1.2, rel=1e-15)
    assert pdo.eflow_weight(10.0, 4.0, 0.0, 1.0) == 1.0 and pdo.eflow_weight(0.0, 0.0, 5.0, 1.0) == 1.0 and pdo.eflow_weight(10.0, 0.0, 12.0, 0.0) == 1.0
    for T, V, E, s in ((10.0, 4.0, 14.0, 1.0), (50.0, 0.3, 20.0, 7.0), (3.0, 9.0, 3.5, 0.1)):
        m = T * pdo.eflow_weight(T, V, E, s)
        assert min(T, E) <= m <= max(T, E)                                   # a mean lies between its arguments
        assert abs(m - (T if V < s * s else E)) <= abs(m - (E if V < s * s else T))  # ... nearer the better measurement

    b = pdo.Card("cms_like")
    eff = [(0.1, "inf", 0.0, 2.5, 1.0)]
    etas = [-1.9, -1.2, -0.6, 0.1, 0.7, 1.3, 2.0]   # distinct towers, all inside the tracker acceptance
    n_ev = 3000
    # pions of 40 GeV each; HCAL threshold 20 GeV: the component (E' ~ 40 +- 4) is always kept, its neutral excess (E' - T ~ 0 +- 5.7)
    # practically never emitted
    ev = wl.from_lists([[P(211, 1, 40.0 / math.cosh(eta), eta, 0.2 + 0.4 * k, 0.13957039) for k, eta in enumerate(etas)] for _ in range(n_ev)])
    E_true = ev.E.astype(np.float64)

    def run(**kw):
        """oracle outputs with the EFlow arrays cut down to the entries of the tracks (classes 0-2: same order as the Track collection)"""
        args = dict(eff=eff, track_res=(0.1, 0.0), hcal=(0.1, 0.0, 0.0), hcal_thr=20.0, eflow_weighted=1)
        args.update(kw)
        o = pdo.simulate(pdo.Card(cards.variant(tmp_path / ("w%d.card" % len(list(tmp_path.iterdir()))), b.edges, b.nphi, **args)), ev, 31)
        rows = o["efl_cls"] < 3
        assert rows.sum() == len(o["trk_E"]) == len(E_true) and (~rows).sum() < 30   # (a neutral is emitted in a handful of cases)
        return dict(o, **{k: o[k][rows] for k in ("efl_E", "efl_pt", "efl_eta", "efl_phi")})

    off = run(eflow_weighted=0)
    assert off["efl_E"].tobytes() == off["trk_E"].tobytes()                  # without the key: EFlow tracks = the tracks
    # 10 % + 10 %: the combination resolves E to 10 % / sqrt(2) (textbook), better than either alone; tracks and towers unchanged
    o = run()
    assert o["trk_E"].tobytes() == off["trk_E"].tobytes() and o["tow_E"].tobytes() == off["tow_E"].tobytes()
    assert len(o["tow_Ehad"]) == len(E_true)
    r_trk, r_cal, r_w = o["trk_E"] / E_true, o["tow_Ehad"] / E_true, o["efl_E"] / E_true
    assert abs(r_trk.std() - 0.1) < 0.004 and abs(r_cal.std() - 0.1) < 0.004
    assert abs(r_w.std() - 0.1 / math.sqrt(2.0)) < 0.004, r_w.std()
    assert np.all(r_w >= np.minimum(r_trk, r_cal) - 1e-6) and np.all(r_w <= np.maximum(r_trk, r_cal) + 1e-6)
    assert np.allclose(o["efl_pt"] / o["trk_pt"], o["efl_E"] / o["trk_E"], rtol=1e-6)   # pT and E by the same factor; eta, phi untouched
    assert o["efl_eta"].tobytes() == o["trk_eta"].tobytes() and o["efl_phi"].tobytes() == o["trk_phi"].tobytes()
    # a perfect tracker ignores the calorimeter; a perfect calorimeter overrules the tracker: EFlow E = the deposited energy
    o = run(track_res=(0.0, 0.0))
    assert o["efl_E"].tobytes() == o["trk_E"].tobytes()
    o = run(hcal=(0.0, 0.0, 0.0))
    assert np.allclose(o["efl_E"], E_true, rtol=2e-7) and not np.allclose(o["trk_E"], E_true, rtol=1e-3)
    # the component cut away (here: by an impossible significance cut): no calorimeter information, the tracks stay
    o = run(hcal_nsigma=1e6)
    assert not o["tow_Ehad"].any() and o["efl_E"].tobytes() == o["trk_E"].tobytes()
    # where the neutral IS emitted the tracks stay as they are: a K0L of 200 GeV joins every pion's tower
    ev2 = wl.from_lists([[p for k, eta in enumerate(etas) for p in (P(211, 1, 20.0, eta, 0.2 + 0.4 * k, 0.13957039), P(130, 0, 200.0 / math.cosh(eta), eta, 0.2 + 0.4 * k, 0.497611))]
                         for _ in range(50)])
    c2 = pdo.Card(cards.variant(tmp_path / "emit.card", b.edges, b.nphi, eff=eff, track_res=(0.1, 0.0), hcal=(0.1, 0.0, 0.0), eflow_weighted=1))
    o = pdo.simulate(c2, ev2, 31)
    nt = len(o["trk_E"])
    assert (o["efl_cls"] == 3).sum() > 300 and nt == 50 * len(etas)
    emitted = set(zip(np.repeat(np.arange(50), np.diff(o["efl_offsets"]))[o["efl_cls"] == 3].tolist(), o["efl_src"][o["efl_cls"] == 3].tolist()))
    trk_ev = np.repeat(np.arange(50), np.diff(o["trk_offsets"]))
    dbg_tower = o["dbg_tower"][o["trk_src"]]
    trk_rows = np.nonzero(o["efl_cls"] < 3)[0]
    for k in range(nt):
        same = o["efl_E"][trk_rows[k]] == o["trk_E"][k]
        assert same == ((int(trk_ev[k]), int(dbg_tower[k])) in emitted), k
    # several tracks in one component share the factor; a muon (no deposit) is never touched
    ev3 = wl.from_lists([[P(211, 1, 20.0, 0.30, 0.50, 0.13957039), P(-211, -1, 35.0, 0.30, 0.50, 0.13957039), P(13, -1, 30.0, 0.30, 0.50, 0.1056584),
                          P(211, 1, 40.0, -1.0, 2.0, 0.13957039)] for _ in range(40)])
    o = pdo.simulate(pdo.Card(cards.variant(tmp_path / "multi.card", b.edges, b.nphi, eff=eff, track_res=(0.1, 0.0), hcal=(0.1, 0.0, 0.0), hcal_thr=30.0,
                                            eflow_weighted=1)), ev3, 31)
    assert (o["efl_cls"] < 3).sum() == 160 == len(o["trk_E"])
    f = (o["efl_E"][o["efl_cls"] < 3] / o["trk_E"]).reshape(40, 4)
    t = o["dbg_tower"].reshape(40, 4)
    assert (t[:, 0] == t[:, 1]).all() and (t[:, 0] != t[:, 3]).all()      # the two pions of 20 and 35 GeV hit one tower
    assert np.allclose(f[:, 0], f[:, 1], rtol=1e-12) and not np.allclose(f[:, 0], f[:, 3], rtol=1e-3)
    assert np.all(f[:, 2] == 1.0) and np.all(np.abs(f[:, 0] - 1.0) > 1e-6) and np.all(np.abs(f[:, 3] - 1.0) > 1e-6)


def test_separate_ecal_and_hcal_grids(tmp_path):
    """Reading K6: a grid of its own for the HCAL (card keys hcal_edges / hcal_nphi).  Tower ids: the ECAL grid's towers first,
    then the HCAL grid's; a deposit is looked up in the grid of its section.  Pinned on closed-form tower ids of uniform grids
    and on the one-grid oracle run with a perfect detector."""
    a = pdo.Card("atlas_like")           # ECAL: 64 eta bins of 0.1 over |eta| < 3.2, 64 phi bins: 4,096 towers
    he = [np.float32(-3.2 + 0.2 * k) if k < 32 else np.float32(3.2) for k in range(33)]
    he = [-float(np.float32(0.2 * k)) for k in range(16, 0, -1)] + [float(np.float32(0.2 * k)) for k in range(17)]   # 32 bins of 0.2
    hn = [32] * 32
    perfect = dict(eff=[(0.1, "inf", 0.0, 2.5, 1.0)], track_res=(0.0, 0.0), ecal=(0.0, 0.0, 0.0), hcal=(0.0, 0.0, 0.0))
    dual = pdo.Card(cards.variant(tmp_path / "dual.card", a.edges, a.nphi, base="atlas_like", hcal_edges=he, hcal_nphi=hn, **perfect))
    one = pdo.Card(cards.variant(tmp_path / "one.card", a.edges, a.nphi, base="atlas_like", **perfect))
    assert (dual.n_towers, one.n_towers) == (4096 + 1024, 4096)
    e, n, base = dual.hcal_grid()
    assert base == 4096 and len(n) == 32 and np.allclose(e, he) and one.hcal_grid() is None
    # closed-form ids of the two uniform grids (hits of neutral particles from the origin are at their own eta, phi)
    id_e = lambda eta, phi: 64 * int(math.floor((eta + 3.2) / 0.1)) + int(math.floor((phi + math.pi) / (2 * math.pi / 64)))   # noqa: E731
    id_h = lambda eta, phi: 4096 + 32 * int(math.floor((eta + 3.2) / 0.2)) + int(math.floor((phi + math.pi) / (2 * math.pi / 32)))  # noqa: E731
    pts = [(0.05, 0.3), (-1.234, -2.5), (2.17, 1.0), (-3.15, 3.0), (1.05, -0.02), (0.31, 2.2)]
    for eta, phi in pts:
        assert dual.tower_index(eta, phi, det=0) == id_e(eta, phi) == one.tower_index(eta, phi, det=1)   # one grid: det does not matter
        assert dual.tower_index(eta, phi, det=1) == id_h(eta, phi)
        ec, pc = dual.tower_centre(id_h(eta, phi))
        assert abs(ec - (-3.2 + 0.2 * (math.floor((eta + 3.2) / 0.2) + 0.5))) < 1e-6
        assert abs(pc - (-math.pi + (math.floor((phi + math.pi) / (2 * math.pi / 32)) + 0.5) * 2 * math.pi / 32)) < 1e-12
    assert dual.tower_index(3.3, 0.0, det=1) == -1 and dual.tower_index(-3.21, 0.0, det=0) == -1
    # through the chain: a photon, a K0L and a muon in each of the directions above
    ev = wl.from_lists([[p for eta, phi in pts for p in (P(22, 0, 10.0, eta, phi, 0.0), P(130, 0, 12.0, eta, phi, 0.497611), P(13, 1, 500.0, eta, phi, 0.1056584))]])
    o = pdo.simulate(dual, ev, 3)
    want_e, want_h = sorted(id_e(*p) for p in pts), sorted(id_h(*p) for p in pts)
    assert list(o["tow_tower"]) == want_e + want_h                       # ascending ids: the ECAL grid's towers first
    k = len(pts)
    assert np.all(o["tow_Ehad"][:k] == 0) and np.all(o["tow_Eem"][:k] > 0) and np.all(o["tow_Eem"][k:] == 0) and np.all(o["tow_Ehad"][k:] > 0)
    assert list(o["dbg_tower"][0::3]) == [id_e(*p) for p in pts] and list(o["dbg_tower"][1::3]) == [id_h(*p) for p in pts]
    mu = o["dbg_tower"][2::3]                                            # 500 GeV muons barely bend: the K0L's HCAL tower or a neighbour; no deposit
    assert np.all(mu >= 4096) and len(o["tow_tower"]) == 2 * k
    assert list(o["efl_src"][o["efl_cls"] == 4]) == want_e and list(o["efl_src"][o["efl_cls"] == 3]) == want_h
    # a perfect detector on realistic events: per event the same energy in each section as with one grid, the HCAL deposits
    # re-binned: summing the one-grid card's HCAL energies over the coarse cells gives the dual card's HCAL towers
    evs = wl.generate(3, 40)
    od, oo = pdo.simulate(dual, evs, 9), pdo.simulate(one, evs, 9)
    assert od["trk_pt"].tobytes() == oo["trk_pt"].tobytes()
    for ev_i in range(40):
        d = slice(int(od["tow_offsets"][ev_i]), int(od["tow_offsets"][ev_i + 1]))
        s = slice(int(oo["tow_offsets"][ev_i]), int(oo["tow_offsets"][ev_i + 1]))
        td, ts = od["tow_tower"][d], oo["tow_tower"][s]
        em_d = {int(t): float(x) for t, x in zip(td, od["tow_Eem"][d]) if t < 4096}
        em_s = {int(t): float(x) for t, x in zip(ts, oo["tow_Eem"][s]) if x > 0}
        assert em_d == em_s
        coarse = {}
        for t, x in zip(ts, oo["tow_Ehad"][s]):
            if x > 0:
                ie, ip = divmod(int(t), 64)
                key = 4096 + 32 * (ie // 2) + ip // 2
                coarse[key] = coarse.get(key, 0.0) + float(x)
        had_d = {int(t): float(x) for t, x in zip(td, od["tow_Ehad"][d]) if t >= 4096}
        # (the one-grid card applies the 1 GeV threshold per fine tower, the dual card per coarse tower: compare what passes both)
        for key, x in had_d.items():
            assert key in coarse and coarse[key] <= x * (1 + 1e-12) + 1e-9
        assert set(coarse) <= set(had_d)
    # K3 on a dual card: the reported position of an HCAL tower lies in its own (coarse) cell
    sm = pdo.Card(cards.variant(tmp_path / "dual_sm.card", a.edges, a.nphi, base="atlas_like", hcal_edges=he, hcal_nphi=hn, smear_tower_center=1, **perfect))
    os_ = pdo.simulate(sm, evs, 9)
    hsel = os_["tow_tower"] >= 4096
    loc = os_["tow_tower"][hsel] - 4096
    u1 = (os_["tow_eta"][hsel] + 3.2) / 0.2 - loc // 32
    u2 = (os_["tow_phi"][hsel] + math.pi) / (2 * math.pi / 32) - loc % 32
    assert hsel.sum() > 300 and (u1 >= -1e-6).all() and (u1 < 1 + 1e-6).all() and (u2 >= -1e-9).all() and (u2 < 1 + 1e-9).all()
    assert scipy.stats.kstest(np.clip(u1, 0, 1), "uniform").pvalue > 1e-4
