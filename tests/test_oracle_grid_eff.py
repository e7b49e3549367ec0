"""Pins of the tower grid (O4) and the tracking efficiency (O3): SURVEY 8c.2 card table, 8c.5 P7."""
import math

import numpy as np
import pytest

import cards
import workloads as W
from workloads.generate import from_lists, particle
from oracle import pdo


def test_builtin_grids():
    cms, atlas, aleph = pdo.Card("cms_like"), pdo.Card("atlas_like"), pdo.Card("aleph_like")
    assert (cms.n_towers, cms.n_bins, cms.grid_coord) == (5904, 94, 0)
    assert (atlas.n_towers, atlas.n_bins, atlas.grid_coord) == (4096, 64, 0)
    assert (aleph.n_towers, aleph.n_bins, aleph.grid_coord) == (19320, 92, 1)
    # cms_like: 0.087 steps to 34 * 0.087 = 2.958, closing edge 3.0, 0.175 steps to 4.925, closing 5.0
    f = lambda x: float(np.float32(x))  # noqa: E731
    assert cms.edges[47] == 0.0 and cms.edges[48] == f(0.087) and cms.edges[81] == f(34 * 0.087)
    assert cms.edges[82] == 3.0 and cms.edges[83] == f(3.175) and cms.edges[93] == f(3 + 11 * 0.175)
    assert cms.edges[94] == 5.0 and cms.edges[0] == -5.0
    assert np.all(cms.edges == -cms.edges[::-1])
    assert list(cms.nphi[:12]) == [36] * 12 and list(cms.nphi[82:]) == [36] * 12 and set(cms.nphi[12:82]) == {72}
    assert np.all(np.diff(cms.edges) > 0) and np.all(np.diff(atlas.edges) > 0) and np.all(np.diff(aleph.edges) > 0)
    assert atlas.edges[0] == f(-3.2) and atlas.edges[64] == f(3.2) and atlas.edges[32] == 0.0
    assert set(atlas.nphi) == {64}
    assert aleph.edges[0] == f(math.acos(0.98)) and aleph.edges[92] == f(math.acos(-0.98))
    assert aleph.edges[46] == f(math.pi / 2) and set(aleph.nphi) == {210}
    for c in (cms, atlas, aleph):
        assert np.all(c.offset == np.concatenate([[0], np.cumsum(c.nphi)[:-1]]))
        assert np.all(c.edges == c.edges.astype(np.float32).astype(np.float64))  # reading A28


@pytest.mark.parametrize("name", ["cms_like", "atlas_like", "aleph_like"])
def test_tower_index_against_numpy_histogram_semantics(name):
    # half-open bins [lo, hi): numpy.searchsorted(side="right") - 1 is the library statement of that rule
    c = pdo.Card(name)
    rng = np.random.default_rng(3)
    lo, hi = c.edges[0], c.edges[-1]
    coord = rng.uniform(lo - 0.3, hi + 0.3, 20000)
    coord[:200] = rng.choice(c.edges, 200)           # exactly on edges
    phi = rng.uniform(-math.pi, math.pi, 20000)
    phi[:50] = math.pi
    phi[50:100] = -math.pi
    i = np.searchsorted(c.edges, coord, side="right") - 1
    inside = (coord >= lo) & (coord < hi)
    for k in range(coord.shape[0]):
        got = c.tower_index(coord[k], phi[k])
        if not inside[k]:
            assert got == -1
            continue
        n = int(c.nphi[i[k]])
        j = min(int(np.floor((phi[k] + math.pi) * n / (2 * math.pi) * (1 + 0.0))), n - 1)
        # the two ways of writing the phi bin may differ only exactly at a bin boundary
        assert got - c.offset[i[k]] in (j, max(j - 1, 0), min(j + 1, n - 1))
        e_c, p_c = c.tower_centre(got)
        w = 2 * math.pi / n
        assert abs(math.remainder(phi[k] - p_c, 2 * math.pi)) <= w / 2 + 1e-12
        mid = 0.5 * (c.edges[i[k]] + c.edges[i[k] + 1])
        assert abs(e_c - (mid if c.grid_coord == 0 else -math.log(math.tan(mid / 2)))) < 1e-12


def test_phi_pi_clamps_to_last_bin():
    c = pdo.Card("cms_like")
    assert c.tower_index(0.01, math.pi) == c.offset[47] + 71
    assert c.tower_index(0.01, -math.pi) == c.offset[47]
    assert c.tower_index(4.0, math.pi) == c.offset[87] + 35  # 3.875 <= 4.0 < 4.05
    assert c.tower_index(5.0, 0.0) == -1 and c.tower_index(-5.0, 0.0) == 0 + 18
    assert c.tower_index(float("inf"), 0.0) == -1 and c.tower_index(float("nan"), 0.0) == -1


def test_efficiency_rows_reading_A8():
    c = pdo.Card("cms_like")
    f = lambda x: float(np.float32(x))  # noqa: E731
    assert c.efficiency(5.0, 0.3) == (f(0.97), 0)
    assert c.efficiency(5.0, -1.2) == (f(0.97), 0)
    assert c.efficiency(5.0, 1.5) == (f(0.85), 1)        # |eta| = 1.5 belongs to the outer row
    assert c.efficiency(5.0, -2.4999) == (f(0.85), 1)
    assert c.efficiency(5.0, 2.5) == (0.0, -1)
    assert c.efficiency(1.0, 0.3) == (f(0.70), 2)        # pT = 1 exactly belongs to the 0.70 row
    assert c.efficiency(1.0000001, 0.3) == (f(0.97), 0)
    assert c.efficiency(0.5, 2.2) == (f(0.70), 2)
    assert c.efficiency(f(0.1), 0.3) == (0.0, -1)        # pT = 0.1f: strict lower edge
    assert c.efficiency(0.05, 0.0) == (0.0, -1)
    a = pdo.Card("aleph_like")
    assert a.efficiency(5.0, 0.3, 0.5)[1] == 0
    assert a.efficiency(5.0, 0.3, f(0.98)) == (0.0, -1)  # |cos theta| >= 0.98f (fp32 value promoted, A28)
    assert a.efficiency(5.0, 0.3, f(0.98) - 1e-9)[1] == 0


def _charged_sample(n, seed):
    rng = np.random.default_rng(seed)
    pt = np.exp(rng.uniform(math.log(0.05), math.log(100.0), n))
    eta = rng.uniform(-3.0, 3.0, n)
    phi = rng.uniform(-math.pi, math.pi, n)
    ev = [[particle(211, 1, pt[i], eta[i], phi[i], 0.13957039) for i in range(n)]]
    return from_lists(ev), pt, eta


def test_all_zero_and_all_one_efficiency(tmp_path):
    base = pdo.Card("cms_like")
    ev, pt, eta = _charged_sample(5000, 5)
    zero = cards.variant(tmp_path / "zero.card", base.edges, base.nphi, eff=[(0.0, "inf", 0.0, "inf", 0.0)])
    one = cards.variant(tmp_path / "one.card", base.edges, base.nphi, eff=[(0.1, "inf", 0.0, 2.5, 1.0)])
    for seed in (1, 2, 99):
        r0 = pdo.simulate(pdo.Card(zero), ev, seed)
        assert r0["trk_offsets"][-1] == 0 and not r0["dbg_accepted"].any()
        r1 = pdo.simulate(pdo.Card(one), ev, seed)
        ptf = np.hypot(ev.px.astype(np.float64), ev.py.astype(np.float64))
        etaf = np.arcsinh(ev.pz.astype(np.float64) / ptf)
        expect = (ptf > np.float32(0.1)) & (np.abs(etaf) < 2.5) & ((r1["dbg_status"] & 3) != 0)
        assert np.array_equal(r1["dbg_accepted"].astype(bool), expect)
        # invariant (iii): nothing is tracked beyond |eta| = 2.5 or at pT <= 0.1
        assert np.all(np.abs(r1["trk_eta"]) < 2.5)


def test_acceptance_frequency_per_row():
    c = pdo.Card("cms_like")
    ev = W.generate(0, 20000)
    r = pdo.simulate(c, ev, 77)
    charged = (ev.charge != 0) & ((r["dbg_status"] & 3) != 0)
    for row, eps in ((0, 0.97), (1, 0.85), (2, 0.70)):
        sel = charged & (r["dbg_eps_row"] == row)
        n = int(sel.sum())
        assert n > 20000
        frac = r["dbg_accepted"][sel].mean()
        assert abs(frac - eps) < 4.0 * math.sqrt(eps * (1 - eps) / n), (row, frac, n)
    assert not r["dbg_accepted"][(r["dbg_eps_row"] == -1)].any()
    assert not r["dbg_accepted"][ev.charge == 0].any()
