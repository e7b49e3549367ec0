"""Pins of the oracle's track impact parameters (Table 2; readings I1-I3 of
DESIGN.md section 14): hand-worked trajectories (tests/golden/impact_I1.txt), RK4 integration of the Lorentz force
forwards and backwards from the vertex with a search for the point nearest to the beam axis (independent of the
oracle's circle geometry), invariance along the helix (the exit point of pdo_propagate with the momentum turned by
the turning angle has the same d0 and z0), the straight-line limit, and the statistics / layout of the smearing."""
import importlib
import math

import numpy as np
import pytest

import cards
from conftest import read_table
from oracle import pdo

wl = importlib.import_module("workloads.generate")
KAPPA = float(np.float32(0.299792458))


def _card(tmp_path, **kw):
    b = pdo.Card("cms_like")
    return pdo.Card(cards.variant(tmp_path / "impact.card", b.edges, b.nphi, **kw))


def test_worked_trajectories(tmp_path):
    card = _card(tmp_path, bz=1.0)
    rows = read_table("impact_I1.txt")
    assert len(rows) == 7
    for r in rows:
        q = int(r[0])
        px, py, pz, vx, vy, vz, d0, z0 = (float(x) for x in r[1:])
        g = card.impact_true(q, px, py, pz, vx, vy, vz)
        assert g[0] == pytest.approx(d0, abs=2e-7), r  # the card's kappa is rounded to fp32: rho = 1 to 4e-8
        assert g[1] == pytest.approx(z0, abs=2e-7), r


def _rk4_pca(q, p, v, B, h=1e-3, span=8.0):
    """Integrate dx/ds = p/|p|, dp/ds = kappa q (p x B zhat)/|p| from the vertex in both directions of s and return
    (d0, z0) at the point of the path nearest to the z axis within half a turn: x t_y - y t_x with t the transverse
    direction of flight there, and z there."""
    pn = float(np.linalg.norm(p))

    def f(y):
        pp = y[3:]
        return np.concatenate([pp / pn, KAPPA * q * np.array([pp[1] * B, -pp[0] * B, 0.0]) / pn])

    def step(y, hh):
        k1 = f(y)
        k2 = f(y + 0.5 * hh * k1)
        k3 = f(y + 0.5 * hh * k2)
        k4 = f(y + hh * k3)
        return y + (hh / 6.0) * (k1 + 2 * k2 + 2 * k3 + k4)

    pt = math.hypot(p[0], p[1])
    # half a turn of the circle in path length: pi rho |p| / pT; stay inside it
    half_turn = math.pi * pt / (KAPPA * abs(q) * abs(B)) * pn / pt if q != 0 and B != 0 else span
    smax = min(span, 0.98 * half_turn)
    y0 = np.concatenate([np.array(v, dtype=np.float64), np.array(p, dtype=np.float64)])
    best = None
    for sign in (1.0, -1.0):
        y, s = y0.copy(), 0.0
        prev = (math.hypot(y[0], y[1]), y.copy())
        while s < smax:
            yn = step(y, sign * h)
            rn = math.hypot(yn[0], yn[1])
            if rn > prev[0] and s > 0:
                break
            prev, y, s = (rn, yn.copy()), yn, s + h
        # refine around the last point: ternary search of r(s) on [-h, h] about y
        lo, hi = -h, h
        for _ in range(80):
            m1, m2 = lo + (hi - lo) / 3, hi - (hi - lo) / 3
            r1 = np.hypot(*step(y, m1)[:2])
            r2 = np.hypot(*step(y, m2)[:2])
            if r1 < r2:
                hi = m2
            else:
                lo = m1
        yb = step(y, 0.5 * (lo + hi))
        rb = math.hypot(yb[0], yb[1])
        if best is None or rb < best[0]:
            best = (rb, yb)
    yb = best[1]
    tn = math.hypot(yb[3], yb[4])
    return (yb[0] * yb[4] - yb[1] * yb[3]) / tn, yb[2]


RK4_CASES = [
    # q, pT, eta, phi, vertex, Bz
    (1, 10.0, 0.5, 0.3, (0.001, -0.002, 0.01), 3.8),
    (-1, 10.0, 0.5, 0.3, (0.001, -0.002, 0.01), 3.8),
    (1, 0.9, 0.2, -2.0, (0.05, 0.02, -0.1), 3.8),     # strongly curved, displaced
    (-1, 0.8, 0.1, 0.0, (0.3, 0.2, 0.0), 3.8),        # far displaced: the circle does not enclose the axis
    (1, 0.3, -0.4, 0.7, (0.02, -0.01, -0.5), 3.8),    # rho = 0.26 m, the circle encloses the axis
    (2, 5.0, 1.2, 2.5, (-0.1, 0.05, 0.2), 3.8),       # doubly charged
    (1, 2.0, -0.7, 2.5, (0.01, -0.02, 0.1), -2.0),    # reversed field
    (-1, 1.5, 2.0, -1.0, (0.2, -0.3, 0.05), 1.5),
    (0, 3.0, 0.4, 1.1, (0.1, 0.2, -0.3), 3.8),        # neutral: straight line
]


@pytest.mark.parametrize("q,pt,eta,phi,v,B", RK4_CASES)
def test_geometry_against_rk4(tmp_path, q, pt, eta, phi, v, B):
    card = _card(tmp_path, bz=B)
    p = (pt * math.cos(phi), pt * math.sin(phi), pt * math.sinh(eta))
    d0, z0 = card.impact_true(q, *p, *v)
    rd0, rz0 = _rk4_pca(q, p, v, float(np.float32(B)))
    assert d0 == pytest.approx(rd0, abs=2e-8)
    assert z0 == pytest.approx(rz0, abs=2e-7)  # z moves by sinh(eta) per metre of transverse path
    # |d0| can never exceed the distance of the vertex itself
    assert abs(d0) <= math.hypot(v[0], v[1]) + 1e-12


def test_invariant_along_the_helix():
    """The impact parameters belong to the trajectory, not to the point it is described from: the calorimeter hit of
    pdo_propagate, with the momentum turned by s * alpha (reading A3), gives the same d0 and z0 (up to whole turns
    in z0, avoided by keeping alpha < pi)."""
    card = pdo.Card("cms_like")
    rng = np.random.default_rng(11)
    n_checked = 0
    for _ in range(400):
        q = int(rng.choice([-1, 1]))
        pt, eta, phi = 1.0 + 20 * rng.random(), rng.uniform(-1.2, 1.2), rng.uniform(-math.pi, math.pi)
        v = (rng.normal(0, 0.02), rng.normal(0, 0.02), rng.normal(0, 0.05))
        p = (pt * math.cos(phi), pt * math.sin(phi), pt * math.sinh(eta))
        hit = card.propagate(q, *p, *v)
        if hit["status"] & 3 == 0 or hit["alpha"] > 2.5:
            continue
        s = -np.sign(q * 3.8)
        ph2 = phi + s * hit["alpha"]
        p2 = (pt * math.cos(ph2), pt * math.sin(ph2), p[2])
        a = card.impact_true(q, *p, *v)
        b = card.impact_true(q, *p2, hit["x"], hit["y"], hit["z"])
        assert a[0] == pytest.approx(b[0], abs=1e-11)
        assert a[1] == pytest.approx(b[1], abs=1e-10)
        n_checked += 1
    assert n_checked > 300


def test_straight_line_limit_and_on_axis_vertices(tmp_path):
    weak = _card(tmp_path, bz=1e-6)   # rho = 3e6 m per GeV: the helix branch, indistinguishable from a line
    rng = np.random.default_rng(3)
    for _ in range(200):
        q = int(rng.choice([-2, -1, 1, 2]))
        px, py, pz = rng.normal(0, 3, 3)
        vx, vy, vz = rng.normal(0, 0.1, 3)
        pt = math.hypot(px, py)
        d0, z0 = weak.impact_true(q, px, py, pz, vx, vy, vz)
        # closed forms of the straight line (the familiar collider convention)
        assert d0 == pytest.approx((vx * py - vy * px) / pt, abs=1e-7)
        assert z0 == pytest.approx(vz - (vx * px + vy * py) / pt * pz / pt, abs=1e-6 * (1 + abs(pz) / pt))
    card = pdo.Card("cms_like")
    for _ in range(100):
        q = int(rng.choice([-1, 1]))
        px, py, pz = rng.normal(0, 3, 3)
        vz = rng.normal(0, 0.1)
        d0, z0 = card.impact_true(q, px, py, pz, 0.0, 0.0, vz)
        assert abs(d0) < 1e-12 * max(1.0, math.hypot(px, py)) and z0 == pytest.approx(vz, abs=1e-12)
    # mirror symmetry: reflecting the event in the x axis (y -> -y, py -> -py) and flipping the charge keeps the circle
    # and reverses the sense of d0
    for _ in range(100):
        q = int(rng.choice([-1, 1]))
        px, py, pz = rng.normal(0, 1, 3)
        vx, vy, vz = rng.normal(0, 0.1, 3)
        a = card.impact_true(q, px, py, pz, vx, vy, vz)
        b = card.impact_true(-q, px, -py, pz, vx, -vy, vz)
        assert a[0] == pytest.approx(-b[0], abs=1e-13) and a[1] == pytest.approx(b[1], abs=1e-12)


def _tracks_of(cfg, n_events):
    ev = wl.generate(cfg, n_events)
    o = pdo.simulate(pdo.Card(wl.config_card(cfg)), ev, wl.CONFIGS[cfg]["seed"], debug=False)
    return ev, o["trk_offsets"], o["trk_src"]


def test_smearing_statistics_layout_and_reproducibility():
    cfg = 0
    ev, off, src = _tracks_of(cfg, 400)
    card = pdo.Card(wl.config_card(cfg))
    d0_res, z0_res = (20e-6, 40e-6), (30e-6, 60e-6)
    r = pdo.track_impact(card, ev, off, src, d0_res, z0_res, seed=5)
    n = len(src)
    assert n > 5000
    pt = np.hypot(ev.px[src].astype(np.float64), ev.py[src].astype(np.float64))
    # reading I2: the errors are a (+) b / pT
    assert np.allclose(r["d0_err"], np.sqrt(d0_res[0] ** 2 + (d0_res[1] / pt) ** 2), rtol=1e-14)
    assert np.allclose(r["z0_err"], np.sqrt(z0_res[0] ** 2 + (z0_res[1] / pt) ** 2), rtol=1e-14)
    # the geometry is that of pdo_impact_true track by track
    for t in range(0, n, 97):
        i = int(src[t])
        g = card.impact_true(int(ev.charge[i]), ev.px[i], ev.py[i], ev.pz[i], ev.vx[i], ev.vy[i], ev.vz[i])
        assert (r["d0_true"][t], r["z0_true"][t]) == g
    # pulls: standard normal, d0 and z0 independent
    pd0 = (r["d0"] - r["d0_true"]) / r["d0_err"]
    pz0 = (r["z0"] - r["z0_true"]) / r["z0_err"]
    for pull in (pd0, pz0):
        assert abs(pull.mean()) < 4 / math.sqrt(n) and abs(pull.std() - 1) < 4 / math.sqrt(2 * n)
        assert abs((np.abs(pull) < 1).mean() - 0.6827) < 4 * math.sqrt(0.6827 * 0.3173 / n)
    assert abs(np.corrcoef(pd0, pz0)[0, 1]) < 4 / math.sqrt(n)
    # reading I3: stream 3, object = particle index within the event, words (0,1) and (2,3)
    e = 17
    t = int(off[e]) + 3
    i = int(src[t])
    w = pdo.rng_block(5, e, i - int(ev.offsets[e]), 3)
    assert r["d0"][t] == r["d0_true"][t] + r["d0_err"][t] * pdo.normal(w[0], w[1])
    assert r["z0"][t] == r["z0_true"][t] + r["z0_err"][t] * pdo.normal(w[2], w[3])
    # zero resolution: measured = true, errors 0; other seed: other values; event_base shifts the events
    z = pdo.track_impact(card, ev, off, src)
    assert np.array_equal(z["d0"], z["d0_true"]) and np.all(z["d0_err"] == 0) and np.all(z["z0_err"] == 0)
    other = pdo.track_impact(card, ev, off, src, d0_res, z0_res, seed=6)
    assert np.all(other["d0"] != r["d0"])
    cut = 150
    sub = wl.slice_events(ev, cut, 400)
    m, mt = int(ev.offsets[cut]), int(off[cut])
    r2 = pdo.track_impact(card, sub, off[cut:] - mt, src[mt:] - m, d0_res, z0_res, seed=5, event_base=cut)
    assert np.array_equal(r2["d0"], r["d0"][mt:]) and np.array_equal(r2["z0"], r["z0"][mt:])
