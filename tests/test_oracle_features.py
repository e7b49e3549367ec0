"""Pins of the oracle's event features and lepton isolation (oracle/pd_oracle.c pdo_event_features; PAPER.md
L119-127 Eq. 1): a hand-worked event, closed forms, invariants, and an independent brute-force numpy
re-derivation.  CPU only."""
import os

import numpy as np

from oracle import pdo

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def _f1():
    rows = [l.split("#")[0].replace("|", " ").split() for l in open(os.path.join(GOLD, "features_F1.txt"))]
    return np.array([[float(x) for x in r] for r in rows if r])


def test_worked_event_F1():
    t = _f1()
    cls, pt, eta, phi = t[:, 0].astype(np.int8), t[:, 1], t[:, 2], t[:, 3]
    r = pdo.event_features([0, len(t)], cls, pt, eta, phi, 0.4, 0.0)
    assert np.allclose(r["iso_charged"], t[:, 4], atol=1e-6) and np.allclose(r["iso_neutral"], t[:, 5], atol=1e-6)
    assert np.allclose(r["iso_photon"], t[:, 6], atol=1e-6) and np.allclose(r["r_iso"], t[:, 7], atol=1e-7)
    assert abs(r["ht"][0] - 51.0) < 1e-5 and np.all(r["iso_amb"] == 0)
    r = pdo.event_features([0, len(t)], cls, pt, eta, phi, 0.4, 0.05)
    assert np.allclose(r["iso_photon"], t[:, 8], atol=1e-6) and np.allclose(r["r_iso"], t[:, 9], atol=1e-7)
    assert np.allclose(r["iso_charged"], t[:, 4], atol=1e-6)


def test_closed_forms_ht_met():
    # one object: MET = pT, pointing opposite to it
    r = pdo.event_features([0, 1], [0], [7.0], [1.2], [0.5])
    assert abs(r["ht"][0] - 7) < 1e-12 and abs(r["met"][0] - 7) < 1e-6
    assert abs(r["met_x"][0] + 7 * np.cos(0.5)) < 1e-9 and abs(r["met_y"][0] + 7 * np.sin(0.5)) < 1e-9
    # n equal objects evenly spread in phi balance: MET = 0, H_T = n pT; along +x only: MET = (-H_T, 0)
    for n in (2, 3, 8, 360):
        phi = -np.pi + 2 * np.pi * (np.arange(n) + 0.5) / n
        r = pdo.event_features([0, n], np.zeros(n), np.full(n, 2.5), np.zeros(n), phi)
        assert abs(r["ht"][0] - 2.5 * n) < 1e-9 and r["met"][0] < 1e-5 * n
    r = pdo.event_features([0, 3], [0, 3, 4], [1.0, 2.0, 4.0], [0.1, -2, 3], [0.0, 0.0, 0.0])
    assert abs(r["met_x"][0] + 7) < 1e-12 and abs(r["met_y"][0]) < 1e-12 and abs(r["met"][0] - 7) < 1e-12
    # empty events and CSR bookkeeping: features of event e only see its own objects
    r = pdo.event_features([0, 0, 2, 2, 3], [0, 0, 0], [1.0, 2.0, 5.0], [0, 0, 0], [0.0, np.pi / 2, 0.0])
    assert r["ht"].tolist() == [0.0, 3.0, 0.0, 5.0] and r["met"][0] == 0 and abs(r["met"][1] - np.sqrt(5)) < 1e-6


def test_isolation_special_cases():
    # a lone lepton is perfectly isolated; non-leptons always get zeros
    r = pdo.event_features([0, 2], [1, 0], [10.0, 3.0], [0.0, 2.0], [0.0, 0.0])
    assert r["r_iso"].tolist() == [0.0, 0.0] and r["iso_charged"].tolist() == [0.0, 0.0]
    # two leptons see each other (charged term), not themselves
    r = pdo.event_features([0, 2], [1, 2], [10.0, 5.0], [0.0, 0.1], [0.0, 0.1])
    assert np.allclose(r["iso_charged"], [5.0, 10.0]) and np.allclose(r["r_iso"], [0.5, 2.0])
    # strict cone, scan across the edge; the near-edge sum flags only the object within 1e-6 of it
    for d, inside in ((0.39, True), (0.3999, True), (0.4001, False), (0.41, False)):
        r = pdo.event_features([0, 2], [2, 3], [10.0, 4.0], [0.0, d], [1.0, 1.0])
        assert (r["iso_neutral"][0] == 4.0) == inside and r["iso_amb"][0] == 0.0
    r = pdo.event_features([0, 2], [2, 3], [10.0, 4.0], [0.0, 0.4], [1.0, 1.0])
    assert r["iso_amb"][0] == 4.0
    # the cone is in (eta, phi), phi periodic; an object in another event never counts
    r = pdo.event_features([0, 2, 3], [1, 4, 4], [8.0, 2.0, 50.0], [0.0, 0.0, 0.0], [3.1, -3.1, 3.1])
    assert np.allclose(r["iso_photon"], [2.0, 0.0, 0.0]) and abs(r["r_iso"][0] - 0.25) < 1e-9
    # FSR reading F4: photons closer than fsr_dr are left out of the photon term only
    r = pdo.event_features([0, 3], [1, 4, 0], [8.0, 2.0, 1.0], [0.0, 0.01, 0.01], [0.0, 0.0, 0.0], 0.4, 0.05)
    assert r["iso_photon"][0] == 0.0 and r["iso_charged"][0] == 1.0


def _brute(offsets, cls, pt, eta, phi, dr_max, fsr_dr):
    """Independent re-derivation: dense pairwise matrices per event, complex phases for the phi wrap."""
    n = len(cls)
    out = {k: np.zeros(n) for k in ("iso_charged", "iso_neutral", "iso_photon", "r_iso")}
    ht, mx, my = [], [], []
    pt, eta, phi = (np.asarray(a, dtype=np.float32).astype(np.float64) for a in (pt, eta, phi))
    for a, b in zip(offsets[:-1], offsets[1:]):
        p, h, f, c = pt[a:b], eta[a:b], phi[a:b], np.asarray(cls[a:b])
        v = (p * np.exp(1j * f)).sum()
        ht.append(p.sum()), mx.append(-v.real), my.append(-v.imag)
        dphi = np.angle(np.exp(1j * (f[None, :] - f[:, None])))
        dr = np.hypot(h[None, :] - h[:, None], dphi)
        np.fill_diagonal(dr, np.inf)
        cone = dr < dr_max
        lep = (c == 1) | (c == 2)
        ch = (cone & (c[None, :] <= 2)) @ p
        nh = (cone & (c[None, :] == 3)) @ p
        ph = (cone & (c[None, :] == 4) & ~(dr < fsr_dr)) @ p
        out["iso_charged"][a:b] = np.where(lep, ch, 0)
        out["iso_neutral"][a:b] = np.where(lep, nh, 0)
        out["iso_photon"][a:b] = np.where(lep, ph, 0)
        out["r_iso"][a:b] = np.where(lep, (ch + nh + ph) / p, 0)
    out.update(ht=np.array(ht), met_x=np.array(mx), met_y=np.array(my), met=np.hypot(mx, my))
    return out


def test_against_brute_force_and_invariants():
    rng = np.random.default_rng(11)
    sizes = rng.poisson(40, 60)
    offsets = np.concatenate([[0], np.cumsum(sizes)])
    n = int(offsets[-1])
    cls = rng.choice([0, 1, 2, 3, 4], n, p=[0.4, 0.1, 0.1, 0.2, 0.2]).astype(np.int8)
    pt = (0.5 * 400 ** rng.random(n)).astype(np.float32)
    eta = rng.uniform(-1.0, 1.0, n).astype(np.float32)   # dense enough for populated cones
    phi = rng.uniform(-np.pi, np.pi, n).astype(np.float32)
    for dr_max, fsr in ((0.4, 0.0), (0.4, 0.07), (0.2, 0.0)):
        r = pdo.event_features(offsets, cls, pt, eta, phi, dr_max, fsr)
        b = _brute(offsets, cls, pt, eta, phi, dr_max, fsr)
        clean = r["iso_amb"] == 0
        assert clean.mean() > 0.99
        for k in ("iso_charged", "iso_neutral", "iso_photon", "r_iso"):
            assert np.allclose(r[k][clean], b[k][clean], rtol=1e-12, atol=1e-9), k
        for k in ("ht", "met_x", "met_y", "met"):
            assert np.allclose(r[k], b[k], rtol=1e-12, atol=1e-9), k
        lep = (cls == 1) | (cls == 2)
        assert np.all(r["r_iso"][~lep] == 0) and np.all(r["r_iso"] >= 0) and (r["r_iso"][lep] > 0).mean() > 0.2
        assert np.all(r["met"] <= r["ht"] + 1e-9)
    # a larger cone never isolates better; rotating the event in phi leaves H_T, MET and the isolation unchanged
    r2, r4 = (pdo.event_features(offsets, cls, pt, eta, phi, d, 0.0) for d in (0.2, 0.4))
    assert np.all(r4["r_iso"] >= r2["r_iso"] - 1e-12)
    rot = ((phi.astype(np.float64) + 1.0 + np.pi) % (2 * np.pi) - np.pi).astype(np.float32)
    rr = pdo.event_features(offsets, cls, pt, eta, rot, 0.4, 0.0)
    ok = (r4["iso_amb"] == 0) & (rr["iso_amb"] == 0)
    assert np.allclose(rr["ht"], r4["ht"]) and np.allclose(rr["met"], r4["met"], rtol=1e-5, atol=1e-4)
    assert np.allclose(rr["r_iso"][ok], r4["r_iso"][ok], rtol=1e-4, atol=1e-4)
