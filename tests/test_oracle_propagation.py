"""Pins of the oracle's propagation O2: RK4 integration of the Lorentz force,
closed forms for on-axis vertices, straight-line neutrals, worked positions."""
import math

import numpy as np
import pytest

from conftest import read_table
from oracle import pdo

KAPPA = float(np.float32(0.299792458))


def _rk4_to_surface(q, p, v, B, R, L, h=2e-4):
    """Integrate dx/ds = p/|p|, dp/ds = kappa q (p x B zhat)/|p| until r = R or |z| = L (independent of the
    oracle's closed form).  Returns (x, y, z, face)."""
    x = np.array(v, dtype=np.float64)
    p = np.array(p, dtype=np.float64)
    pn = np.linalg.norm(p)

    def f(y):
        pp = y[3:]
        return np.concatenate([pp / pn, KAPPA * q * np.array([pp[1] * B, -pp[0] * B, 0.0]) / pn])

    y = np.concatenate([x, p])
    for _ in range(int(400.0 / h)):
        k1 = f(y)
        k2 = f(y + 0.5 * h * k1)
        k3 = f(y + 0.5 * h * k2)
        k4 = f(y + h * k3)
        yn = y + (h / 6.0) * (k1 + 2 * k2 + 2 * k3 + k4)
        rn = math.hypot(yn[0], yn[1])
        if rn >= R or abs(yn[2]) >= L:
            # bisect the last step for the crossing
            lo, hi = 0.0, h
            face = None
            for _ in range(60):
                mid = 0.5 * (lo + hi)
                k1 = f(y)
                k2 = f(y + 0.5 * mid * k1)
                k3 = f(y + 0.5 * mid * k2)
                k4 = f(y + mid * k3)
                ym = y + (mid / 6.0) * (k1 + 2 * k2 + 2 * k3 + k4)
                out_r = math.hypot(ym[0], ym[1]) >= R
                out_z = abs(ym[2]) >= L
                if out_r or out_z:
                    hi = mid
                    face = 1 if out_r and not out_z else 2
                else:
                    lo = mid
            return ym[0], ym[1], ym[2], face
        y = yn
    raise AssertionError("never reached the surface")


def _mom(pt, eta, phi):
    return pt * math.cos(phi), pt * math.sin(phi), pt * math.sinh(eta)


RK4_CASES = [
    # q, pT, eta, phi, vertex
    (1, 10.0, 0.5, 0.3, (0, 0, 0)),           # barrel
    (-1, 10.0, 0.5, 0.3, (0, 0, 0)),          # other charge
    (1, 0.9, 0.2, -2.0, (0, 0, 0)),           # strongly curved, barrel
    (1, 0.5, 1.0, 1.0, (0, 0, 0.03)),         # looper to the endcap
    (-1, 50.0, 2.0, 3.0, (0, 0, -0.05)),      # endcap
    (1, 2.0, -0.7, 2.5, (0.01, -0.02, 0.1)),  # displaced vertex
    (-1, 0.8, 0.1, 0.0, (0.3, 0.2, 0.0)),     # far-displaced vertex
    (1, 0.3, -0.4, 0.7, (0.2, -0.1, -0.5)),   # looper, displaced
]


@pytest.mark.parametrize("q,pt,eta,phi,v", RK4_CASES)
def test_helix_against_rk4(q, pt, eta, phi, v):
    card = pdo.Card("cms_like")
    px, py, pz = _mom(pt, eta, phi)
    h = card.propagate(q, px, py, pz, *v)
    x, y, z, face = _rk4_to_surface(q, (px, py, pz), v, card.bz, card.radius, card.half_length)
    assert (h["status"] & pdo.PDO_FACE_MASK) == face
    assert abs(h["x"] - x) < 2e-7 and abs(h["y"] - y) < 2e-7 and abs(h["z"] - z) < 2e-7


def test_rotation_sense_positive_charge_turns_clockwise():
    # reading A3: B along +z, q > 0: momentum azimuth decreases
    card = pdo.Card("cms_like")
    px, py, pz = _mom(5.0, 0.1, 0.0)
    plus = card.propagate(+1, px, py, pz)
    minus = card.propagate(-1, px, py, pz)
    assert plus["phi_pos"] < 0.0 < minus["phi_pos"]
    assert abs(plus["phi_pos"] + minus["phi_pos"]) < 1e-14


@pytest.mark.parametrize("name", ["cms_like", "atlas_like", "aleph_like"])
def test_on_axis_closed_forms(name):
    card = pdo.Card(name)
    B, R, L = card.bz, card.radius, card.half_length
    row = [r for r in read_table("closed_forms.txt") if r[0] == name][0]
    pt_min, eta_corner = float(row[1]), float(row[2])
    assert abs(KAPPA * B * R / 2.0 - pt_min) < 1e-6
    assert abs(math.asinh(L / R) - eta_corner) < 1e-6
    rng = np.random.default_rng(7)
    for _ in range(300):
        pt = float(np.exp(rng.uniform(math.log(0.11), math.log(300.0))))
        eta = float(rng.uniform(-1.0, 1.0))
        phi = float(rng.uniform(-math.pi, math.pi))
        q = int(rng.choice([-1, 1]))
        px, py, pz = _mom(pt, eta, phi)
        h = card.propagate(q, px, py, pz)
        rho = pt / (KAPPA * B)
        if pt < pt_min * (1 - 1e-9):
            assert h["status"] & pdo.PDO_LOOPER  # cannot reach r = R
            continue
        if pt <= pt_min * (1 + 1e-9):
            continue
        a_r = 2.0 * math.asin(R / (2.0 * rho))
        z_r = rho * a_r * math.sinh(eta)
        if abs(z_r) < L:
            assert h["status"] == pdo.PDO_BARREL
            assert abs(h["alpha"] - a_r) < 1e-10
            dphi = math.remainder(h["phi_pos"] - (phi - q * a_r / 2.0), 2 * math.pi)
            assert abs(dphi) < 1e-10
            assert abs(h["z"] - z_r) < 1e-10
            assert abs(math.hypot(h["x"], h["y"]) - R) < 1e-10


def test_rho_of_one_gev():
    # rho(pT = 1 GeV) = 0.877800 m at 3.8 T: chord of a barrel hit R = 2 rho sin(alpha/2)
    card = pdo.Card("cms_like")
    h = card.propagate(1, 1.0, 0.0, 0.0)
    rho = card.radius / (2.0 * math.sin(h["alpha"] / 2.0))
    assert abs(rho - 0.877800) < 1e-6


@pytest.mark.parametrize("name", ["cms_like", "atlas_like", "aleph_like"])
def test_neutral_from_axis_keeps_direction(name):
    card = pdo.Card(name)
    R, L = card.radius, card.half_length
    rng = np.random.default_rng(11)
    for _ in range(500):
        pt = float(rng.uniform(0.2, 100))
        eta = float(rng.uniform(-4.5, 4.5))
        phi = float(rng.uniform(-math.pi, math.pi))
        vz = float(rng.uniform(-0.2, 0.2))
        px, py, pz = _mom(pt, eta, phi)
        h0 = card.propagate(0, px, py, pz)
        assert abs(h0["eta_pos"] - eta) < 1e-12 and abs(h0["phi_pos"] - phi) < 1e-12
        assert h0["alpha"] == 0.0
        h = card.propagate(0, px, py, pz, 0, 0, vz)
        barrel = abs(eta) < math.asinh((L - math.copysign(1.0, pz) * vz) / R)
        assert (h["status"] & 3) == (pdo.PDO_BARREL if barrel else pdo.PDO_ENDCAP)
        if not barrel:
            assert h["z"] == math.copysign(L, pz)
        else:
            assert abs(math.hypot(h["x"], h["y"]) - R) < 1e-12


def test_dropped_cases():
    card = pdo.Card("cms_like")
    R, L = card.radius, card.half_length
    assert card.propagate(1, 1, 0, 1, R, 0, 0)["status"] == pdo.PDO_DROPPED        # born on the cylinder
    assert card.propagate(0, 1, 0, 1, 0, 2.0, 0)["status"] == pdo.PDO_DROPPED      # outside
    assert card.propagate(0, 1, 0, 1, 0, 0, L)["status"] == pdo.PDO_DROPPED
    assert card.propagate(0, 1e-5, 0, 1)["status"] == pdo.PDO_DROPPED              # pT^2 < 1e-9
    assert (card.propagate(1, 0.3, 0, 0)["status"] & 3) == pdo.PDO_DROPPED         # trapped: pz = 0 looper
    assert (card.propagate(0, 0.3, 0, 0)["status"] & 3) == pdo.PDO_BARREL          # neutral pz = 0 is fine


def test_worked_positions_and_towers():
    card = pdo.Card("cms_like")
    for row in read_table("positions_cms_like.txt"):
        pid, q = int(row[0]), int(row[1])
        pt, eta, phi, vx, vy, vz = map(float, row[2:8])
        eta_pos, phi_pos = float(row[8]), float(row[9])
        face, looper, ieta, iphi, tower = map(int, row[10:15])
        h = card.propagate(q, *_mom(pt, eta, phi), vx, vy, vz)
        assert (h["status"] & 3) == face and bool(h["status"] & 4) == bool(looper)
        assert abs(h["eta_pos"] - eta_pos) < 1.5e-6 and abs(h["phi_pos"] - phi_pos) < 1.5e-6
        assert card.tower_index(h["eta_pos"], h["phi_pos"]) == tower
        assert card.offset[ieta] + iphi == tower


def test_worked_xyz_and_turning_angles():
    card = pdo.Card("cms_like")
    for row in read_table("positions_xyz.txt"):
        q = int(row[0])
        pt, eta, phi, vx, vy, vz, x, y, z = map(float, row[1:])
        h = card.propagate(q, *_mom(pt, eta, phi), vx, vy, vz)
        assert abs(h["x"] - x) < 1e-6 and abs(h["y"] - y) < 1e-6 and abs(h["z"] - z) < 1e-6
    for row in read_table("turning_angles.txt"):
        q = int(row[0])
        pt, eta, phi, vz, alpha = map(float, row[1:])
        h = card.propagate(q, *_mom(pt, eta, phi), 0, 0, vz)
        # the card's B, R, L, kappa are rounded to fp32 at load (reading A28): ~3e-8 relative
        assert abs(h["alpha"] - alpha) < 1e-7 * max(1.0, alpha)
