"""Pins of the oracle's smearing (O3 track, O5 tower): SURVEY 8c.5 P8 — closed forms, moments, worked values."""
import math

import numpy as np

from conftest import read_table
from oracle import pdo


def test_lognormal_special_cases_and_median():
    assert pdo.lognormal(0.0, 1.0, 0.3) == 0.0      # m <= 0 -> 0
    assert pdo.lognormal(-1.0, 1.0, 0.3) == 0.0
    assert pdo.lognormal(7.5, 0.0, 2.0) == 7.5      # s <= 0 -> unchanged
    for m, s in ((50.0, 5.0), (1.0, 2.0), (0.3, 0.01)):
        # z = 0 gives the median m / sqrt(1 + s^2/m^2)
        assert abs(pdo.lognormal(m, s, 0.0) - m / math.sqrt(1.0 + (s / m) ** 2)) < 1e-12 * m
        # ln LN is linear in z with slope sqrt(ln(1 + s^2/m^2))
        b = math.sqrt(math.log1p((s / m) ** 2))
        assert abs(math.log(pdo.lognormal(m, s, 1.5) / pdo.lognormal(m, s, -0.5)) - 2.0 * b) < 1e-12


def test_lognormal_moments_are_mean_m_and_std_s():
    # Gauss-Hermite quadrature over z ~ N(0,1): E[LN] = m, Var[LN] = s^2 (moment matching, reading A21)
    x, w = np.polynomial.hermite_e.hermegauss(80)
    w = w / math.sqrt(2.0 * math.pi)
    for m, s in ((10.0, 1.0), (2.0, 3.0), (100.0, 0.7), (0.5, 0.45)):
        v = np.array([pdo.lognormal(m, s, float(z)) for z in x])
        mean = float((w * v).sum())
        var = float((w * (v - mean) ** 2).sum())
        assert abs(mean - m) < 1e-9 * m
        assert abs(math.sqrt(var) - s) < 1e-7 * s


def test_worked_smearing_values():
    for row in read_table("smearing.txt"):
        kind, vals = row[0], list(map(float, row[1:]))
        if kind == "LN":
            m, s, z, out = vals
            assert abs(pdo.lognormal(m, s, z) - out) < 1e-8
        elif kind == "TRK":
            pt, z, srel, out = vals
            got_srel = math.sqrt(float(np.float32(0.01)) ** 2 + (float(np.float32(1.5e-4)) * pt) ** 2)
            assert abs(got_srel - srel) < 1e-8
            assert abs(pdo.lognormal(pt, got_srel * pt, z) - out) < 2e-7
        else:
            E, C, S, N, z, sigma, out = vals
            C, S, N = (float(np.float32(v)) for v in (C, S, N))
            got_sigma = math.sqrt(C * C * E * E + S * S * E + N * N)
            assert abs(got_sigma - sigma) < 2e-7
            assert abs(pdo.lognormal(E, got_sigma, z) - out) < 5e-6
