"""Pins of the oracle's RNG: known-answer vectors, layout values, mapping, moments."""
import math

import numpy as np

from conftest import read_table
from oracle import pdo


def test_philox_known_answer_vectors():
    for row in read_table("philox_kat.txt"):
        v = [int(x, 16) for x in row]
        assert pdo.philox(v[0:4], v[4:6]) == tuple(v[6:10])


def test_rng_layout_worked_values():
    for seed, event, obj, stream, *out in read_table("rng_layout.txt"):
        got = pdo.rng_block(int(seed, 16), int(event), int(obj), int(stream))
        assert got == tuple(int(x, 16) for x in out)


def test_rng_derived_draws():
    for kind, a, b, val in read_table("rng_derived.txt"):
        a, b, val = int(a, 16), int(b, 16), float(val)
        got = pdo.uniform(a) if kind == "u" else pdo.normal(a, b)
        assert abs(got - val) < 6e-10, (kind, hex(a), hex(b), got, val)


def test_uniform_mapping_end_points():
    assert pdo.uniform(0) == 0.0
    assert pdo.uniform(0xFFFFFFFF) == 1.0 - 2.0 ** -24
    assert pdo.uniform_pos(0) == 2.0 ** -24
    assert pdo.uniform_pos(0xFFFFFFFF) == 1.0
    assert pdo.uniform(0x000000FF) == 0.0  # low 8 bits are dropped
    assert pdo.uniform(0x00000100) == 2.0 ** -24


def test_normal_bound_and_extremes():
    # |z| <= sqrt(-2 ln 2^-24) = sqrt(48 ln 2)
    zmax = pdo.normal(0, 0)
    assert abs(zmax - math.sqrt(48.0 * math.log(2.0))) < 1e-12
    assert abs(zmax - 5.768108) < 1e-6
    assert pdo.normal(0xFFFFFFFF, 0) == 0.0  # u+ = 1 -> radius 0
    # cos branch: u(xb) = 0.5 -> z = -radius ; u(xb) = 0.25 -> ~0
    assert abs(pdo.normal(0, 0x80000000) + zmax) < 1e-12
    assert abs(pdo.normal(0, 0x40000000)) < 1e-12


def test_normal_moments_and_key_sensitivity():
    # distinct (seed, event, object, stream) give distinct blocks; draws have mean 0, variance 1
    n = 200_000
    zs = np.empty(n)
    us = np.empty(n)
    seen = set()
    for i in range(n):
        r = pdo.rng_block(12345, i // 1000, i % 1000, 0)
        zs[i] = pdo.normal(r[1], r[2])
        us[i] = pdo.uniform(r[0])
        if i < 2000:
            seen.add(r)
    assert len(seen) == 2000
    assert abs(zs.mean()) < 4.0 / math.sqrt(n)
    assert abs(zs.var() - 1.0) < 4.0 * math.sqrt(2.0 / n)
    assert abs(us.mean() - 0.5) < 4.0 * math.sqrt(1.0 / 12.0 / n)
    assert np.abs(zs).max() <= 5.768109
    # the four key ingredients all matter
    base = pdo.rng_block(1, 2, 3, 0)
    assert base != pdo.rng_block(2, 2, 3, 0)
    assert base != pdo.rng_block(1, 3, 3, 0)
    assert base != pdo.rng_block(1, 2, 4, 0)
    assert base != pdo.rng_block(1, 2, 3, 1)
    assert base != pdo.rng_block(1 + (1 << 32), 2, 3, 0)   # seed high word
    assert base != pdo.rng_block(1, 2 + (1 << 32), 3, 0)   # event high word
