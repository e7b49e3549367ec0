"""Pins of the oracle's pile-up merging (oracle/pd_oracle.c pdo_pileup_merge; Listing 8,
Table C.9): the Poisson inversion against scipy's quantile function, the truncated normal against its
closed-form moments, structural identities (mu = 0, one-event pool, order, copies), uniform pool picks,
determinism and batching.  CPU only."""
import importlib

import numpy as np
from scipy import stats

from oracle import pdo

wl = importlib.import_module("workloads.generate")


def _segments(r, hs, pool):
    """Split every output event into its source segments by walking the pool sizes along n_pileup; returns
    (event, k, out_start, out_end) with k = -1 for the hard scatter, plus the pool index of each pile-up segment
    recovered from the copied momenta."""
    segs = []
    for e in range(len(r["n_pileup"])):
        a, b = int(r["offsets"][e]), int(r["offsets"][e + 1])
        nh = int(hs.offsets[e + 1] - hs.offsets[e])
        segs.append((e, -1, a, a + nh))
        assert not r["is_pu"][a:a + nh].any() and r["is_pu"][a + nh:b].all()
    return segs


def test_poisson_is_the_quantile_of_the_block0_uniform():
    hs = wl.generate(0, 4000)
    pool = wl.generate(3, 50)
    for mu in (0.0, 0.3, 3.0, 50.0, 200.0):
        r = pdo.pileup_merge(hs, pool, mu, seed=11, event_base=5)
        u = np.array([pdo.uniform(pdo.rng_block(11, 5 + e, 0, 2)[0]) for e in range(hs.n_events)])
        want = stats.poisson.ppf(u, mu) if mu > 0 else np.zeros_like(u)
        # ppf = smallest n with cdf >= u, the oracle takes cdf > u: they differ only where cdf == u exactly
        assert np.array_equal(r["n_pileup"], want.astype(np.int32)), mu
        if mu > 0:
            n = r["n_pileup"].astype(np.float64)
            assert abs(n.mean() - mu) < 4 * np.sqrt(mu / len(n)) and abs(n.var() - mu) < 6 * mu * np.sqrt(2 / len(n)) + 0.05


def test_truncated_vertex_shift_moments_and_bounds():
    hs = wl.generate(0, 3000)
    one = wl.from_lists([[wl.particle(211, 1, 1.0, 0.0, 0.0, 0.13957039, vz=0.0)]])
    for sigma, zmax in ((0.053, 0.25), (0.05, 0.05), (0.1, 0.02)):
        r = pdo.pileup_merge(hs, one, 6.0, sigma, zmax, True, seed=3)
        dz = r["vz"][r["is_pu"] == 1].astype(np.float64)   # pool vertex is at z = 0: vz of a pile-up particle = its shift
        assert len(dz) > 15000 and np.abs(dz).max() <= zmax * (1 + 1e-6)
        t = stats.truncnorm(-zmax / sigma, zmax / sigma, scale=sigma)
        assert abs(dz.mean()) < 4 * t.std() / np.sqrt(len(dz)) and abs(dz.std() - t.std()) < 0.02 * t.std()
        assert stats.kstest(dz, t.cdf).pvalue > 1e-3
    # sigma_z = 0: no shift at all
    r = pdo.pileup_merge(hs, one, 2.0, 0.0, 0.25, True, seed=3)
    assert np.all(r["vz"][r["is_pu"] == 1] == 0)


def test_structure_order_and_copies():
    hs = wl.generate(1, 40)
    pool = wl.generate(3, 300)
    # mu = 0 without vertex smearing: the identity
    r = pdo.pileup_merge(hs, pool, 0.0, smear_hs_vertex=False, seed=9)
    assert np.array_equal(r["offsets"], hs.offsets) and not r["is_pu"].any()
    for k in ("pid", "charge", "px", "py", "pz", "E", "vx", "vy", "vz"):
        assert r[k].tobytes() == getattr(hs, k).tobytes(), k
    # mu = 0 with smearing: one common shift per event, nothing else touched
    r = pdo.pileup_merge(hs, pool, 0.0, smear_hs_vertex=True, seed=9)
    d = r["vz"].astype(np.float64) - hs.vz
    for e in range(hs.n_events):
        a, b = hs.offsets[e], hs.offsets[e + 1]
        assert np.ptp(d[a:b]) < 1e-6 and abs(d[a]) <= 0.25
    assert r["px"].tobytes() == hs.px.tobytes() and np.std(d) > 0.03
    # general case: hard scatter first and unchanged, then whole pool events, each with one common shift
    r = pdo.pileup_merge(hs, pool, 8.0, smear_hs_vertex=False, seed=9)
    sizes = np.diff(pool.offsets)
    first = {}                               # first particle's (px, E) -> pool event (unique in practice)
    for j in range(pool.n_events):
        if sizes[j] > 0:
            first[(float(pool.px[pool.offsets[j]]), float(pool.E[pool.offsets[j]]))] = j
    picks = []
    for e in range(hs.n_events):
        a, b = int(r["offsets"][e]), int(r["offsets"][e + 1])
        nh = int(hs.offsets[e + 1] - hs.offsets[e])
        assert r["px"][a:a + nh].tobytes() == hs.px[hs.offsets[e]:hs.offsets[e + 1]].tobytes()
        assert r["vz"][a:a + nh].tobytes() == hs.vz[hs.offsets[e]:hs.offsets[e + 1]].tobytes()
        pos, n_seen = a + nh, 0
        while pos < b:
            j = first[(float(r["px"][pos]), float(r["E"][pos]))]
            s = int(sizes[j])
            pa = int(pool.offsets[j])
            for k in ("pid", "charge", "px", "py", "pz", "E", "vx", "vy"):
                assert r[k][pos:pos + s].tobytes() == getattr(pool, k)[pa:pa + s].tobytes(), k
            dz = r["vz"][pos:pos + s].astype(np.float64) - pool.vz[pa:pa + s]
            assert np.ptp(dz) < 1e-6 and abs(dz[0]) <= 0.25 + 1e-6
            picks.append(j)
            pos += s
            n_seen += 1
        assert pos == b and n_seen <= r["n_pileup"][e]      # (empty pool events leave no trace)
    # the pick is floor(u * n_pool) of word 0 of the interaction's block
    e, k = 3, 0
    j0 = int(pdo.uniform(pdo.rng_block(9, e, 1 + k, 2)[0]) * pool.n_events)
    a = int(r["offsets"][e]) + int(hs.offsets[e + 1] - hs.offsets[e])
    if sizes[j0] > 0:
        assert first[(float(r["px"][a]), float(r["E"][a]))] == j0
    # picks are uniform over the pool
    r = pdo.pileup_merge(wl.generate(0, 2000), wl.from_lists([[wl.particle(22, 0, 1.0 + i, 0, 0, 0)] for i in range(16)]), 20.0, seed=2)
    cnt = np.bincount((r["E"][r["is_pu"] == 1] - 1.0 + 0.5).astype(int), minlength=16)
    assert stats.chisquare(cnt).pvalue > 1e-3


def test_deterministic_and_independent_of_batching():
    hs = wl.generate(0, 60)
    pool = wl.generate(3, 100)
    a = pdo.pileup_merge(hs, pool, 5.0, seed=4)
    b = pdo.pileup_merge(hs, pool, 5.0, seed=4)
    c = pdo.pileup_merge(hs, pool, 5.0, seed=5)
    assert all(a[k].tobytes() == b[k].tobytes() for k in a) and not np.array_equal(a["n_pileup"], c["n_pileup"])
    h1 = pdo.pileup_merge(wl.slice_events(hs, 0, 25), pool, 5.0, seed=4, event_base=0)
    h2 = pdo.pileup_merge(wl.slice_events(hs, 25, 60), pool, 5.0, seed=4, event_base=25)
    for k in ("pid", "px", "vz", "is_pu", "n_pileup"):
        assert np.concatenate([h1[k], h2[k]]).tobytes() == a[k].tobytes(), k


def test_truncated_normal_is_the_quantile_formula():
    """Reading H4 against scipy's normal quantile: |z| = -sigma Phi^-1(Phi(-a) + (1 - v)(1/2 - Phi(-a)))."""
    one = wl.from_lists([[wl.particle(22, 0, 1.0, 0.0, 0.0, 0.0)]])
    hs = wl.from_lists([[] for _ in range(300)])
    sigma, zmax = 0.053, 0.25
    r = pdo.pileup_merge(hs, one, 1.0, sigma, zmax, False, seed=21)
    pos = 0
    for e in range(300):
        for k in range(int(r["n_pileup"][e])):
            r1 = pdo.rng_block(21, e, 1 + k, 2)[1]
            u = ((r1 >> 8) + 0.5) / 2**24
            v = abs(2 * u - 1)
            lo = stats.norm.cdf(-zmax / sigma)
            z = -np.sign(u - 0.5) * sigma * stats.norm.ppf(lo + (1 - v) * (0.5 - lo))
            assert abs(float(r["vz"][pos]) - z) < 1e-7
            pos += 1
    assert pos == len(r["vz"])
