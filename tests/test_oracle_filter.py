"""Pins of the oracle's particle filter (oracle/pd_oracle.c pdo_filter_eflow, Table C.13):
a hand-worked case, every operator, AND / OR semantics, an independent numpy boolean-mask re-derivation, and
invariants.  CPU only."""
import numpy as np

from oracle import pdo


def _coll(seed=3, sizes=(0, 5, 1, 0, 40, 17)):
    rng = np.random.default_rng(seed)
    off = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int64)
    n = int(off[-1])
    cls = rng.integers(0, 5, n).astype(np.int8)
    src = rng.integers(0, 10000, n).astype(np.int32)
    pt = (0.1 * 1000 ** rng.random(n)).astype(np.float32)
    eta = rng.uniform(-4, 4, n).astype(np.float32)
    phi = rng.uniform(-np.pi, np.pi, n).astype(np.float32)
    E = (pt * np.cosh(eta)).astype(np.float32)
    return off, cls, src, pt, eta, phi, E


def test_hand_worked_case():
    # two events; keep pT > 0.5 AND |eta| < 2.5 (the paper's own example of conditions: "pT, eta ... cuts", abs flag)
    off = [0, 3, 5]
    cls, src = [1, 0, 4, 3, 2], [7, 8, 9, 10, 11]
    pt, eta = [10, 0.4, 2, 3, 8], [0, 2.7, -1, 0.3, -2.6]
    phi, E = [0.1, 0.2, 0.3, 0.4, 0.5], [10, 3, 2, 3, 50]
    conds = [{"field": "pt", "op": ">", "value": 0.5}, {"field": "eta", "op": "<", "value": 2.5, "abs": True}]
    r = pdo.filter_eflow(off, cls, src, pt, eta, phi, E, conds, "all")
    assert r["keep"].tolist() == [1, 0, 1, 1, 0] and r["offsets"].tolist() == [0, 2, 3]
    assert r["src"].tolist() == [7, 9, 10] and r["cls"].tolist() == [1, 4, 3] and r["pt"].tolist() == [10, 2, 3]
    assert np.allclose(r["phi"], [0.1, 0.3, 0.4]) and r["E"].tolist() == [10, 2, 3]
    r = pdo.filter_eflow(off, cls, src, pt, eta, phi, E, conds, "any")  # OR: object 1 fails both, object 4 passes pT
    assert r["keep"].tolist() == [1, 0, 1, 1, 1] and r["offsets"].tolist() == [0, 2, 4]
    # class-id cuts ("PDG-ID cuts"): leptons only; everything but photons and neutral hadrons
    r = pdo.filter_eflow(off, cls, src, pt, eta, phi, E, [{"field": "cls", "op": "in", "value": [1, 2]}])
    assert r["keep"].tolist() == [1, 0, 0, 0, 1]
    r = pdo.filter_eflow(off, cls, src, pt, eta, phi, E, [{"field": "cls", "op": "not in", "value": [3, 4]}])
    assert r["keep"].tolist() == [1, 1, 0, 0, 1]
    # no condition: nothing is dropped (reading G1)
    for comb in ("all", "any"):
        r = pdo.filter_eflow(off, cls, src, pt, eta, phi, E, [], comb)
        assert r["keep"].tolist() == [1] * 5 and r["offsets"].tolist() == [0, 3, 5]


def test_every_operator_on_the_threshold():
    off = [0, 3]
    vals = np.array([1.0, 2.0, 3.0], dtype=np.float32)
    z = np.zeros(3, dtype=np.float32)
    expect = {">": [0, 0, 1], ">=": [0, 1, 1], "<": [1, 0, 0], "<=": [1, 1, 0], "==": [0, 1, 0], "!=": [1, 0, 1]}
    for op, want in expect.items():
        r = pdo.filter_eflow(off, [0, 0, 0], [0, 1, 2], vals, z, z, z, [{"field": "pt", "op": op, "value": 2.0}])
        assert r["keep"].tolist() == want, op
    # abs applies to the attribute, not to the value
    r = pdo.filter_eflow(off, [0, 0, 0], [0, 1, 2], z, [-3.0, 0.5, 2.0], z, z, [{"field": "eta", "op": ">", "value": 1.0, "abs": True}])
    assert r["keep"].tolist() == [1, 0, 1]
    r = pdo.filter_eflow(off, [0, 0, 0], [0, 1, 2], z, [-3.0, 0.5, 2.0], z, z, [{"field": "eta", "op": ">", "value": 1.0}])
    assert r["keep"].tolist() == [0, 0, 1]


def _mask(coll, conds, combine):
    off, cls, src, pt, eta, phi, E = coll
    col = {"pt": pt, "eta": eta, "phi": phi, "E": E, "cls": cls.astype(np.float32)}
    ms = []
    for c in conds:
        x = np.abs(col[c["field"]]) if c.get("abs") else col[c["field"]]
        v = c["value"]
        m = {">": lambda: x > np.float32(v), ">=": lambda: x >= np.float32(v), "<": lambda: x < np.float32(v),
             "<=": lambda: x <= np.float32(v), "==": lambda: x == np.float32(v), "!=": lambda: x != np.float32(v),
             "in": lambda: np.isin(x, np.asarray(v, dtype=np.float32)),
             "not in": lambda: ~np.isin(x, np.asarray(v, dtype=np.float32))}[c["op"]]()
        ms.append(m)
    if not ms:
        return np.ones(len(pt), dtype=bool)
    return np.logical_or.reduce(ms) if combine == "any" else np.logical_and.reduce(ms)


def test_against_numpy_masks_and_invariants():
    coll = _coll(sizes=np.random.default_rng(1).poisson(30, 200))
    off = coll[0]
    sets = [
        [{"field": "pt", "op": ">", "value": 1.0}],
        [{"field": "pt", "op": ">=", "value": 0.7}, {"field": "eta", "op": "<", "value": 2.5, "abs": True}],
        [{"field": "cls", "op": "in", "value": [0, 1, 2]}, {"field": "pt", "op": "<=", "value": 50.0}, {"field": "phi", "op": ">", "value": 0.0}],
        [{"field": "cls", "op": "not in", "value": [4]}, {"field": "E", "op": ">", "value": 5.0}],
        [{"field": "cls", "op": "==", "value": 3}, {"field": "eta", "op": "!=", "value": 0.0}],
    ]
    for conds in sets:
        kept = {}
        for comb in ("all", "any"):
            r = pdo.filter_eflow(*coll, conds, comb)
            m = _mask(coll, conds, comb)
            assert np.array_equal(r["keep"].astype(bool), m)
            ev = np.repeat(np.arange(len(off) - 1), np.diff(off))
            assert np.array_equal(r["offsets"], np.concatenate([[0], np.cumsum(np.bincount(ev[m], minlength=len(off) - 1))]))
            for k, a in zip(("cls", "src", "pt", "eta", "phi", "E"), coll[1:]):
                assert np.array_equal(r[k], a[m]), k        # survivors unchanged and in order
            kept[comb] = m
        assert np.all(kept["any"] | ~kept["all"])               # AND keeps a subset of OR
    # idempotent: filtering the survivors again drops nothing
    r1 = pdo.filter_eflow(*coll, sets[1], "all")
    r2 = pdo.filter_eflow(r1["offsets"], r1["cls"], r1["src"], r1["pt"], r1["eta"], r1["phi"], r1["E"], sets[1], "all")
    assert r2["keep"].all() and np.array_equal(r2["offsets"], r1["offsets"])
