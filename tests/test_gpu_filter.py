"""-m gpu: pd_filter_eflow (the paper's particle filter, PAPER.md L119 / Table C.13) through the C ABI against the
oracle: bit-exact (integers, order, offsets, and the floats, which are copied, never computed).  Inputs come
from the ORACLE's chain output and from seeded synthetic generators."""
import importlib

import numpy as np
import pytest

wl = importlib.import_module("workloads.generate")

pytestmark = pytest.mark.gpu

SETS = [
    ([{"field": "pt", "op": ">", "value": 1.0}], "all"),
    ([{"field": "pt", "op": ">=", "value": 0.7}, {"field": "eta", "op": "<", "value": 2.5, "abs": True}], "all"),
    ([{"field": "pt", "op": ">", "value": 20.0}, {"field": "cls", "op": "in", "value": [1, 2]}], "any"),
    ([{"field": "cls", "op": "not in", "value": [3, 4]}, {"field": "E", "op": "<=", "value": 30.0}, {"field": "phi", "op": "!=", "value": 0.0}], "all"),
    ([], "all"),
    ([{"field": "pt", "op": "<", "value": 0.0}], "all"),   # drops everything
]


def _gpu(arrays, conds, comb):
    import paper_2606_26089_b200 as pd

    ne, n = len(arrays["offsets"]) - 1, int(arrays["offsets"][-1])
    src = pd.DeviceEFlow(ne, n, arrays)
    dst = pd.DeviceEFlow(ne, n)
    ws = pd.filter_eflow(src, dst, conds, comb)
    assert pd.last_launch_count() == 2
    out = dst.to_numpy()
    del ws
    return out, dst


def _same(g, o):
    assert np.array_equal(g["offsets"], o["offsets"])
    for k in ("cls", "src", "pt", "eta", "phi", "E"):
        assert g[k].tobytes() == o[k].tobytes(), k


@pytest.mark.parametrize("cfg,n_events", [(0, 800), (2, 10), (3, 3000), (4, 2000)])
def test_filter_of_oracle_eflow(cfg, n_events):
    from oracle import pdo

    ev = wl.generate(cfg, n_events)
    o = pdo.simulate(pdo.Card(wl.config_card(cfg)), ev, wl.CONFIGS[cfg]["seed"], debug=False)
    arrays = {"offsets": o["efl_offsets"], "cls": o["efl_cls"], "src": o["efl_src"]}
    arrays.update({k: o["efl_" + k].astype(np.float32) for k in ("pt", "eta", "phi", "E")})
    for conds, comb in SETS:
        ref = pdo.filter_eflow(arrays["offsets"], arrays["cls"], arrays["src"], arrays["pt"], arrays["eta"], arrays["phi"], arrays["E"], conds, comb)
        got, _ = _gpu(arrays, conds, comb)
        _same(got, ref)


def test_ragged_tile_boundaries_and_features_of_survivors():
    import paper_2606_26089_b200 as pd
    from oracle import pdo

    rng = np.random.default_rng(4)
    # sizes around the 2,048-object tiles, empty events at the start / end / in runs, one object, exact multiples
    for sizes in ([0, 0, 2047, 1, 0, 2048, 4096, 3, 0, 0], [2048], [2047], [2049], [0], [1], [], [5] * 3000, [0] * 5000 + [7]):
        off = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int64)
        n = int(off[-1])
        arrays = {"offsets": off, "cls": rng.integers(0, 5, n).astype(np.int8), "src": rng.integers(0, 1 << 20, n).astype(np.int32),
                  "pt": (0.1 * 1000 ** rng.random(n)).astype(np.float32), "eta": rng.uniform(-4, 4, n).astype(np.float32),
                  "phi": rng.uniform(-np.pi, np.pi, n).astype(np.float32), "E": rng.random(n).astype(np.float32) * 100}
        for conds, comb in SETS[:3] + SETS[4:]:
            ref = pdo.filter_eflow(off, arrays["cls"], arrays["src"], arrays["pt"], arrays["eta"], arrays["phi"], arrays["E"], conds, comb)
            got, dst = _gpu(arrays, conds, comb)
            _same(got, ref)
        # "update_event_features": H_T / MET / isolation of the survivors, on the device-resident filter output
        if len(sizes) > 0 and n > 0:
            feat = pd.DeviceFeatures(dst.n_events, max(n, 1))
            pd.event_features(dst, feat)
            g = feat.to_numpy(int(got["offsets"][-1]))
            # the oracle's inputs are the ORACLE's survivors (bit-identical to the device's, checked by _same above)
            r = pdo.event_features(ref["offsets"], ref["cls"], ref["pt"], ref["eta"], ref["phi"])
            assert np.all(np.abs(g["ht"] - r["ht"]) <= np.maximum(1e-5 * r["ht"], 1e-6))
            ok = r["iso_amb"] == 0
            assert np.all(np.abs(g["r_iso"] - r["r_iso"])[ok] <= np.maximum(1e-5 * r["r_iso"], 1e-6)[ok])


def test_unaligned_arrays_nan_fields_and_many_tiles():
    """arrays that do not start at a multiple of 16 bytes (every tile then comes by plain loads instead of bulk copies) give the same
    survivors as aligned ones; NaN in a field fails every ordered comparison and == / "in", passes != / "not in" (the C operators
    the oracle applies); 40 tiles and a ragged tail"""
    import paper_2606_26089_b200 as pd
    from oracle import pdo
    from paper_2606_26089_b200 import binding as B

    torch = B._torch()
    rng = np.random.default_rng(11)
    sizes = rng.integers(0, 90, 1900)
    off = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int64)
    n = int(off[-1])
    assert n > 40 * 2048 and n % 2048 not in (0, 1)
    arrays = {"offsets": off, "cls": rng.integers(0, 5, n).astype(np.int8), "src": rng.integers(0, 1 << 20, n).astype(np.int32),
              "pt": (0.1 * 1000 ** rng.random(n)).astype(np.float32), "eta": rng.uniform(-4, 4, n).astype(np.float32),
              "phi": rng.uniform(-np.pi, np.pi, n).astype(np.float32), "E": rng.random(n).astype(np.float32) * 100}
    for k in ("pt", "eta", "phi", "E"):
        arrays[k][rng.integers(0, n, 500)] = np.nan
    arrays["E"][rng.integers(0, n, 500)] = 30.0  # equality cases of <=, ==, "in"
    sets = SETS + [
        ([{"field": "E", "op": "!=", "value": 30.0}], "all"),
        ([{"field": "E", "op": "==", "value": 30.0}, {"field": "eta", "op": ">", "value": 3.9}], "any"),
        ([{"field": "E", "op": "in", "value": [30.0, 12.0]}], "all"),
        ([{"field": "E", "op": "not in", "value": [30.0]}, {"field": "phi", "op": "<=", "value": -1.0, "abs": False}], "all"),
        ([{"field": "eta", "op": ">=", "value": 1.0, "abs": True}, {"field": "cls", "op": "==", "value": 2}], "all"),
    ]
    ne = len(off) - 1
    for conds, comb in sets:
        ref = pdo.filter_eflow(off, arrays["cls"], arrays["src"], arrays["pt"], arrays["eta"], arrays["phi"], arrays["E"], conds, comb)
        got, _ = _gpu(arrays, conds, comb)
        _same(got, ref)
        # the same input one element into larger buffers: 4 bytes (1 for cls) past a 16-byte boundary
        src = pd.DeviceEFlow(ne, n, arrays)
        keep = []
        for k, _dt in B.EFLOW_FIELDS:
            big = torch.empty(n + 1, dtype=src.t[k].dtype, device="cuda")
            big[1:].copy_(src.t[k][:n])
            keep.append(big)
            src.t[k] = big[1:]
            assert src.t[k].data_ptr() % 16 != 0
        src.c_efl = B.EFlow(src.capacity, B._tptr(src.t["offsets"]), *[B._tptr(src.t[k]) for k, _dt in B.EFLOW_FIELDS])
        dst = pd.DeviceEFlow(ne, n)
        ws = pd.filter_eflow(src, dst, conds, comb)
        _same(dst.to_numpy(), ref)
        del ws, keep


def test_argument_checks():
    import ctypes as C

    import paper_2606_26089_b200 as pd
    from paper_2606_26089_b200 import binding as B

    arrays = {"offsets": np.array([0, 2]), "cls": np.zeros(2, np.int8), "src": np.zeros(2, np.int32), "pt": np.ones(2, np.float32),
              "eta": np.zeros(2, np.float32), "phi": np.zeros(2, np.float32), "E": np.ones(2, np.float32)}
    src, small = pd.DeviceEFlow(1, 2, arrays), pd.DeviceEFlow(1, 1)
    with pytest.raises(pd.PdError):
        pd.filter_eflow(src, small, [], "all")  # PD_ECAPACITY
    bad = B.make_conditions([{"field": "pt", "op": ">", "value": 1.0}])
    bad[0].op = 99
    L = B.lib()
    assert L.pd_filter_eflow(C.byref(src.c_efl), 1, bad, 1, 0, C.byref(src.c_efl), None, 0, None) == B.PD_EINVAL
    assert L.pd_filter_workspace_bytes(-1) == B.PD_EINVAL
