"""-m gpu: what stands in for compute-sanitizer (closed on this pool, profiles/r02_sanitizer.md).

1. Guard bands: every output array is filled with a sentinel byte before the call, the workspace is followed by a guard
   band; after the call nothing beyond the collections' totals and nothing in the guard band has changed -- no kernel
   variant writes where it should not (the capacities of pd.h are bounds, not sizes).
2. Schedule independence: the two persistent kernels are run with 1, 2 and the maximum number of resident CTAs per SM
   (PD_P_PER_SM / PD_T_PER_SM, read at every launch: other interleavings of the tiles, other look-back distances); the
   outputs are bitwise identical.  A race between CTAs, or between the warps of a tile, does not survive that for long.
"""
import importlib

import numpy as np
import pytest

wl = importlib.import_module("workloads.generate")

pytestmark = pytest.mark.gpu

SENTINEL = 0xA5


def _glued(n):
    ev = wl.generate(2, n // 4000 + 2)
    return wl.Events(offsets=np.array([0, n], dtype=np.int64),
                     **{k: np.ascontiguousarray(getattr(ev, k)[:n]) for k in ("pid", "charge", "px", "py", "pz", "E", "vx", "vy", "vz")})


CASES = {
    "dense": lambda: ("cms_like", wl.generate(1, 150)),
    "sparse": lambda: ("aleph_like", wl.generate(4, 2500)),
    "one_event_tiles": lambda: ("cms_like", wl.generate(2, 5)),
    "huge_1024": lambda: ("cms_like", wl.concat_events([_glued(7000), _glued(6500)])),
    "big_tile": lambda: ("cms_like", wl.concat_events([wl.generate(0, 40), _glued(12000), wl.generate(0, 10)])),
}


def _run(card_name, ev, debug):
    import torch

    import paper_2606_26089_b200 as pd

    card = pd.Card(card_name)
    dev = pd.DeviceEvents(ev)
    out = pd.DeviceOutputs(card, dev.n_events, dev.n_particles, debug=debug)
    groups = [out.trk, out.tow, out.efl] + ([out.dbg] if debug else [])
    for d in groups:
        for t in d.values():
            t.view(torch.uint8).fill_(SENTINEL)
    out.ws.fill_(SENTINEL)  # the 16 bytes behind ws_bytes are the guard band
    pd.simulate(card, dev, out, 19)
    torch.cuda.synchronize()
    assert pd.last_status(out) == 0
    return out


@pytest.mark.parametrize("case", sorted(CASES))
def test_nothing_is_written_beyond_the_totals(case):
    import torch

    card_name, ev = CASES[case]()
    for debug in (False, True):
        out = _run(card_name, ev, debug)
        assert bool((out.ws[out.ws_bytes:] == SENTINEL).all()), "workspace guard band overwritten"
        for d in (out.trk, out.tow, out.efl):
            tot = int(d["offsets"][-1])
            assert 0 < tot <= next(v for k, v in d.items() if k != "offsets").shape[0]
            for k, t in d.items():
                if k == "offsets":
                    continue
                tail = t[tot:].view(torch.uint8)
                assert bool((tail == SENTINEL).all()), (case, debug, k, "written beyond the total")
                # and everything up to the total WAS written (no gaps of uninitialised memory): a run of sentinel
                # bytes as long as an element would be a float / int that no event produces
                head = t[:tot].view(torch.uint8).reshape(tot, -1)
                assert not bool((head == SENTINEL).all(dim=1).any()) or t.element_size() == 1, (case, debug, k, "gap")


@pytest.mark.parametrize("case", ["dense", "sparse", "one_event_tiles", "big_tile"])
def test_results_do_not_depend_on_the_number_of_resident_ctas(case, monkeypatch):
    card_name, ev = CASES[case]()
    ref = None
    for p_per_sm, t_per_sm in ((None, None), ("1", "1"), ("2", "1"), ("1", "2"), ("3", "2")):
        for name, val in (("PD_P_PER_SM", p_per_sm), ("PD_T_PER_SM", t_per_sm)):
            if val is None:
                monkeypatch.delenv(name, raising=False)
            else:
                monkeypatch.setenv(name, val)
        got = _run(card_name, ev, False).to_numpy()
        if ref is None:
            ref = got
            continue
        for k, v in got.items():
            assert v.tobytes() == ref[k].tobytes(), (case, p_per_sm, t_per_sm, k)


def test_after_card_upload_a_step_allocates_no_device_memory():
    """pd_card_upload (pd.h): the one allocation of the chain -- the card's tables on a device -- done ahead of time; the step
    itself (pd_simulate_ex with caller-owned buffers and workspace) then leaves the free device memory as it found it."""
    import torch

    import paper_2606_26089_b200 as pd

    card = pd.Card("atlas_like")  # a card object no earlier test has used on the device
    ev = wl.generate(3, 2000)
    dev = pd.DeviceEvents(ev)
    out = pd.DeviceOutputs(card, dev.n_events, dev.n_particles, debug=False)
    warm = pd.Card("cms_like")    # module load, kernel attributes and first launches, on another card
    pd.simulate(warm, pd.DeviceEvents(wl.generate(0, 50)), pd.DeviceOutputs(warm, 50, wl.generate(0, 50).n_particles), 1)
    torch.cuda.synchronize()
    pd.card_upload(card)
    pd.card_upload(card)  # idempotent
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    pd.simulate(card, dev, out, 7)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert pd.last_status(out) == 0 and int(out.trk["offsets"][-1]) > 0
    assert free1 == free0, (free0, free1)


def test_the_on_axis_copy_of_the_row_loop_is_bitwise_the_general_one():
    """Kernel P keeps two copies of its row loop: warps whose vertices all sit on the beam axis take one in which the terms that
    vanish for vx = vy = 0 are left out.  A vertex 1e-20 m off the axis on every 50th particle sends (nearly) every warp through
    the general copy instead: the positions, towers and decisions of all the OTHER particles must not change by a bit."""
    import paper_2606_26089_b200 as pd

    for card_name, cfg, ne in (("cms_like", 0, 600), ("cms_like", 2, 6), ("aleph_like", 4, 900)):
        ev = wl.generate(cfg, ne)
        assert not ev.vx.any() and not ev.vy.any()
        nudged = np.zeros(ev.n_particles, dtype=bool)
        nudged[::50] = True
        vx = ev.vx.copy()
        vx[nudged] = np.float32(1e-20)
        ev2 = wl.Events(offsets=ev.offsets, **{k: (vx if k == "vx" else getattr(ev, k)) for k in ("pid", "charge", "px", "py", "pz", "E", "vx", "vy", "vz")})
        res = []
        for e in (ev, ev2):
            card = pd.Card(card_name)
            dev = pd.DeviceEvents(e)
            out = pd.DeviceOutputs(card, dev.n_events, dev.n_particles, debug=True)
            pd.simulate(card, dev, out, 23)
            res.append(out.to_numpy())
        for k in ("dbg_status", "dbg_eta_pos", "dbg_phi_pos", "dbg_tower", "dbg_accepted", "dbg_pt_smeared"):
            a, b = res[0][k][~nudged], res[1][k][~nudged]
            assert a.tobytes() == b.tobytes(), (card_name, cfg, k)
