"""-m gpu: pd_track_impact (d0, z0 and their errors; Table 2, readings I1-I3 of DESIGN.md section 14)
through the C ABI against the fp64 oracle, element by element.  The track lists (offsets, src) come from the
ORACLE's own chain output or from seeded generators -- never from the CUDA chain.  (One test feeds pd_simulate's
device output to pd_track_impact; the oracle it is compared with runs on the oracle's own track list, and the two are
matched by particle index.)

Tolerance: 1e-5 relative / 1e-6 absolute (metres) on d0 and z0, true and smeared; errors
1e-5 relative.  (Stress test with vertices a metre off the axis: the absolute bound of z0 scales with its two terms.)  The geometry is arranged so that nothing cancels (error-free products, d0 as a quotient), and the
normals are those of the chain (Box-Muller on 24-bit uniforms, |error| < 1e-6)."""
import importlib

import numpy as np
import pytest

import cards

wl = importlib.import_module("workloads.generate")

pytestmark = pytest.mark.gpu


def _close(g, o, what, atol=1e-6):
    bad = np.abs(g.astype(np.float64) - o) > np.maximum(1e-5 * np.abs(o), atol)
    assert not bad.any(), "%s: %d of %d off, worst %g" % (what, int(bad.sum()), bad.size, float(np.abs(g - o).max()))


def _run_gpu(card_name, ev, off, src, d0_res, z0_res, seed=0, event_base=0):
    import paper_2606_26089_b200 as pd

    card = pd.Card(card_name)
    dev = pd.DeviceEvents(ev)
    refs = pd.DeviceTrackRefs(off, src)
    out = pd.DeviceImpact(max(dev.n_particles, 1))
    pd.track_impact(card, dev, refs, out, d0_res, z0_res, seed, event_base)
    assert pd.last_launch_count() == (1 if dev.n_events > 0 and dev.n_particles > 0 else 0)
    return out.to_numpy(refs.n_tracks)


RES = ((20e-6, 40e-6), (30e-6, 60e-6))


@pytest.mark.parametrize("cfg,n_events", [(0, 600), (1, 150), (2, 10), (3, 1500), (4, 1500)])
def test_impact_of_oracle_tracks(cfg, n_events):
    from oracle import pdo

    ev = wl.generate(cfg, n_events)
    name = wl.config_card(cfg)
    seed = wl.CONFIGS[cfg]["seed"]
    o = pdo.simulate(pdo.Card(name), ev, seed, debug=False)
    off, src = o["trk_offsets"], o["trk_src"]
    assert len(src) > 1000
    # true values (zero resolution), then smeared
    ref = pdo.track_impact(pdo.Card(name), ev, off, src)
    got = _run_gpu(name, ev, off, src, (0, 0), (0, 0))
    _close(got["d0"], ref["d0_true"], "d0 true")
    _close(got["z0"], ref["z0_true"], "z0 true")
    assert np.all(got["d0_err"] == 0) and np.all(got["z0_err"] == 0)
    ref = pdo.track_impact(pdo.Card(name), ev, off, src, *RES, seed=seed, event_base=7)
    got = _run_gpu(name, ev, off, src, *RES, seed=seed, event_base=7)
    for k in ("d0", "z0"):
        _close(got[k], ref[k], k)
    for k in ("d0_err", "z0_err"):
        assert np.allclose(got[k], ref[k], rtol=1e-5, atol=0)
    print("cfg%d: %d tracks, |d0| up to %.3g m, |z0| up to %.3g m" % (cfg, len(src), np.abs(ref["d0_true"]).max(), np.abs(ref["z0_true"]).max()))


def _displaced(seed, sizes, pt_lo=0.15, r_max=1.0, charges=(-2, -1, 1, 2)):
    """All-charged events with vertices anywhere in the tracker volume and any direction of flight: circles that
    enclose the axis, circles that do not, looping low-pT tracks, large turning angles to the nearest point."""
    rng = np.random.default_rng(seed)
    events = []
    for n in sizes:
        parts = []
        for _ in range(n):
            pt = pt_lo * (2000.0 / pt_lo) ** rng.random()
            r, a = r_max * np.sqrt(rng.random()), rng.uniform(-np.pi, np.pi)
            parts.append(wl.particle(211, int(rng.choice(charges)), pt, rng.uniform(-2.5, 2.5), rng.uniform(-np.pi, np.pi), 0.13957,
                                     r * np.cos(a), r * np.sin(a), rng.uniform(-2.0, 2.0)))
        events.append(parts)
    return wl.from_lists(events)


def _all_tracks(ev):
    """Every particle a track (the kernel does not care how the list was selected)."""
    return ev.offsets.copy(), np.arange(int(ev.offsets[-1]), dtype=np.int32)


def test_displaced_vertices_ragged_events_and_edge_cases(tmp_path):
    from oracle import pdo

    sizes = [0, 1, 0, 2, 33, 0, 257, 1, 1500, 64, 0, 0, 31, 32, 900, 1025, 0]
    ev = _displaced(5, sizes)
    off, src = _all_tracks(ev)
    b = pdo.Card("cms_like")
    for name in ("cms_like", "aleph_like",
                 cards.variant(tmp_path / "rev.card", b.edges, b.nphi, bz=-2.5),
                 cards.variant(tmp_path / "nofield.card", b.edges, b.nphi, bz=0.0)):
        ref = pdo.track_impact(pdo.Card(name), ev, off, src, *RES, seed=3)
        got = _run_gpu(name, ev, off, src, *RES, seed=3)
        # a vertex half a turn away from the nearest point makes z0 two-valued (pd.h): leave out the rare tracks
        # whose turning angle to the nearest point is within 1e-4 of pi
        tr = pdo.track_impact(pdo.Card(name), ev, off, src)
        ok = np.ones(len(src), dtype=bool)
        if "nofield" not in name:
            pt = np.hypot(ev.px[src].astype(np.float64), ev.py[src].astype(np.float64))
            turn = np.abs(tr["z0_true"] - ev.vz[src]) * pt / np.maximum(np.abs(ev.pz[src].astype(np.float64)), 1e-30)
            bz = abs(float(np.float32(-2.5 if "rev" in name else {"cms_like": 3.8, "aleph_like": 1.5}[name])))
            rho = pt / (float(np.float32(0.299792458)) * np.abs(ev.charge[src]) * bz)
            ok = np.abs(turn / rho - np.pi) > 1e-4
        assert ok.mean() > 0.999
        # z0 = vz + (arc to the nearest point) * pz/pT: with vertices metres away from the axis at |eta| up to 2.5 the
        # two terms reach tens of metres and may cancel; the absolute bound scales with them
        scale = np.maximum(1.0, np.abs(ev.vz[src].astype(np.float64)) + np.abs(tr["z0_true"] - ev.vz[src]))
        _close(got["d0"][ok], ref["d0"][ok], name + " d0")
        _close(got["z0"][ok], ref["z0"][ok], name + " z0", atol=1e-6 * scale[ok])
    # only some particles are tracks, several thousand small events: offsets staged on chip vs read from global
    rng = np.random.default_rng(9)
    ev = _displaced(6, rng.poisson(3, 6000), r_max=0.05)
    keep = rng.random(int(ev.offsets[-1])) < 0.6
    src = np.nonzero(keep)[0].astype(np.int32)
    off = np.concatenate([[0], np.cumsum(keep)])[ev.offsets].astype(np.int64)
    ref = pdo.track_impact(pdo.Card("cms_like"), ev, off, src, *RES, seed=4)
    got = _run_gpu("cms_like", ev, off, src, *RES, seed=4)
    for k in ("d0", "z0"):
        _close(got[k], ref[k], k)
    # no tracks at all; zero events
    empty = np.zeros(ev.offsets.shape[0], dtype=np.int64)
    assert _run_gpu("cms_like", ev, empty, np.zeros(0, np.int32), *RES)["d0"].shape == (0,)
    z = wl.from_lists([])
    assert _run_gpu("cms_like", z, np.zeros(1, np.int64), np.zeros(0, np.int32), *RES)["d0"].shape == (0,)


def test_reproducible_split_invariant_and_fed_by_the_chain():
    import paper_2606_26089_b200 as pd
    from oracle import pdo

    cfg, n_events = 0, 800
    ev = wl.generate(cfg, n_events)
    name, seed = wl.config_card(cfg), 21
    card, dev = pd.Card(name), pd.DeviceEvents(ev)
    out = pd.DeviceOutputs(card, dev.n_events, dev.n_particles)
    pd.simulate(card, dev, out, seed)
    imp = pd.DeviceImpact(dev.n_particles)
    pd.track_impact(card, dev, out, imp, *RES, seed=seed)
    chain = out.to_numpy()
    n = int(chain["trk_offsets"][-1])
    a = imp.to_numpy(n)
    pd.track_impact(card, dev, out, imp, *RES, seed=seed)
    b = imp.to_numpy(n)
    for k in a:
        assert a[k].tobytes() == b[k].tobytes(), k
    # the same list uploaded again (pd_simulate's device output and a host copy of it are the same input)
    refs = pd.DeviceTrackRefs(chain["trk_offsets"], chain["trk_src"])
    imp2 = pd.DeviceImpact(dev.n_particles)
    pd.track_impact(card, dev, refs, imp2, *RES, seed=seed)
    c = imp2.to_numpy(n)
    for k in a:
        assert a[k].tobytes() == c[k].tobytes(), k
    # against the oracle run on ITS OWN track list (no oracle input comes from the CUDA path): a value depends only on
    # (seed, event, particle), so the two lists are matched by particle index
    o = pdo.simulate(pdo.Card(name), ev, seed, debug=False)
    ref = pdo.track_impact(pdo.Card(name), ev, o["trk_offsets"], o["trk_src"], *RES, seed=seed)
    common, ig, io = np.intersect1d(chain["trk_src"], o["trk_src"], return_indices=True)
    assert len(common) >= 0.999 * max(n, len(o["trk_src"]))  # near-edge efficiency decisions may differ
    for k in ("d0", "z0"):
        _close(a[k][ig], ref[k][io], k)
    # the second half of the batch as its own call with event_base
    cut = 300
    sub = wl.slice_events(ev, cut, n_events)
    m, mt = int(ev.offsets[cut]), int(chain["trk_offsets"][cut])
    h = _run_gpu(name, sub, chain["trk_offsets"][cut:] - mt, chain["trk_src"][mt:] - m, *RES, seed=seed, event_base=cut)
    for k in a:
        assert h[k].tobytes() == a[k][mt:].tobytes(), k


def test_unaligned_arrays_take_the_scalar_path():
    """The C ABI accepts any 4-byte-aligned arrays: with src / outputs off the 16-byte grid the kernel must fall back
    from its vector loads and stores and give the same bits."""
    import paper_2606_26089_b200 as pd
    from paper_2606_26089_b200 import binding as B
    import torch

    ev = _displaced(12, np.random.default_rng(4).poisson(40, 300), r_max=0.1)
    off, src = _all_tracks(ev)
    n = len(src)
    card, dev = pd.Card("cms_like"), pd.DeviceEvents(ev)
    refs = pd.DeviceTrackRefs(off, src)
    out = pd.DeviceImpact(n)
    pd.track_impact(card, dev, refs, out, *RES, seed=8)
    a = out.to_numpy(n)
    # same call with every array shifted by one element
    big_src = torch.zeros(n + 1, dtype=torch.int32, device="cuda")
    big_src[1:] = refs.src
    refs.src = big_src[1:]
    refs.c_trk = B.Tracks(n, B._tptr(refs.offsets), B._tptr(refs.src), *([None] * (len(B.TRACK_FIELDS) - 1)))
    assert refs.src.data_ptr() % 16 == 4
    out2 = pd.DeviceImpact(n + 1)
    views = {k: t[1:] for k, t in out2.t.items()}
    out2.c = B.Impact(*[B._tptr(views[k]) for k in out2.FIELDS])
    pd.track_impact(card, dev, refs, out2, *RES, seed=8)
    torch.cuda.synchronize()
    for k in a:
        assert views[k][:n].cpu().numpy().tobytes() == a[k].tobytes(), k


@pytest.mark.parametrize("card_name,cfg,n_events", [("cms_like", 0, 3000), ("cms_like", 2, 12), ("aleph_like", 4, 4000)])
def test_impact_from_the_chain_itself(card_name, cfg, n_events):
    """pd_options.impact: kernel P computes d0, z0 and their errors for the tracks it accepts (the particle is on chip there) and
    kernel T writes them beside the Track collection -- bit for bit what pd_track_impact gives after the step (the same
    device function), hence the oracle's values too (checked above); the collections themselves do not change.  With an event
    that goes through the big-tile path."""
    import paper_2606_26089_b200 as pd

    ev = wl.generate(cfg, n_events)
    if cfg == 0:
        big = wl.generate(2, 3)
        big = wl.Events(offsets=np.array([0, big.n_particles], dtype=np.int64),
                        **{k: getattr(big, k) for k in ("pid", "charge", "px", "py", "pz", "E", "vx", "vy", "vz")})
        ev = wl.concat_events([wl.slice_events(ev, 0, 1500), big, wl.slice_events(ev, 1500, n_events)])
    card = pd.Card(card_name)
    dev = pd.DeviceEvents(ev)
    res = ((2e-5, 1e-4), (3e-5, 2e-4))
    plain = pd.DeviceOutputs(card, dev.n_events, dev.n_particles)
    pd.simulate(card, dev, plain, 9, event_base=17)
    n_trk = int(plain.trk["offsets"][-1])
    assert n_trk > 1000
    want = pd.DeviceImpact(dev.n_particles)
    pd.track_impact(card, dev, plain, want, d0_res=res[0], z0_res=res[1], seed=9, event_base=17)
    w = want.to_numpy(n_trk)
    fused = pd.DeviceOutputs(card, dev.n_events, dev.n_particles, impact=res)
    assert fused.ws_bytes > plain.ws_bytes
    for t in fused.impact.t.values():
        t.fill_(float("nan"))
    pd.simulate(card, dev, fused, 9, event_base=17)
    assert pd.last_status(fused) == 0
    g = fused.impact.to_numpy(n_trk)
    for k in ("d0", "z0", "d0_err", "z0_err"):
        assert g[k].tobytes() == w[k].tobytes(), k
    a, b = plain.to_numpy(), fused.to_numpy()
    for k in a:
        assert a[k].tobytes() == b[k].tobytes(), k
    # nothing written beyond the tracks
    assert bool(fused.impact.t["d0"][n_trk:].isnan().all())
