"""CPU tests of the boundary: libpd.so builds, loads and exports every symbol include/pd.h declares;
card loading (pure host work) agrees with the oracle's independent loader; argument checking works
without a GPU.  No compute call is made here."""
import ctypes as C
import os
import re

import pytest

from paper_2606_26089_b200 import binding as B

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "pd.h")).read()
    declared = set(re.findall(r"\b(pd_[a-z_]+)\s*\(", hdr))
    assert declared == set(B.SYMBOLS), declared ^ set(B.SYMBOLS)
    L = B.lib()
    for name in declared:
        assert hasattr(L, name), name


@pytest.mark.parametrize("name,towers,bins,coord", [("cms_like", 5904, 94, 0), ("atlas_like", 4096, 64, 0), ("aleph_like", 19320, 92, 1)])
def test_builtin_cards_match_oracle_loader(name, towers, bins, coord):
    from oracle import pdo

    c = B.Card(name)
    o = pdo.Card(name)
    assert (c.n_towers, c.n_bins, c.grid_coord) == (towers, bins, coord) == (o.n_towers, o.n_bins, o.grid_coord)
    assert (c.bz, c.radius, c.half_length, c.n_eff_rows) == (o.bz, o.radius, o.half_length, o.n_eff_rows)


def test_card_file_and_errors(tmp_path):
    from oracle import pdo
    import cards

    o = pdo.Card("cms_like")
    path = cards.variant(tmp_path / "v.card", o.edges, o.nphi, bz=-2.5, ecal_thr=0.0)
    c = B.Card(path)
    assert c.n_towers == 5904 and abs(c.bz + 2.5) < 1e-6
    with pytest.raises(B.PdError) as e:
        B.Card("no_such_card")
    assert e.value.code == B.PD_ECARD
    bad = tmp_path / "bad.card"
    bad.write_text("bz = 1\nradius = 1\nhalf_length = 1\nedges = 0 1 0.5\nnphi = 4 4\n")
    with pytest.raises(B.PdError):
        B.Card(str(bad))
    # numbers out of range are refused at load (a negative threshold would make the kernel count neutrals it never
    # writes): thresholds / resolutions < 0 or NaN, efficiencies outside [0, 1], a |cos theta| cut outside (0, 1]
    for k, kw in enumerate((dict(ecal_thr=-0.1), dict(hcal_thr=float("nan")), dict(hcal=(0.05, -1.5, 0.0)), dict(track_res=(-0.01, 0.0)),
                            dict(eff=[(1.0, "inf", 0.0, 1.5, 1.2)]), dict(eff=[(1.0, 0.5, 0.0, 1.5, 0.9)]), dict(abs_costheta_max=1.5),
                            dict(bz=float("inf")), dict(eff=[(0.1, 1.0, 2.0, 1.0, 0.5)]))):
        with pytest.raises(B.PdError) as e:
            B.Card(cards.variant(tmp_path / ("r%d.card" % k), o.edges, o.nphi, **kw))
        assert e.value.code == B.PD_ECARD, kw


def test_argument_checking_without_gpu():
    L = B.lib()
    c = B.Card("cms_like")
    assert B.workspace_bytes(c, 1000, 60000) >= 16 + 24
    assert L.pd_workspace_bytes(c._h, -1, 0) == B.PD_EINVAL
    ev = B.Events(1, 10, None, None, None, None, None, None, None, None, None, None)
    trk, tow, efl = B.Tracks(), B.Towers(), B.EFlow()
    assert L.pd_simulate(c._h, C.byref(ev), 1, 0, C.byref(trk), C.byref(tow), C.byref(efl), None, None, 0, None) == B.PD_EINVAL
    assert L.pd_simulate(None, C.byref(ev), 1, 0, C.byref(trk), C.byref(tow), C.byref(efl), None, None, 0, None) == B.PD_EINVAL
    assert L.pd_strerror(B.PD_ECAPACITY).decode().startswith("output capacity")
    # options (pd_options): NULL and all-zero are the defaults; the workspace size depends on the events per tile;
    # negative values and non-zero reserved fields are refused; the library keeps no per-thread setting
    dflt = B.workspace_bytes(c, 1000, 60000)
    assert L.pd_workspace_bytes_ex(c._h, 1000, 60000, None) == dflt == L.pd_workspace_bytes(c._h, 1000, 60000)
    assert 0 < B.workspace_bytes(c, 1000, 60000, tile_events=1) != dflt
    assert B.workspace_bytes(c, 1000, 60000) == dflt  # ... and the call before left nothing behind
    bad = B.Options(-1)
    assert L.pd_workspace_bytes_ex(c._h, 1000, 60000, C.byref(bad)) == B.PD_EINVAL
    bad = B.Options(0)
    bad.reserved[3] = 1
    assert L.pd_workspace_bytes_ex(c._h, 1000, 60000, C.byref(bad)) == B.PD_EINVAL
    assert L.pd_simulate_ex(c._h, C.byref(ev), 1, 0, C.byref(trk), C.byref(tow), C.byref(efl), None, None, 0, C.byref(bad), None) == B.PD_EINVAL
    assert L.pd_card_upload(None) == B.PD_EINVAL


def test_no_cpu_fallback():
    import torch

    if torch.cuda.is_available():
        pytest.skip("GPU present")
    import importlib

    wl = importlib.import_module("workloads.generate")

    ev = wl.generate(0, 2)
    with pytest.raises((B.PdError, RuntimeError, AssertionError)):
        dev = B.DeviceEvents(ev, device="cuda")
        out = B.DeviceOutputs(B.Card("cms_like"), dev.n_events, dev.n_particles)
        B.simulate(B.Card("cms_like"), dev, out, 1)


def test_header_is_plain_c(tmp_path):
    """include/pd.h is a C ABI: it must compile as C99 on its own (no C++ types, no torch types)."""
    import subprocess

    src = tmp_path / "t.c"
    src.write_text('#include "pd.h"\nint main(void) { pd_events e; pd_condition c; pd_pileup_config p; (void)e; (void)c; (void)p; return 0; }\n')
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Wextra", "-pedantic", "-Werror", "-I", os.path.join(ROOT, "include"),
                           "-fsyntax-only", str(src)])


def test_host_buffers_packed_layout():
    """HostBuffers(packed=True): the 4-byte arrays of every collection are equally spaced rows of one block, in the
    order include/pd.h names for the strided copies of pd_simulate_host; packed=False: separate arrays.  (Host logic
    only: no CUDA call is made.)"""
    import importlib

    import numpy as np

    from paper_2606_26089_b200 import binding as B

    wl = importlib.import_module("workloads.generate")
    ev = wl.generate(0, 20)
    hb = B.HostBuffers(ev, pin=False, packed=True)
    n = ev.n_particles
    groups = ((hb.ev, ("pid", "px", "py", "pz", "E", "vx", "vy", "vz"), n), (hb.trk, ("src", "pid", "pt", "eta", "phi", "E", "eta_out", "phi_out"), n),
              (hb.tow, ("tower", "eta", "phi", "E", "Eem", "Ehad", "ET"), n), (hb.efl, ("src", "pt", "eta", "phi", "E"), 2 * n))
    for d, names, m in groups:
        ptrs = [d[k].data_ptr() for k in names]
        assert all(b - a == 4 * m for a, b in zip(ptrs, ptrs[1:])), names
        assert all(d[k].numel() == m for k in names)
    for k in ("pid", "charge", "px", "vz"):
        assert np.array_equal(hb.ev[k].numpy()[:n], getattr(ev, k))
    assert np.array_equal(hb.ev["offsets"].numpy(), ev.offsets)
    loose = B.HostBuffers(ev, pin=False, packed=False)
    assert np.array_equal(loose.ev["px"].numpy()[:n], ev.px) and loose.trk["pt"].numel() == n
