"""Helper: write detector-card text files (the `pd_load_card` / `pdo_load_card` file format) for tests.

Format ("key = values", '#' comments): name, bz, radius, half_length, kappa, grid (eta|theta),
edges (may repeat), nphi (may repeat), eff (pt_lo pt_hi aeta_lo aeta_hi eps; one line per row),
abs_costheta_max, track_res (a b), ecal_res (C S N), hcal_res (C S N), ecal_thr, hcal_thr;
ecal_res_eta / hcal_res_eta (aeta_lo aeta_hi C S N; one line per row), ecal_nsigma, hcal_nsigma, smear_tower_center,
track_res_eta (aeta_lo aeta_hi a b [species]; one line per row: DESIGN.md section 17, reading K4).
Per-species cards: an eff row may carry a sixth number and a track_res line a third one,
the species it applies to (1 electrons, 2 muons, 3 charged hadrons; 0 or absent: every charged particle).
"""
import numpy as np

BASE = {
    "cms_like": dict(bz=3.8, radius=1.29, half_length=3.0, ecal=(0.007, 0.07, 0.35), hcal=(0.05, 1.5, 0.0)),
    "atlas_like": dict(bz=2.0, radius=1.15, half_length=3.5, ecal=(0.0017, 0.101, 0.0), hcal=(0.0302, 0.5205, 0.0)),
    "aleph_like": dict(bz=1.5, radius=1.8, half_length=2.5, ecal=(0.009, 0.18, 0.0), hcal=(0.0, 0.85, 0.0),
                       abs_costheta_max=0.98),
}
DEFAULT_EFF = [(1.0, "inf", 0.0, 1.5, 0.97), (1.0, "inf", 1.5, 2.5, 0.85), (0.1, 1.0, 0.0, 2.5, 0.70)]


def card_text(edges, nphi, grid="eta", bz=3.8, radius=1.29, half_length=3.0, kappa=0.299792458,
              eff=DEFAULT_EFF, abs_costheta_max=None, track_res=(0.01, 1.5e-4), ecal=(0.007, 0.07, 0.35),
              hcal=(0.05, 1.5, 0.0), ecal_thr=0.5, hcal_thr=1.0, name="custom", track_res_species=None,
              ecal_res_eta=(), hcal_res_eta=(), ecal_nsigma=None, hcal_nsigma=None, smear_tower_center=None, track_res_eta=(), eflow_weighted=None, hcal_edges=None, hcal_nphi=None):
    lines = ["name = %s" % name, "bz = %r" % bz, "radius = %r" % radius, "half_length = %r" % half_length,
             "kappa = %r" % kappa, "grid = %s" % grid]
    edges = [float(x) for x in edges]
    for i in range(0, len(edges), 8):
        lines.append("edges = " + " ".join(repr(x) for x in edges[i:i + 8]))
    nphi = [int(x) for x in nphi]
    for i in range(0, len(nphi), 16):
        lines.append("nphi = " + " ".join(str(x) for x in nphi[i:i + 16]))
    if hcal_edges is not None:  # reading K6: the HCAL's own grid
        he = [float(x) for x in hcal_edges]
        for i in range(0, len(he), 8):
            lines.append("hcal_edges = " + " ".join(repr(x) for x in he[i:i + 8]))
        hn = [int(x) for x in hcal_nphi]
        for i in range(0, len(hn), 16):
            lines.append("hcal_nphi = " + " ".join(str(x) for x in hn[i:i + 16]))
    for row in eff:
        lines.append("eff = " + " ".join(str(x) for x in row))
    if abs_costheta_max is not None:
        lines.append("abs_costheta_max = %r" % abs_costheta_max)
    lines.append("track_res = %r %r" % tuple(track_res))
    for sp, ab in sorted((track_res_species or {}).items()):
        lines.append("track_res = %r %r %d" % (ab[0], ab[1], sp))
    for row in track_res_eta:  # (aeta_lo, aeta_hi, a, b[, species]): reading K4
        lines.append("track_res_eta = " + " ".join("inf" if x == "inf" else repr(float(x)) for x in row[:4]) + (" %d" % row[4] if len(row) > 4 else ""))
    lines.append("ecal_res = %r %r %r" % tuple(ecal))
    lines.append("hcal_res = %r %r %r" % tuple(hcal))
    for row in ecal_res_eta:  # (aeta_lo, aeta_hi, C, S, N): DESIGN.md section 17, reading K1
        lines.append("ecal_res_eta = " + " ".join(repr(float(x)) for x in row))
    for row in hcal_res_eta:
        lines.append("hcal_res_eta = " + " ".join(repr(float(x)) for x in row))
    if ecal_nsigma is not None:
        lines.append("ecal_nsigma = %r" % ecal_nsigma)
    if hcal_nsigma is not None:
        lines.append("hcal_nsigma = %r" % hcal_nsigma)
    if smear_tower_center is not None:
        lines.append("smear_tower_center = %d" % int(smear_tower_center))
    if eflow_weighted is not None:
        lines.append("eflow_weighted = %d" % int(eflow_weighted))  # reading K5
    lines.append("ecal_thr = %r" % ecal_thr)
    lines.append("hcal_thr = %r" % hcal_thr)
    return "\n".join(lines) + "\n"


def variant(path, base_edges, base_nphi, base="cms_like", **kw):
    """Write a card file that is `base` with fields replaced by kw; returns str(path).
    base_edges / base_nphi: the grid of the base card (taken from a loaded card by the caller)."""
    b = dict(BASE[base])
    args = dict(bz=b["bz"], radius=b["radius"], half_length=b["half_length"], ecal=b["ecal"], hcal=b["hcal"],
                grid="theta" if base == "aleph_like" else "eta")
    if "abs_costheta_max" in b:
        args["abs_costheta_max"] = b["abs_costheta_max"]
    args.update(kw)
    with open(path, "w") as f:
        f.write(card_text(np.asarray(base_edges, dtype=np.float64), base_nphi, **args))
    return str(path)
