"""ctypes binding of the fp64 CPU oracle (oracle/libpd_oracle.so).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this module.  It shares nothing with the CUDA path (paper_2606_26089_b200/).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

_lib = None

PDO_DROPPED, PDO_BARREL, PDO_ENDCAP, PDO_FACE_MASK, PDO_LOOPER = 0, 1, 2, 3, 4
NEAR_VERTEX, NEAR_FACE, NEAR_EFF, NEAR_ETA, NEAR_PHI, NEAR_LOWPT = 1, 2, 4, 8, 16, 32
NEAR_EEM, NEAR_EHAD, NEAR_NEM, NEAR_NHAD = 1, 2, 4, 8
PDO_OK, PDO_EINVAL, PDO_ECARD, PDO_ECAPACITY, PDO_EOVERRIDE = 0, -1, -2, -3, -4

_p = C.c_void_p


class _CardInfo(C.Structure):
    _fields_ = [("n_towers", C.c_int32), ("n_eta_bins", C.c_int32), ("grid_coord", C.c_int32),
                ("bz", C.c_float), ("radius", C.c_float), ("half_length", C.c_float),
                ("n_eff_rows", C.c_int32)]


class _Events(C.Structure):
    _fields_ = [("n_events", C.c_int64), ("n_particles", C.c_int64), ("offsets", _p), ("pid", _p),
                ("charge", _p), ("px", _p), ("py", _p), ("pz", _p), ("E", _p), ("vx", _p), ("vy", _p),
                ("vz", _p)]


class _Tracks(C.Structure):
    _fields_ = [("capacity", C.c_int64), ("offsets", _p), ("src", _p), ("pid", _p), ("charge", _p),
                ("pt", _p), ("eta", _p), ("phi", _p), ("E", _p), ("eta_out", _p), ("phi_out", _p)]


class _Towers(C.Structure):
    _fields_ = [("capacity", C.c_int64), ("offsets", _p), ("tower", _p), ("eta", _p), ("phi", _p),
                ("E", _p), ("Eem", _p), ("Ehad", _p), ("ET", _p)]


class _EFlow(C.Structure):
    _fields_ = [("capacity", C.c_int64), ("offsets", _p), ("cls", _p), ("src", _p), ("pt", _p),
                ("eta", _p), ("phi", _p), ("E", _p)]


class _Debug(C.Structure):
    _fields_ = [("status", _p), ("x", _p), ("y", _p), ("z", _p), ("eta_pos", _p), ("phi_pos", _p),
                ("tower", _p), ("accepted", _p), ("eps_row", _p), ("pt_smeared", _p), ("near", _p),
                ("tw_capacity", C.c_int64), ("tw_offsets", _p), ("tw_id", _p), ("Eem_true", _p),
                ("Ehad_true", _p), ("Tem", _p), ("Thad", _p), ("Eem_smeared", _p), ("Ehad_smeared", _p),
                ("tw_near", _p)]


class _Objects(C.Structure):
    _fields_ = [("n_events", C.c_int64), ("offsets", _p), ("cls", _p), ("pt", _p), ("eta", _p), ("phi", _p)]


class _Condition(C.Structure):
    _fields_ = [("field", C.c_int32), ("op", C.c_int32), ("use_abs", C.c_int32), ("n_values", C.c_int32),
                ("value", C.c_float), ("values", C.c_float * 8)]


FIELDS = {"pt": 0, "eta": 1, "phi": 2, "E": 3, "cls": 4}
OPS = {">": 0, ">=": 1, "<": 2, "<=": 3, "==": 4, "!=": 5, "in": 6, "not in": 7}


class _Overrides(C.Structure):
    _fields_ = [("face", _p), ("tower", _p), ("eps_row", _p), ("n_tower_ov", C.c_int64),
                ("tw_event", _p), ("tw_id", _p), ("tw_mask", _p), ("tw_value", _p), ("n_rejected", _p)]


def lib():
    global _lib
    if _lib is None:
        # PD_ORACLE_LIB: another build of oracle/pd_oracle.c (tests/test_oracle_sanitizers.py loads an ASan + UBSan build this way)
        L = C.CDLL(os.environ.get("PD_ORACLE_LIB") or _build.build())
        L.pdo_load_card.argtypes = [C.c_char_p, C.POINTER(_p)]
        L.pdo_free_card.argtypes = [_p]
        L.pdo_free_card.restype = None
        L.pdo_card_info.argtypes = [_p, C.POINTER(_CardInfo)]
        L.pdo_card_grid.argtypes = [_p, _p, _p, _p]
        L.pdo_tower_centre.argtypes = [_p, C.c_int32, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.pdo_tower_position.argtypes = [_p, C.c_uint64, C.c_int64, C.c_int32, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.pdo_simulate.argtypes = [_p, C.POINTER(_Events), C.c_uint64, C.c_int64, C.POINTER(_Tracks),
                                   C.POINTER(_Towers), C.POINTER(_EFlow), C.POINTER(_Debug),
                                   C.POINTER(_Overrides)]
        L.pdo_strerror.argtypes = [C.c_int]
        L.pdo_strerror.restype = C.c_char_p
        L.pdo_philox4x32_10.argtypes = [C.POINTER(C.c_uint32), C.POINTER(C.c_uint32), C.POINTER(C.c_uint32)]
        L.pdo_philox4x32_10.restype = None
        L.pdo_rng_block.argtypes = [C.c_uint64, C.c_int64, C.c_uint32, C.c_uint32, C.POINTER(C.c_uint32)]
        L.pdo_rng_block.restype = None
        for name in ("pdo_uniform", "pdo_uniform_pos"):
            getattr(L, name).argtypes = [C.c_uint32]
            getattr(L, name).restype = C.c_double
        L.pdo_normal.argtypes = [C.c_uint32, C.c_uint32]
        L.pdo_normal.restype = C.c_double
        L.pdo_lognormal.argtypes = [C.c_double] * 3
        L.pdo_lognormal.restype = C.c_double
        L.pdo_propagate.argtypes = [_p, C.c_int] + [C.c_double] * 6 + [C.POINTER(C.c_double)] * 6
        L.pdo_tower_index.argtypes = [_p, C.c_double, C.c_double]
        L.pdo_tower_index.restype = C.c_int32
        L.pdo_efficiency.argtypes = [_p, C.c_double, C.c_double, C.c_double, C.POINTER(C.c_int)]
        L.pdo_efficiency.restype = C.c_double
        L.pdo_efficiency_species.argtypes = [_p, C.c_double, C.c_double, C.c_double, C.c_int, C.POINTER(C.c_int)]
        L.pdo_efficiency_species.restype = C.c_double
        L.pdo_track_resolution.argtypes = [_p, C.c_int, C.c_double, C.c_double, C.c_double, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.pdo_track_resolution.restype = C.c_int
        L.pdo_eflow_weight.argtypes = [C.c_double] * 4
        L.pdo_eflow_weight.restype = C.c_double
        L.pdo_pileup_merge.argtypes = [C.POINTER(_Events), C.POINTER(_Events), C.c_double, C.c_double, C.c_double, C.c_int,
                                       C.c_uint64, C.c_int64, C.c_int64] + [_p] * 12
        L.pdo_filter_eflow.argtypes = [C.c_int64] + [_p] * 7 + [C.POINTER(_Condition), C.c_int32, C.c_int32] + [_p] * 8
        L.pdo_event_features.argtypes = [C.POINTER(_Objects), C.c_double, C.c_double] + [_p] * 9
        L.pdo_truth_features.argtypes = [C.POINTER(_Events), C.c_int] + [_p] * 4
        L.pdo_impact_true.argtypes = [_p, C.c_int] + [C.c_double] * 6 + [C.POINTER(C.c_double)] * 2
        L.pdo_track_impact.argtypes = [_p, C.POINTER(_Events), _p, _p] + [C.c_double] * 4 + [C.c_uint64, C.c_int64] + [_p] * 6
        _lib = L
    return _lib


def _ptr(a):
    return None if a is None else a.ctypes.data_as(_p)


class OracleError(RuntimeError):
    def __init__(self, code, n_rejected=0):
        super().__init__("oracle: %s (code %d, rejected overrides %d)"
                         % (lib().pdo_strerror(code).decode(), code, n_rejected))
        self.code = code
        self.n_rejected = n_rejected


class Card:
    """A detector card: "cms_like" | "atlas_like" | "aleph_like" | path of a card text file."""

    def __init__(self, name_or_path: str):
        self._h = _p()
        rc = lib().pdo_load_card(str(name_or_path).encode(), C.byref(self._h))
        if rc != PDO_OK:
            raise OracleError(rc)
        info = _CardInfo()
        lib().pdo_card_info(self._h, C.byref(info))
        self.n_towers, self.n_bins, self.grid_coord = info.n_towers, info.n_eta_bins, info.grid_coord
        self.bz, self.radius, self.half_length = info.bz, info.radius, info.half_length
        self.n_eff_rows = info.n_eff_rows
        self.edges = np.zeros(self.n_bins + 1)
        self.nphi = np.zeros(self.n_bins, dtype=np.int32)
        self.offset = np.zeros(self.n_bins, dtype=np.int32)
        lib().pdo_card_grid(self._h, _ptr(self.edges), _ptr(self.nphi), _ptr(self.offset))

    def __del__(self):
        if getattr(self, "_h", None):
            lib().pdo_free_card(self._h)
            self._h = None

    def tower_centre(self, tower: int):
        e, p = C.c_double(), C.c_double()
        if lib().pdo_tower_centre(self._h, int(tower), C.byref(e), C.byref(p)) != PDO_OK:
            raise OracleError(PDO_EINVAL)
        return e.value, p.value

    def tower_index(self, coord: float, phi: float, det: int = 0) -> int:
        """tower of a hit; det: section of the deposit (0 ECAL, 1 HCAL), which matters on a card with two grids (reading K6)"""
        L = lib()
        L.pdo_tower_index_det.argtypes = [_p, C.c_int, C.c_double, C.c_double]
        L.pdo_tower_index_det.restype = C.c_int32
        return int(L.pdo_tower_index_det(self._h, int(det), float(coord), float(phi)))

    def hcal_grid(self):
        """(edges, nphi, base) of the HCAL's own grid, or None for a card with one grid (reading K6)"""
        L = lib()
        L.pdo_card_hcal_grid.argtypes = [_p, C.c_void_p, C.c_void_p, C.c_void_p]
        n = int(L.pdo_card_hcal_grid(self._h, None, None, None))
        if n <= 0:
            return None
        e, p, b = np.zeros(n + 1), np.zeros(n, dtype=np.int32), C.c_int32(0)
        L.pdo_card_hcal_grid(self._h, e.ctypes.data_as(C.c_void_p), p.ctypes.data_as(C.c_void_p), C.cast(C.byref(b), C.c_void_p))
        return e, p, int(b.value)

    def efficiency(self, pt, eta_mom, abs_costheta=0.0, species=None):
        """(eps, row) of the card's table; species: None (a charged hadron), 1 electron, 2 muon, 3 charged hadron."""
        row = C.c_int(-1)
        if species is None:
            eps = lib().pdo_efficiency(self._h, float(pt), float(eta_mom), float(abs_costheta), C.byref(row))
        else:
            eps = lib().pdo_efficiency_species(self._h, float(pt), float(eta_mom), float(abs_costheta), int(species), C.byref(row))
        return eps, row.value

    def track_resolution(self, species, px, py, pz):
        """(row, a, b) of reading K4 / J2 for a track of the species (1 electron, 2 muon, 3 charged hadron)"""
        a, b = C.c_double(), C.c_double()
        row = lib().pdo_track_resolution(self._h, int(species), float(px), float(py), float(pz), C.byref(a), C.byref(b))
        return int(row), a.value, b.value

    def propagate(self, q, px, py, pz, vx=0.0, vy=0.0, vz=0.0):
        out = [C.c_double() for _ in range(6)]
        st = lib().pdo_propagate(self._h, int(q), float(px), float(py), float(pz), float(vx), float(vy),
                                 float(vz), *[C.byref(o) for o in out])
        x, y, z, alpha, eta_pos, phi_pos = [o.value for o in out]
        return dict(status=st, x=x, y=y, z=z, alpha=alpha, eta_pos=eta_pos, phi_pos=phi_pos)

    def impact_true(self, q, px, py, pz, vx=0.0, vy=0.0, vz=0.0):
        """pdo_impact_true (reading I1): (d0, z0) of one trajectory, metres."""
        d0, z0 = C.c_double(), C.c_double()
        rc = lib().pdo_impact_true(self._h, int(q), float(px), float(py), float(pz), float(vx), float(vy), float(vz),
                                   C.byref(d0), C.byref(z0))
        if rc != 0:
            raise OracleError(rc)
        return d0.value, z0.value


def philox(ctr, key):
    c = (C.c_uint32 * 4)(*ctr)
    k = (C.c_uint32 * 2)(*key)
    o = (C.c_uint32 * 4)()
    lib().pdo_philox4x32_10(c, k, o)
    return tuple(int(x) for x in o)


def rng_block(seed, event, obj, stream):
    o = (C.c_uint32 * 4)()
    lib().pdo_rng_block(int(seed), int(event), int(obj), int(stream), o)
    return tuple(int(x) for x in o)


def uniform(x):
    return lib().pdo_uniform(int(x))


def uniform_pos(x):
    return lib().pdo_uniform_pos(int(x))


def normal(xa, xb):
    return lib().pdo_normal(int(xa), int(xb))


def lognormal(m, s, z):
    return lib().pdo_lognormal(float(m), float(s), float(z))


def tower_position(card: Card, seed: int, event: int, tower: int):
    """Reported (eta, phi) of a tower: uniform inside the cell if the card smears tower centres (reading K3)."""
    e, p = C.c_double(), C.c_double()
    if lib().pdo_tower_position(card._h, int(seed), int(event), int(tower), C.byref(e), C.byref(p)) != PDO_OK:
        raise OracleError(PDO_EINVAL)
    return e.value, p.value


def simulate(card: Card, ev, seed: int, event_base: int = 0, overrides: dict | None = None,
             debug: bool = True) -> dict:
    """Run the oracle on an `Events`-like record (attributes offsets, pid, charge, px..vz).

    Returns a dict of numpy arrays: trk_*, tow_*, efl_* (CSR, trimmed to their totals) and, with
    debug=True, per-particle dbg_* and per-deposited-tower dtw_* arrays.
    overrides: dict with optional keys face (int8[n], -1 none), tower (int32[n], -2 none),
    eps_row (int8[n], -2 none), tw_event (int64[m]), tw_id (int32[m]), tw_mask (uint8[m]), tw_value (uint8[m]).
    """
    L = lib()
    ne, n = int(ev.offsets.shape[0] - 1), int(ev.offsets[-1])
    keep = [np.ascontiguousarray(getattr(ev, k)) for k in
            ("offsets", "pid", "charge", "px", "py", "pz", "E", "vx", "vy", "vz")]
    cevt = _Events(ne, n, *[_ptr(a) for a in keep])
    cap = max(n, 1)
    i64, i32, i8, u8, f8 = np.int64, np.int32, np.int8, np.uint8, np.float64
    z = lambda m, t: np.zeros(m, dtype=t)  # noqa: E731
    T = dict(offsets=z(ne + 1, i64), src=z(cap, i32), pid=z(cap, i32), charge=z(cap, i8), pt=z(cap, f8),
             eta=z(cap, f8), phi=z(cap, f8), E=z(cap, f8), eta_out=z(cap, f8), phi_out=z(cap, f8))
    W = dict(offsets=z(ne + 1, i64), tower=z(cap, i32), eta=z(cap, f8), phi=z(cap, f8), E=z(cap, f8),
             Eem=z(cap, f8), Ehad=z(cap, f8), ET=z(cap, f8))
    F = dict(offsets=z(ne + 1, i64), cls=z(2 * cap, i8), src=z(2 * cap, i32), pt=z(2 * cap, f8),
             eta=z(2 * cap, f8), phi=z(2 * cap, f8), E=z(2 * cap, f8))
    ct = _Tracks(cap, *[_ptr(T[k]) for k in ("offsets", "src", "pid", "charge", "pt", "eta", "phi", "E", "eta_out", "phi_out")])
    cw = _Towers(cap, *[_ptr(W[k]) for k in ("offsets", "tower", "eta", "phi", "E", "Eem", "Ehad", "ET")])
    cf = _EFlow(2 * cap, *[_ptr(F[k]) for k in ("offsets", "cls", "src", "pt", "eta", "phi", "E")])
    D = None
    cd = None
    if debug:
        D = dict(status=z(cap, u8), x=z(cap, f8), y=z(cap, f8), z=z(cap, f8), eta_pos=z(cap, f8),
                 phi_pos=z(cap, f8), tower=z(cap, i32), accepted=z(cap, u8), eps_row=z(cap, i8),
                 pt_smeared=z(cap, f8), near=z(cap, np.uint32))
        DT = dict(tw_offsets=z(ne + 1, i64), tw_id=z(cap, i32), Eem_true=z(cap, f8), Ehad_true=z(cap, f8),
                  Tem=z(cap, f8), Thad=z(cap, f8), Eem_smeared=z(cap, f8), Ehad_smeared=z(cap, f8),
                  tw_near=z(cap, u8))
        cd = _Debug(*[_ptr(D[k]) for k in ("status", "x", "y", "z", "eta_pos", "phi_pos", "tower",
                                           "accepted", "eps_row", "pt_smeared", "near")],
                    cap, *[_ptr(DT[k]) for k in ("tw_offsets", "tw_id", "Eem_true", "Ehad_true", "Tem",
                                                 "Thad", "Eem_smeared", "Ehad_smeared", "tw_near")])
    co = None
    n_rej = np.zeros(1, dtype=i64)
    if overrides:
        ov = {}
        for k, t in (("face", i8), ("tower", i32), ("eps_row", i8)):
            ov[k] = None if overrides.get(k) is None else np.ascontiguousarray(overrides[k], dtype=t)
        m = 0
        for k, t in (("tw_event", i64), ("tw_id", i32), ("tw_mask", u8), ("tw_value", u8)):
            ov[k] = None if overrides.get(k) is None else np.ascontiguousarray(overrides[k], dtype=t)
            if ov[k] is not None:
                m = int(ov[k].shape[0])
        co = _Overrides(_ptr(ov["face"]), _ptr(ov["tower"]), _ptr(ov["eps_row"]), m, _ptr(ov["tw_event"]),
                        _ptr(ov["tw_id"]), _ptr(ov["tw_mask"]), _ptr(ov["tw_value"]), _ptr(n_rej))
    rc = L.pdo_simulate(card._h, C.byref(cevt), int(seed) & (2**64 - 1), int(event_base), C.byref(ct),
                        C.byref(cw), C.byref(cf), C.byref(cd) if cd is not None else None,
                        C.byref(co) if co is not None else None)
    if rc != PDO_OK:
        raise OracleError(rc, int(n_rej[0]))
    out = {}
    for prefix, d in (("trk", T), ("tow", W), ("efl", F)):
        tot = int(d["offsets"][-1])
        for k, a in d.items():
            out["%s_%s" % (prefix, k)] = a if k == "offsets" else a[:tot]
    if debug:
        for k, a in D.items():
            out["dbg_" + k] = a[:n]
        tot = int(DT["tw_offsets"][-1])
        for k, a in DT.items():
            out["dtw_" + k.replace("tw_", "")] = a if k == "tw_offsets" else a[:tot]
    return out


def event_features(offsets, cls, pt, eta, phi, dr_max: float = 0.4, fsr_dr: float = 0.0) -> dict:
    """pdo_event_features on an EFlow-like CSR collection (Eq. 1): per event ht, met_x,
    met_y, met; per object iso_charged, iso_neutral, iso_photon, r_iso, and iso_amb (pT of the objects whose
    dR is within 1e-6 of a cone edge).  All float64."""
    offsets = np.ascontiguousarray(offsets, dtype=np.int64)
    cls = np.ascontiguousarray(cls, dtype=np.int8)
    pt, eta, phi = (np.ascontiguousarray(a, dtype=np.float32) for a in (pt, eta, phi))
    ne, n = int(offsets.shape[0] - 1), int(offsets[-1])
    assert cls.shape[0] >= n and pt.shape[0] >= n and eta.shape[0] >= n and phi.shape[0] >= n
    ev = {k: np.zeros(max(ne, 1), dtype=np.float64) for k in ("ht", "met_x", "met_y", "met")}
    ob = {k: np.zeros(max(n, 1), dtype=np.float64) for k in ("iso_charged", "iso_neutral", "iso_photon", "r_iso", "iso_amb")}
    o = _Objects(ne, _ptr(offsets), _ptr(cls), _ptr(pt), _ptr(eta), _ptr(phi))
    rc = lib().pdo_event_features(C.byref(o), float(dr_max), float(fsr_dr), _ptr(ev["ht"]), _ptr(ev["met_x"]),
                                  _ptr(ev["met_y"]), _ptr(ev["met"]), _ptr(ob["iso_charged"]), _ptr(ob["iso_neutral"]),
                                  _ptr(ob["iso_photon"]), _ptr(ob["r_iso"]), _ptr(ob["iso_amb"]))
    if rc != 0:
        raise OracleError(rc)
    out = {k: v[:ne] for k, v in ev.items()}
    out.update({k: v[:n] for k, v in ob.items()})
    return out


def make_conditions(conditions, ctype=_Condition):
    """[{field, op, value, abs}] (the paper's Table C.13 grammar) -> ctypes array."""
    arr = (ctype * max(len(conditions), 1))()
    for k, c in enumerate(conditions):
        arr[k].field, arr[k].op, arr[k].use_abs = FIELDS[c["field"]], OPS[c["op"]], int(bool(c.get("abs", False)))
        if c["op"] in ("in", "not in"):
            vals = list(c["value"])
            assert len(vals) <= 8
            arr[k].n_values = len(vals)
            for j, v in enumerate(vals):
                arr[k].values[j] = float(v)
        else:
            arr[k].n_values, arr[k].value = 0, float(c["value"])
    return arr


def filter_eflow(offsets, cls, src, pt, eta, phi, E, conditions, combine: str = "all") -> dict:
    """pdo_filter_eflow (Table C.13): returns offsets, cls, src, pt, eta, phi, E of the survivors and keep."""
    offsets = np.ascontiguousarray(offsets, dtype=np.int64)
    ne, n = int(offsets.shape[0] - 1), int(offsets[-1])
    cls, src = np.ascontiguousarray(cls, dtype=np.int8), np.ascontiguousarray(src, dtype=np.int32)
    fl = [np.ascontiguousarray(a, dtype=np.float32) for a in (pt, eta, phi, E)]
    out = {"offsets": np.zeros(ne + 1, dtype=np.int64), "cls": np.zeros(max(n, 1), dtype=np.int8), "src": np.zeros(max(n, 1), dtype=np.int32)}
    for k in ("pt", "eta", "phi", "E"):
        out[k] = np.zeros(max(n, 1), dtype=np.float32)
    keep = np.zeros(max(n, 1), dtype=np.uint8)
    conds = make_conditions(conditions)
    rc = lib().pdo_filter_eflow(ne, _ptr(offsets), _ptr(cls), _ptr(src), *[_ptr(a) for a in fl], conds, len(conditions),
                                1 if combine == "any" else 0, _ptr(out["offsets"]), _ptr(out["cls"]), _ptr(out["src"]),
                                _ptr(out["pt"]), _ptr(out["eta"]), _ptr(out["phi"]), _ptr(out["E"]), _ptr(keep))
    if rc != 0:
        raise OracleError(rc)
    m = int(out["offsets"][-1])
    res = {k: (v if k == "offsets" else v[:m]) for k, v in out.items()}
    res["keep"] = keep[:n]
    return res


def _events_struct(ev):
    keep = [np.ascontiguousarray(getattr(ev, k)) for k in ("offsets", "pid", "charge", "px", "py", "pz", "E", "vx", "vy", "vz")]
    return _Events(int(ev.offsets.shape[0] - 1), int(ev.offsets[-1]), *[_ptr(a) for a in keep]), keep


def _vp(a):
    return a.ctypes.data_as(C.c_void_p)


def eflow_weight(T, V, Ec, sigma_c):
    """pdo_eflow_weight (reading K5)"""
    return float(lib().pdo_eflow_weight(float(T), float(V), float(Ec), float(sigma_c)))


def pileup_merge(hs, pool, mean_pileup: float, sigma_z: float = 0.053, max_z_spread: float = 0.25,
                 smear_hs_vertex: bool = True, seed: int = 0, event_base: int = 0, sigma_t: float = 160e-12,
                 max_t_spread: float = 800e-12) -> dict:
    """pdo_pileup_merge_t (Listing 8, Table C.9): returns offsets, pid, charge, px..vz, is_pu, vt, n_pileup."""
    chs, k1 = _events_struct(hs)
    cpool, k2 = _events_struct(pool)
    ne = chs.n_events
    off = np.zeros(ne + 1, dtype=np.int64)
    npu = np.zeros(max(ne, 1), dtype=np.int32)
    dt = dict(pid=np.int32, charge=np.int8, px=np.float32, py=np.float32, pz=np.float32, E=np.float32, vx=np.float32,
              vy=np.float32, vz=np.float32, is_pu=np.uint8)
    L = lib()
    L.pdo_pileup_merge_t.restype = C.c_int
    L.pdo_pileup_merge_t.argtypes = [C.POINTER(_Events), C.POINTER(_Events), C.c_double, C.c_double, C.c_double, C.c_double, C.c_double,
                                     C.c_int, C.c_uint64, C.c_int64, C.c_int64] + [C.c_void_p] * 13
    cap = 0
    for _ in range(2):  # first pass sizes the output (PDO_ECAPACITY with complete offsets), second fills it
        out = {k: np.zeros(max(cap, 1), dtype=d) for k, d in dt.items()}
        vt = np.zeros(max(cap, 1), dtype=np.float32)
        rc = L.pdo_pileup_merge_t(C.byref(chs), C.byref(cpool), float(mean_pileup), float(sigma_z), float(max_z_spread),
                                  float(sigma_t), float(max_t_spread), int(bool(smear_hs_vertex)), int(seed) & (2**64 - 1),
                                  int(event_base), cap, _vp(off), *[_vp(out[k]) for k in dt], _vp(npu), _vp(vt))
        if rc == 0:
            break
        if rc != -3:
            raise OracleError(rc)
        cap = int(off[-1])
    res = {k: v[: int(off[-1])] for k, v in out.items()}
    res["vt"] = vt[: int(off[-1])]
    res["offsets"], res["n_pileup"] = off, npu[:ne]
    return res


def track_impact(card: Card, ev, trk_offsets, trk_src, d0_res=(0.0, 0.0), z0_res=(0.0, 0.0), seed: int = 0,
                 event_base: int = 0) -> dict:
    """pdo_track_impact (readings I1..I3): d0_true, z0_true, d0, z0, d0_err, z0_err per track (fp64, metres)."""
    cev, keep = _events_struct(ev)
    off = np.ascontiguousarray(trk_offsets, dtype=np.int64)
    src = np.ascontiguousarray(trk_src, dtype=np.int32)
    n = int(off[-1])
    out = {k: np.zeros(max(n, 1), dtype=np.float64) for k in ("d0_true", "z0_true", "d0", "z0", "d0_err", "z0_err")}
    rc = lib().pdo_track_impact(card._h, C.byref(cev), _ptr(off), _ptr(src), float(d0_res[0]), float(d0_res[1]),
                                float(z0_res[0]), float(z0_res[1]), int(seed) & (2**64 - 1), int(event_base),
                                *[_ptr(out[k]) for k in ("d0_true", "z0_true", "d0", "z0", "d0_err", "z0_err")])
    if rc != 0:
        raise OracleError(rc)
    return {k: v[:n] for k, v in out.items()}


def truth_features(ev, skip_neutrinos: bool = True) -> dict:
    """pdo_truth_features (readings T1, T2): ht, met_x, met_y, met per event over the truth collection."""
    cev, keep = _events_struct(ev)
    ne = cev.n_events
    out = {k: np.zeros(max(ne, 1), dtype=np.float64) for k in ("ht", "met_x", "met_y", "met")}
    rc = lib().pdo_truth_features(C.byref(cev), int(bool(skip_neutrinos)), *[_ptr(out[k]) for k in ("ht", "met_x", "met_y", "met")])
    if rc != 0:
        raise OracleError(rc)
    return {k: v[:ne] for k, v in out.items()}
