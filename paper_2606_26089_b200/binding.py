"""Thin ctypes binding of libpd.so (include/pd.h).  Argument marshalling only: every step of the chain
runs in the CUDA kernels of the library.  torch is used for device memory and streams.

There is no CPU fallback: if libpd.so cannot be built/loaded, importing `lib()` raises; if no CUDA
device is present `simulate` raises PdError(PD_ECUDA)."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

PD_OK, PD_EINVAL, PD_ECARD, PD_ECAPACITY, PD_EWORKSPACE, PD_ECUDA, PD_EEVENTSIZE = 0, -1, -2, -3, -4, -5, -6
PD_DROPPED, PD_BARREL, PD_ENDCAP, PD_FACE_MASK, PD_LOOPER = 0, 1, 2, 3, 4
PD_DEC_EEM, PD_DEC_EHAD, PD_DEC_NEM, PD_DEC_NHAD = 1, 2, 4, 8

# every symbol include/pd.h declares
SYMBOLS = ("pd_load_card", "pd_free_card", "pd_card_info", "pd_workspace_bytes", "pd_simulate", "pd_last_status",
           "pd_last_launch_count", "pd_workspace_bytes_ex", "pd_simulate_ex", "pd_card_upload", "pd_event_features", "pd_filter_workspace_bytes", "pd_filter_eflow", "pd_pileup_workspace_bytes", "pd_pileup_merge", "pd_track_impact", "pd_truth_workspace_bytes", "pd_truth_features", "pd_truth_features_static", "pd_simulate_host", "pd_strerror")

_p = C.c_void_p
_lib = None


class CardInfo(C.Structure):
    _fields_ = [("n_towers", C.c_int32), ("n_eta_bins", C.c_int32), ("grid_coord", C.c_int32), ("bz", C.c_float),
                ("radius", C.c_float), ("half_length", C.c_float), ("n_eff_rows", C.c_int32)]


class Features(C.Structure):
    _fields_ = [(k, _p) for k in ("ht", "met_x", "met_y", "met", "iso_charged", "iso_neutral", "iso_photon", "r_iso")]


class Condition(C.Structure):
    _fields_ = [("field", C.c_int32), ("op", C.c_int32), ("use_abs", C.c_int32), ("n_values", C.c_int32),
                ("value", C.c_float), ("values", C.c_float * 8)]


FIELDS = {"pt": 0, "eta": 1, "phi": 2, "E": 3, "cls": 4}
OPS = {">": 0, ">=": 1, "<": 2, "<=": 3, "==": 4, "!=": 5, "in": 6, "not in": 7}


class ImpactConfig(C.Structure):
    _fields_ = [("d0_a", C.c_float), ("d0_b", C.c_float), ("z0_a", C.c_float), ("z0_b", C.c_float)]


class Impact(C.Structure):
    _fields_ = [(k, _p) for k in ("d0", "z0", "d0_err", "z0_err")]


class Options(C.Structure):
    """pd_options"""
    _fields_ = [("tile_events", C.c_int32), ("reserved", C.c_int32 * 7), ("impact_config", C.POINTER(ImpactConfig)),
                ("impact", C.POINTER(Impact))]


class PileupConfig(C.Structure):
    _fields_ = [("mean_pileup", C.c_float), ("sigma_z", C.c_float), ("max_z_spread", C.c_float), ("smear_hs_vertex", C.c_int32),
                ("sigma_t", C.c_float), ("max_t_spread", C.c_float)]


class MergedEvents(C.Structure):
    _fields_ = [("capacity", C.c_int64)] + [(k, _p) for k in ("offsets", "pid", "charge", "px", "py", "pz", "E", "vx", "vy", "vz",
                                                        "is_pu", "n_pileup", "vt")]


class Events(C.Structure):
    _fields_ = [("n_events", C.c_int64), ("n_particles", C.c_int64), ("offsets", _p), ("pid", _p), ("charge", _p),
                ("px", _p), ("py", _p), ("pz", _p), ("E", _p), ("vx", _p), ("vy", _p), ("vz", _p)]


class Tracks(C.Structure):
    _fields_ = [("capacity", C.c_int64), ("offsets", _p), ("src", _p), ("pid", _p), ("charge", _p), ("pt", _p),
                ("eta", _p), ("phi", _p), ("E", _p), ("eta_out", _p), ("phi_out", _p)]


class Towers(C.Structure):
    _fields_ = [("capacity", C.c_int64), ("offsets", _p), ("tower", _p), ("eta", _p), ("phi", _p), ("E", _p),
                ("Eem", _p), ("Ehad", _p), ("ET", _p)]


class EFlow(C.Structure):
    _fields_ = [("capacity", C.c_int64), ("offsets", _p), ("cls", _p), ("src", _p), ("pt", _p), ("eta", _p),
                ("phi", _p), ("E", _p)]


class Debug(C.Structure):
    _fields_ = [("status", _p), ("eta_pos", _p), ("phi_pos", _p), ("tower", _p), ("accepted", _p), ("eps_row", _p),
                ("pt_smeared", _p), ("tw_first", _p), ("tw_Eem_true", _p), ("tw_Ehad_true", _p), ("tw_Tem", _p),
                ("tw_Thad", _p), ("tw_Eem_smeared", _p), ("tw_Ehad_smeared", _p), ("tw_decisions", _p)]


TRACK_FIELDS = (("src", "int32"), ("pid", "int32"), ("charge", "int8"), ("pt", "float32"), ("eta", "float32"),
                ("phi", "float32"), ("E", "float32"), ("eta_out", "float32"), ("phi_out", "float32"))
TOWER_FIELDS = (("tower", "int32"), ("eta", "float32"), ("phi", "float32"), ("E", "float32"), ("Eem", "float32"),
                ("Ehad", "float32"), ("ET", "float32"))
EFLOW_FIELDS = (("cls", "int8"), ("src", "int32"), ("pt", "float32"), ("eta", "float32"), ("phi", "float32"),
                ("E", "float32"))
DEBUG_FIELDS = (("status", "uint8"), ("eta_pos", "float32"), ("phi_pos", "float32"), ("tower", "int32"),
                ("accepted", "uint8"), ("eps_row", "int8"), ("pt_smeared", "float32"), ("tw_first", "uint8"),
                ("tw_Eem_true", "float32"), ("tw_Ehad_true", "float32"), ("tw_Tem", "float32"), ("tw_Thad", "float32"),
                ("tw_Eem_smeared", "float32"), ("tw_Ehad_smeared", "float32"), ("tw_decisions", "uint8"))
EVENT_FIELDS = (("offsets", "int64"), ("pid", "int32"), ("charge", "int8"), ("px", "float32"), ("py", "float32"),
                ("pz", "float32"), ("E", "float32"), ("vx", "float32"), ("vy", "float32"), ("vz", "float32"))


def lib():
    """Load libpd.so (building it in-tree if stale).  Raises if that is impossible: no fallback."""
    global _lib
    if _lib is None:
        path = _build.LIB
        if not os.path.exists(path) or os.environ.get("PD_REBUILD"):
            path = _build.build()
        L = C.CDLL(path)
        L.pd_load_card.argtypes = [C.c_char_p, C.POINTER(_p)]
        L.pd_free_card.argtypes = [_p]
        L.pd_free_card.restype = None
        L.pd_card_info.argtypes = [_p, C.POINTER(CardInfo)]
        L.pd_workspace_bytes.argtypes = [_p, C.c_int64, C.c_int64]
        L.pd_workspace_bytes.restype = C.c_int64
        L.pd_simulate.argtypes = [_p, C.POINTER(Events), C.c_uint64, C.c_int64, C.POINTER(Tracks), C.POINTER(Towers),
                                  C.POINTER(EFlow), C.POINTER(Debug), _p, C.c_int64, _p]
        L.pd_last_status.argtypes = [_p, _p]
        L.pd_last_launch_count.argtypes = []
        L.pd_workspace_bytes_ex.argtypes = [_p, C.c_int64, C.c_int64, C.POINTER(Options)]
        L.pd_workspace_bytes_ex.restype = C.c_int64
        L.pd_simulate_ex.argtypes = [_p, C.POINTER(Events), C.c_uint64, C.c_int64, C.POINTER(Tracks), C.POINTER(Towers),
                                     C.POINTER(EFlow), C.POINTER(Debug), _p, C.c_int64, C.POINTER(Options), _p]
        L.pd_card_upload.argtypes = [_p]
        L.pd_pileup_workspace_bytes.argtypes = [C.c_int64]
        L.pd_pileup_workspace_bytes.restype = C.c_int64
        L.pd_pileup_merge.argtypes = [C.POINTER(Events), C.POINTER(Events), C.POINTER(PileupConfig), C.c_uint64, C.c_int64,
                                      C.POINTER(MergedEvents), _p, C.c_int64, _p]
        L.pd_filter_workspace_bytes.argtypes = [C.c_int64]
        L.pd_filter_workspace_bytes.restype = C.c_int64
        L.pd_filter_eflow.argtypes = [C.POINTER(EFlow), C.c_int64, C.POINTER(Condition), C.c_int32, C.c_int32, C.POINTER(EFlow), _p,
                                      C.c_int64, _p]
        L.pd_event_features.argtypes = [C.POINTER(EFlow), C.c_int64, C.c_float, C.c_float, C.POINTER(Features), _p]
        L.pd_truth_workspace_bytes.argtypes = [C.c_int64]
        L.pd_truth_workspace_bytes.restype = C.c_int64
        L.pd_truth_features.argtypes = [C.POINTER(Events), C.c_int32, C.POINTER(Features), _p, C.c_int64, _p]
        L.pd_truth_features_static.argtypes = [C.POINTER(Events), C.c_int32, C.POINTER(Features), _p]
        L.pd_truth_features_static.restype = C.c_int
        L.pd_track_impact.argtypes = [_p, C.POINTER(Events), C.POINTER(Tracks), C.POINTER(ImpactConfig), C.c_uint64, C.c_int64,
                                      C.POINTER(Impact), _p]
        L.pd_simulate_host.argtypes = [_p, C.POINTER(Events), C.c_uint64, C.c_int64, C.POINTER(Tracks),
                                       C.POINTER(Towers), C.POINTER(EFlow), _p]
        L.pd_strerror.argtypes = [C.c_int]
        L.pd_strerror.restype = C.c_char_p
        _lib = L
    return _lib


class PdError(RuntimeError):
    def __init__(self, code):
        super().__init__("pd: %s (code %d)" % (lib().pd_strerror(int(code)).decode(), int(code)))
        self.code = int(code)


def _check(rc):
    if rc != PD_OK:
        raise PdError(rc)


class Card:
    """pd_load_card / pd_card_info / pd_free_card."""

    def __init__(self, name_or_path: str):
        self._h = _p()
        _check(lib().pd_load_card(str(name_or_path).encode(), C.byref(self._h)))
        info = CardInfo()
        _check(lib().pd_card_info(self._h, C.byref(info)))
        self.n_towers, self.n_bins, self.grid_coord = info.n_towers, info.n_eta_bins, info.grid_coord
        self.bz, self.radius, self.half_length, self.n_eff_rows = info.bz, info.radius, info.half_length, info.n_eff_rows

    def __del__(self):
        if getattr(self, "_h", None):
            try:
                lib().pd_free_card(self._h)
            except Exception:
                pass
            self._h = None


def workspace_bytes(card: Card, n_events: int, n_particles: int, tile_events: int = 0, impact: bool = False) -> int:
    """pd_workspace_bytes_ex; tile_events: pd_options.tile_events (0 = automatic; a tuning knob); impact: with room for the
    impact parameters computed by the chain (pd_options.impact)."""
    opt = Options(int(tile_events))
    if impact:
        cfg, dummy = ImpactConfig(0.0, 0.0, 0.0, 0.0), Impact(*[C.c_void_p(16)] * 4)  # only their presence matters for the size
        opt.impact_config, opt.impact = C.pointer(cfg), C.pointer(dummy)
    n = lib().pd_workspace_bytes_ex(card._h, int(n_events), int(n_particles), C.byref(opt))
    if n < 0:
        raise PdError(n)
    return int(n)


def card_upload(card: Card):
    """pd_card_upload: the card's tables to the current device now, so that simulate() allocates nothing later."""
    _check(lib().pd_card_upload(card._h))


def last_launch_count() -> int:
    return int(lib().pd_last_launch_count())


def _torch():
    import torch

    return torch


def _tptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


class DeviceEvents:
    """Truth events resident in device memory (torch tensors), CSR."""

    def __init__(self, ev, device="cuda"):
        torch = _torch()
        self.n_events = int(ev.offsets.shape[0] - 1)
        self.n_particles = int(ev.offsets[-1])
        self.t = {}
        for name, dt in EVENT_FIELDS:
            a = np.ascontiguousarray(getattr(ev, name), dtype=dt)
            self.t[name] = torch.from_numpy(a).to(device)
        self.c = Events(self.n_events, self.n_particles, *[_tptr(self.t[k]) for k, _ in EVENT_FIELDS])

    def nbytes(self):
        return sum(t.numel() * t.element_size() for t in self.t.values())


class DeviceOutputs:
    """Output buffers (torch tensors) sized to the sufficient bounds of pd.h, plus the workspace."""

    def __init__(self, card: Card, n_events: int, n_particles: int, debug: bool = False, device="cuda", tile_events: int = 0, impact=None):
        """impact: None, or (d0_res, z0_res) = ((a, b), (a, b)): the chain itself writes d0, z0 and their errors of every track
        to self.impact (a DeviceImpact), pd_options.impact"""
        torch = _torch()
        self.tile_events = int(tile_events)  # pd_options.tile_events for the calls that use these buffers (sizes the workspace)
        self.impact_res = impact
        self.impact = None
        n = max(int(n_particles), 1)
        self.n_events, self.n_particles = int(n_events), int(n_particles)
        mk = lambda m, dt: torch.empty(m, dtype=getattr(torch, dt), device=device)  # noqa: E731
        self.trk = {"offsets": mk(n_events + 1, "int64"), **{k: mk(n, dt) for k, dt in TRACK_FIELDS}}
        self.tow = {"offsets": mk(n_events + 1, "int64"), **{k: mk(n, dt) for k, dt in TOWER_FIELDS}}
        self.efl = {"offsets": mk(n_events + 1, "int64"), **{k: mk(2 * n, dt) for k, dt in EFLOW_FIELDS}}
        # (zero-filled: the per-tower debug arrays are written only at the first depositing particle of each tower)
        self.dbg = {k: torch.zeros(n, dtype=getattr(torch, dt), device=device) for k, dt in DEBUG_FIELDS} if debug else None
        self.ws_bytes = workspace_bytes(card, n_events, n_particles, self.tile_events, impact is not None)
        if impact is not None:
            self.impact = DeviceImpact(n, device=device)
        self.ws = torch.empty(self.ws_bytes + 16, dtype=torch.uint8, device=device)
        self.c_trk = Tracks(n, _tptr(self.trk["offsets"]), *[_tptr(self.trk[k]) for k, _ in TRACK_FIELDS])
        self.c_tow = Towers(n, _tptr(self.tow["offsets"]), *[_tptr(self.tow[k]) for k, _ in TOWER_FIELDS])
        self.c_efl = EFlow(2 * n, _tptr(self.efl["offsets"]), *[_tptr(self.efl[k]) for k, _ in EFLOW_FIELDS])
        self.c_dbg = Debug(*[_tptr(self.dbg[k]) for k, _ in DEBUG_FIELDS]) if debug else None

    def to_numpy(self) -> dict:
        """Synchronise and return trimmed numpy arrays: trk_*, tow_*, efl_*, dbg_*."""
        torch = _torch()
        torch.cuda.synchronize()
        out = {}
        for prefix, d in (("trk", self.trk), ("tow", self.tow), ("efl", self.efl)):
            off = d["offsets"].cpu().numpy()
            tot = int(off[-1])
            out[prefix + "_offsets"] = off
            for k, t in d.items():
                if k != "offsets":
                    out["%s_%s" % (prefix, k)] = t[:tot].cpu().numpy()
        if self.dbg is not None:
            for k, t in self.dbg.items():
                out["dbg_" + k] = t[: self.n_particles].cpu().numpy()
        return out


class DeviceFeatures:
    """Buffers of pd_event_features for a DeviceOutputs' EFlow collection (per event: ht, met_x, met_y, met; per
    EFlow object: iso_charged, iso_neutral, iso_photon, r_iso)."""

    EVENT_FIELDS = ("ht", "met_x", "met_y", "met")
    OBJECT_FIELDS = ("iso_charged", "iso_neutral", "iso_photon", "r_iso")

    def __init__(self, n_events: int, capacity: int, device="cuda"):
        torch = _torch()
        self.n_events = int(n_events)
        self.ev = {k: torch.empty(max(self.n_events, 1), dtype=torch.float32, device=device) for k in self.EVENT_FIELDS}
        self.ob = {k: torch.empty(max(int(capacity), 1), dtype=torch.float32, device=device) for k in self.OBJECT_FIELDS}
        self.c = Features(*[_tptr(self.ev[k]) for k in self.EVENT_FIELDS], *[_tptr(self.ob[k]) for k in self.OBJECT_FIELDS])

    def to_numpy(self, n_objects: int) -> dict:
        _torch().cuda.synchronize()
        out = {k: t[: self.n_events].cpu().numpy() for k, t in self.ev.items()}
        out.update({k: t[: int(n_objects)].cpu().numpy() for k, t in self.ob.items()})
        return out


class DeviceObjects:
    """An EFlow-like collection uploaded from numpy (offsets, cls, pt, eta, phi): the input of pd_event_features
    when it does not come from a DeviceOutputs."""

    def __init__(self, offsets, cls, pt, eta, phi, device="cuda"):
        torch = _torch()
        import numpy as np

        self.n_events = int(len(offsets) - 1)
        self.n_objects = int(offsets[-1])
        pad = lambda a, dt: torch.from_numpy(np.ascontiguousarray(np.concatenate([np.asarray(a, dtype=dt), np.zeros(1, dtype=dt)]))).to(device)  # noqa: E731
        self.t = {"offsets": torch.from_numpy(np.ascontiguousarray(offsets, dtype=np.int64)).to(device), "cls": pad(cls, np.int8),
                  "pt": pad(pt, np.float32), "eta": pad(eta, np.float32), "phi": pad(phi, np.float32)}
        self.c_efl = EFlow(self.n_objects, _tptr(self.t["offsets"]), _tptr(self.t["cls"]), None, _tptr(self.t["pt"]),
                           _tptr(self.t["eta"]), _tptr(self.t["phi"]), None)


class DeviceEFlow:
    """An EFlow collection on the device with all its fields: the input (from numpy) or the output (empty, of a
    given capacity) of pd_filter_eflow; also accepted by event_features."""

    def __init__(self, n_events: int, capacity: int, arrays: dict | None = None, device="cuda"):
        torch = _torch()
        import numpy as np

        self.n_events, self.capacity = int(n_events), int(capacity)
        cap = max(self.capacity, 1)
        if arrays is None:
            self.t = {"offsets": torch.empty(self.n_events + 1, dtype=torch.int64, device=device)}
            self.t.update({k: torch.empty(cap, dtype=getattr(torch, dt), device=device) for k, dt in EFLOW_FIELDS})
        else:
            self.t = {"offsets": torch.from_numpy(np.ascontiguousarray(arrays["offsets"], dtype=np.int64)).to(device)}
            for k, dt in EFLOW_FIELDS:
                a = np.zeros(cap, dtype=dt)
                a[: len(arrays[k])] = arrays[k]
                self.t[k] = torch.from_numpy(a).to(device)
        self.c_efl = EFlow(self.capacity, _tptr(self.t["offsets"]), *[_tptr(self.t[k]) for k, _ in EFLOW_FIELDS])

    def to_numpy(self) -> dict:
        _torch().cuda.synchronize()
        off = self.t["offsets"].cpu().numpy()
        out = {"offsets": off}
        out.update({k: self.t[k][: int(off[-1])].cpu().numpy() for k, _ in EFLOW_FIELDS})
        return out


def make_conditions(conditions):
    """[{field, op, value, abs}] (the paper's Table C.13 grammar) -> ctypes array of pd_condition."""
    arr = (Condition * max(len(conditions), 1))()
    for k, c in enumerate(conditions):
        arr[k].field, arr[k].op, arr[k].use_abs = FIELDS[c["field"]], OPS[c["op"]], int(bool(c.get("abs", False)))
        if c["op"] in ("in", "not in"):
            vals = list(c["value"])
            arr[k].n_values = len(vals)
            for j, v in enumerate(vals[:8]):
                arr[k].values[j] = float(v)
        else:
            arr[k].n_values, arr[k].value = 0, float(c["value"])
    return arr


def filter_eflow(src, dst: "DeviceEFlow", conditions, combine: str = "all", stream=None, workspace=None):
    """pd_filter_eflow: `src` is a DeviceOutputs (its EFlow collection) or a DeviceEFlow; survivors go to `dst`.
    Asynchronous.  Returns the workspace tensor (to be kept alive until the stream is synchronised; pass it back as
    `workspace` to reuse it)."""
    torch = _torch()
    if not torch.cuda.is_available():
        raise PdError(PD_ECUDA)
    st = torch.cuda.current_stream() if stream is None else stream
    cap = int(src.c_efl.capacity)
    nbytes = int(lib().pd_filter_workspace_bytes(cap))
    ws = workspace if workspace is not None else torch.empty(nbytes + 16, dtype=torch.uint8, device="cuda")
    assert ws.numel() >= nbytes
    _check(lib().pd_filter_eflow(C.byref(src.c_efl), int(src.n_events), make_conditions(conditions), len(conditions),
                                 1 if combine == "any" else 0, C.byref(dst.c_efl), _tptr(ws), nbytes, C.c_void_p(st.cuda_stream)))
    return ws


def event_features(out, feat: DeviceFeatures, dr_max: float = 0.4, fsr_dr: float = 0.0, stream=None):
    """pd_event_features on the EFlow collection of `out` (torch's current stream or `stream`).  Asynchronous."""
    torch = _torch()
    if not torch.cuda.is_available():
        raise PdError(PD_ECUDA)
    st = torch.cuda.current_stream() if stream is None else stream
    _check(lib().pd_event_features(C.byref(out.c_efl), int(out.n_events), float(dr_max), float(fsr_dr), C.byref(feat.c),
                                   C.c_void_p(st.cuda_stream)))


def truth_features(dev_events: "DeviceEvents", feat: "DeviceFeatures", skip_neutrinos: bool = True, stream=None, workspace=None):
    """pd_truth_features: H_T and E_T^miss of the truth collection into feat's per-event arrays.  Asynchronous.
    Returns the workspace tensor (pass it back in to reuse it)."""
    torch = _torch()
    if not torch.cuda.is_available():
        raise PdError(PD_ECUDA)
    st = torch.cuda.current_stream() if stream is None else stream
    need = int(lib().pd_truth_workspace_bytes(int(dev_events.n_events)))
    if workspace is None or workspace.numel() * workspace.element_size() < need:
        workspace = torch.empty((need + 7) // 8, dtype=torch.int64, device="cuda")
    _check(lib().pd_truth_features(C.byref(dev_events.c), int(bool(skip_neutrinos)), C.byref(feat.c), _tptr(workspace),
                                   workspace.numel() * workspace.element_size(), C.c_void_p(st.cuda_stream)))
    return workspace


TRUTH_STATIC_MAX_EVENTS = 262144  # PD_TRUTH_STATIC_MAX_EVENTS of pd.h


def truth_features_static(dev_events: "DeviceEvents", feat: "DeviceFeatures", skip_neutrinos: bool = True, stream=None):
    """pd_truth_features_static: as truth_features, with the scratch in a fixed array inside the library (no workspace,
    no allocation; at most TRUTH_STATIC_MAX_EVENTS events; calls that overlap on the GPU race on it).  Asynchronous."""
    torch = _torch()
    if not torch.cuda.is_available():
        raise PdError(PD_ECUDA)
    st = torch.cuda.current_stream() if stream is None else stream
    _check(lib().pd_truth_features_static(C.byref(dev_events.c), int(bool(skip_neutrinos)), C.byref(feat.c), C.c_void_p(st.cuda_stream)))


class DeviceTrackRefs:
    """The two arrays of a track collection that pd_track_impact reads (offsets, src), uploaded from numpy: its input
    when the tracks do not come from a DeviceOutputs."""

    def __init__(self, offsets, src, device="cuda"):
        torch = _torch()
        self.n_events = int(len(offsets) - 1)
        self.n_tracks = int(offsets[-1])
        self.offsets = torch.from_numpy(np.ascontiguousarray(offsets, dtype=np.int64)).to(device)
        src = np.ascontiguousarray(src, dtype=np.int32)
        self.src = torch.from_numpy(src if src.size else np.zeros(1, dtype=np.int32)).to(device)
        self.c_trk = Tracks(max(self.n_tracks, 1), _tptr(self.offsets), _tptr(self.src), *([None] * (len(TRACK_FIELDS) - 1)))


class DeviceImpact:
    """Buffers of pd_track_impact: d0, z0, d0_err, z0_err per track (fp32, metres)."""

    FIELDS = ("d0", "z0", "d0_err", "z0_err")

    def __init__(self, capacity: int, device="cuda"):
        torch = _torch()
        self.t = {k: torch.empty(max(int(capacity), 1), dtype=torch.float32, device=device) for k in self.FIELDS}
        self.c = Impact(*[_tptr(self.t[k]) for k in self.FIELDS])

    def to_numpy(self, n_tracks: int) -> dict:
        _torch().cuda.synchronize()
        return {k: t[: int(n_tracks)].cpu().numpy() for k, t in self.t.items()}


def track_impact(card: Card, dev_events: DeviceEvents, tracks, out: DeviceImpact, d0_res=(0.0, 0.0), z0_res=(0.0, 0.0),
                 seed: int = 0, event_base: int = 0, stream=None):
    """pd_track_impact for the tracks of `tracks` (a DeviceOutputs after simulate, or a DeviceTrackRefs).  Asynchronous."""
    torch = _torch()
    if not torch.cuda.is_available():
        raise PdError(PD_ECUDA)
    st = torch.cuda.current_stream() if stream is None else stream
    cfg = ImpactConfig(float(d0_res[0]), float(d0_res[1]), float(z0_res[0]), float(z0_res[1]))
    _check(lib().pd_track_impact(card._h, C.byref(dev_events.c), C.byref(tracks.c_trk), C.byref(cfg), int(seed) & (2**64 - 1),
                                 int(event_base), C.byref(out.c), C.c_void_p(st.cuda_stream)))


def simulate(card: Card, dev_events: DeviceEvents, out: DeviceOutputs, seed: int, event_base: int = 0, stream=None):
    """pd_simulate_ex on torch's current stream (or `stream`), with the options `out` was made for.  Asynchronous."""
    torch = _torch()
    if not torch.cuda.is_available():
        raise PdError(PD_ECUDA)
    st = torch.cuda.current_stream() if stream is None else stream
    opt = Options(int(getattr(out, "tile_events", 0)))
    if getattr(out, "impact", None) is not None:
        (d0a, d0b), (z0a, z0b) = out.impact_res
        icfg = ImpactConfig(float(d0a), float(d0b), float(z0a), float(z0b))
        opt.impact_config, opt.impact = C.pointer(icfg), C.pointer(out.impact.c)
    rc = lib().pd_simulate_ex(card._h, C.byref(dev_events.c), int(seed) & (2**64 - 1), int(event_base), C.byref(out.c_trk),
                              C.byref(out.c_tow), C.byref(out.c_efl), C.byref(out.c_dbg) if out.c_dbg is not None else None,
                              _tptr(out.ws), out.ws_bytes, C.byref(opt), C.c_void_p(st.cuda_stream))
    _check(rc)


class DeviceMerged:
    """Output buffers of pd_pileup_merge: a pd_events-shaped batch (plus is_pu, n_pileup) of a given capacity."""

    def __init__(self, n_events: int, capacity: int, device="cuda"):
        torch = _torch()
        self.n_events, self.capacity = int(n_events), int(capacity)
        cap = max(self.capacity, 1)
        self.t = {"offsets": torch.empty(self.n_events + 1, dtype=torch.int64, device=device)}
        for name, dt in EVENT_FIELDS[1:]:
            self.t[name] = torch.empty(cap, dtype=getattr(torch, dt), device=device)
        self.t["is_pu"] = torch.empty(cap, dtype=torch.uint8, device=device)
        self.t["n_pileup"] = torch.empty(max(self.n_events, 1), dtype=torch.int32, device=device)
        self.t["vt"] = torch.empty(cap, dtype=torch.float32, device=device)
        nbytes = int(lib().pd_pileup_workspace_bytes(self.n_events))
        self.ws_bytes = nbytes
        self.ws = torch.empty(nbytes + 16, dtype=torch.uint8, device=device)
        self.c = MergedEvents(self.capacity, *[_tptr(self.t[k]) for k in ("offsets", "pid", "charge", "px", "py", "pz", "E", "vx", "vy",
                                                                            "vz", "is_pu", "n_pileup", "vt")])

    def total(self) -> int:
        _torch().cuda.synchronize()
        return int(self.t["offsets"][-1])

    def as_events(self):
        """The merged batch as the input of pd_simulate (synchronises to learn the particle count)."""
        ev = DeviceEvents.__new__(DeviceEvents)
        ev.n_events, ev.n_particles = self.n_events, self.total()
        ev.t = {k: self.t[k] for k, _ in EVENT_FIELDS}
        ev.c = Events(ev.n_events, ev.n_particles, *[_tptr(ev.t[k]) for k, _ in EVENT_FIELDS])
        return ev

    def to_numpy(self) -> dict:
        n = self.total()
        out = {"offsets": self.t["offsets"].cpu().numpy(), "n_pileup": self.t["n_pileup"][: self.n_events].cpu().numpy()}
        for k in [name for name, _ in EVENT_FIELDS[1:]] + ["is_pu", "vt"]:
            out[k] = self.t[k][:n].cpu().numpy()
        return out


def pileup_merge(hs: "DeviceEvents", pool: "DeviceEvents", out: DeviceMerged, mean_pileup: float, sigma_z: float = 0.053,
                 max_z_spread: float = 0.25, smear_hs_vertex: bool = True, seed: int = 0, event_base: int = 0, stream=None,
                 sigma_t: float = 160e-12, max_t_spread: float = 800e-12):
    """pd_pileup_merge (asynchronous).  pileup_status(out) afterwards reports PD_ECAPACITY if `out` was too small."""
    torch = _torch()
    if not torch.cuda.is_available():
        raise PdError(PD_ECUDA)
    st = torch.cuda.current_stream() if stream is None else stream
    cfg = PileupConfig(float(mean_pileup), float(sigma_z), float(max_z_spread), int(bool(smear_hs_vertex)), float(sigma_t), float(max_t_spread))
    _check(lib().pd_pileup_merge(C.byref(hs.c), C.byref(pool.c), C.byref(cfg), int(seed) & (2**64 - 1), int(event_base),
                                 C.byref(out.c), _tptr(out.ws), out.ws_bytes, C.c_void_p(st.cuda_stream)))


def pileup_status(out: DeviceMerged, stream=None) -> int:
    torch = _torch()
    st = torch.cuda.current_stream() if stream is None else stream
    return int(lib().pd_last_status(_tptr(out.ws), C.c_void_p(st.cuda_stream)))


def last_status(out: DeviceOutputs, stream=None) -> int:
    torch = _torch()
    st = torch.cuda.current_stream() if stream is None else stream
    return int(lib().pd_last_status(_tptr(out.ws), C.c_void_p(st.cuda_stream)))


class HostBuffers:
    """Pinned host buffers for pd_simulate_host (the end-to-end path).  packed=True (default) lays the 4-byte arrays of
    each collection out as the rows of one block; packed=False allocates every array on its own (the C ABI takes
    either: equal spacing is detected, not required)."""

    def __init__(self, ev, pin=True, packed=True):
        torch = _torch()
        self.n_events = int(ev.offsets.shape[0] - 1)
        self.n_particles = int(ev.offsets[-1])
        n = max(self.n_particles, 1)
        pin = bool(pin and torch.cuda.is_available())

        def host(a):
            t = torch.from_numpy(np.ascontiguousarray(a))
            return t.pin_memory() if pin else t

        def rows(fields, m):
            """The 4-byte arrays of a collection as the rows of ONE pinned block (equal spacing lets pd_simulate_host move
            a chunk of all of them with one strided copy); the others on their own."""
            four = [k for k, dt in fields if np.dtype(dt).itemsize == 4 and packed]
            block = torch.empty((len(four), m), dtype=torch.int32, pin_memory=pin)
            out = {}
            for k, dt in fields:
                if k in four:
                    out[k] = block[four.index(k)].view(getattr(torch, dt))
                else:
                    out[k] = torch.empty(m, dtype=getattr(torch, dt), pin_memory=pin)
            return out, block

        ev_fields = [(k, np.dtype(dt).name) for k, dt in EVENT_FIELDS if k != "offsets"]
        self.ev, self._ev_block = rows(ev_fields, n)
        for k, dt in ev_fields:
            self.ev[k][: self.n_particles].copy_(torch.from_numpy(np.ascontiguousarray(getattr(ev, k), dtype=dt)))
        self.ev = {"offsets": host(np.ascontiguousarray(ev.offsets, dtype=np.int64)), **self.ev}
        mk = lambda m, dt: torch.empty(m, dtype=getattr(torch, dt), pin_memory=pin)  # noqa: E731
        trk, self._trk_block = rows(TRACK_FIELDS, n)
        tow, self._tow_block = rows(TOWER_FIELDS, n)
        efl, self._efl_block = rows(EFLOW_FIELDS, 2 * n)
        self.trk = {"offsets": mk(self.n_events + 1, "int64"), **trk}
        self.tow = {"offsets": mk(self.n_events + 1, "int64"), **tow}
        self.efl = {"offsets": mk(self.n_events + 1, "int64"), **efl}
        self.c_ev = Events(self.n_events, self.n_particles, *[_tptr(self.ev[k]) for k, _ in EVENT_FIELDS])
        self.c_trk = Tracks(n, _tptr(self.trk["offsets"]), *[_tptr(self.trk[k]) for k, _ in TRACK_FIELDS])
        self.c_tow = Towers(n, _tptr(self.tow["offsets"]), *[_tptr(self.tow[k]) for k, _ in TOWER_FIELDS])
        self.c_efl = EFlow(2 * n, _tptr(self.efl["offsets"]), *[_tptr(self.efl[k]) for k, _ in EFLOW_FIELDS])

    def h2d_bytes(self):
        return sum(t.numel() * t.element_size() for t in self.ev.values())

    def d2h_bytes(self):
        b = 3 * 8 * (self.n_events + 1)
        for d, fields in ((self.trk, TRACK_FIELDS), (self.tow, TOWER_FIELDS), (self.efl, EFLOW_FIELDS)):
            tot = int(d["offsets"][-1])
            b += tot * sum(np.dtype(dt).itemsize for _, dt in fields)
        return b

    def to_numpy(self) -> dict:
        out = {}
        for prefix, d in (("trk", self.trk), ("tow", self.tow), ("efl", self.efl)):
            off = d["offsets"].numpy()
            tot = int(off[-1])
            out[prefix + "_offsets"] = off.copy()
            for k, t in d.items():
                if k != "offsets":
                    out["%s_%s" % (prefix, k)] = t[:tot].numpy().copy()
        return out


def simulate_host(card: Card, hb: HostBuffers, seed: int, event_base: int = 0, stream=None):
    """pd_simulate_host: host buffers in, host buffers out, copies inside the call.  Synchronous."""
    torch = _torch()
    if not torch.cuda.is_available():
        raise PdError(PD_ECUDA)
    st = torch.cuda.current_stream() if stream is None else stream
    _check(lib().pd_simulate_host(card._h, C.byref(hb.c_ev), int(seed) & (2**64 - 1), int(event_base), C.byref(hb.c_trk),
                                  C.byref(hb.c_tow), C.byref(hb.c_efl), C.c_void_p(st.cuda_stream)))
