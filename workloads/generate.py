"""Synthetic truth-event generators for the five BASELINE.json configs (no detector arithmetic here).

Every recipe: numpy `Generator(PCG64(seed))`, fp64 arithmetic, ONE rounding to fp32 at the end.
`generate(cfg, n_events=None)` returns an `Events` record with CSR offsets (int64), pid (int32),
charge (int8) and px, py, pz, E, vx, vy, vz (float32; GeV and metres).  `n_events=None` gives the full
size of the config; smaller values give a prefix-free *re-draw* of the same recipe (not a prefix of the
full sample), which is all the parity tests need: oracle and GPU always see the same arrays.
"""
from __future__ import annotations

import dataclasses
import hashlib

import numpy as np

# species table (SURVEY 8d "common conventions"): cumulative mix, pid magnitude, |charge|, mass [GeV]
_SPECIES_CUM = np.array([0.60, 0.85, 0.95, 0.975, 1.0])
_SPECIES_PID = np.array([211, 22, 130, 11, 13], dtype=np.int64)
_SPECIES_CHG = np.array([1, 0, 0, 1, 1], dtype=np.int64)
_SPECIES_MASS = np.array([0.13957039, 0.0, 0.497611, 0.00051099895, 0.1056584])

CONFIGS = {
    0: dict(card="cms_like", n_events=1_000, seed=1, name="cfg0 CMS-like 1k x Poisson(60)"),
    1: dict(card="cms_like", n_events=100_000, seed=2, name="cfg1 CMS-like ttbar-like 100k x Poisson(250)"),
    2: dict(card="cms_like", n_events=10_000, seed=3, name="cfg2 CMS-like PU200-like 10k x ~4060"),
    3: dict(card="atlas_like", n_events=1_000_000, seed=4, name="cfg3 ATLAS-like 1M x Poisson(40)"),
    4: dict(card="aleph_like", n_events=1_000_000, seed=5, name="cfg4 ALEPH-like Z->qq 1M x Poisson(30)"),
}


@dataclasses.dataclass
class Events:
    offsets: np.ndarray  # int64 [n_events + 1]
    pid: np.ndarray      # int32
    charge: np.ndarray   # int8
    px: np.ndarray       # float32 ...
    py: np.ndarray
    pz: np.ndarray
    E: np.ndarray
    vx: np.ndarray
    vy: np.ndarray
    vz: np.ndarray

    FLOAT_FIELDS = ("px", "py", "pz", "E", "vx", "vy", "vz")

    @property
    def n_events(self) -> int:
        return int(self.offsets.shape[0] - 1)

    @property
    def n_particles(self) -> int:
        return int(self.offsets[-1])

    def sha256(self) -> str:
        h = hashlib.sha256()
        for name in ("offsets", "pid", "charge") + self.FLOAT_FIELDS:
            h.update(np.ascontiguousarray(getattr(self, name)).tobytes())
        return h.hexdigest()


def config_card(cfg: int) -> str:
    return CONFIGS[cfg]["card"]


def _finish(offsets, pid, charge, pt, eta, phi, mass, vx, vy, vz) -> Events:
    """(pT, eta, phi, m) -> (px, py, pz, E) in fp64, then one rounding to fp32."""
    px = pt * np.cos(phi)
    py = pt * np.sin(phi)
    pz = pt * np.sinh(eta)
    E = np.sqrt(px * px + py * py + pz * pz + mass * mass)
    f = lambda a: np.ascontiguousarray(a, dtype=np.float32)  # noqa: E731
    return Events(
        offsets=np.ascontiguousarray(offsets, dtype=np.int64),
        pid=np.ascontiguousarray(pid, dtype=np.int32),
        charge=np.ascontiguousarray(charge, dtype=np.int8),
        px=f(px), py=f(py), pz=f(pz), E=f(E), vx=f(vx), vy=f(vy), vz=f(vz),
    )


def _species(rng, n):
    """pid, charge, mass for n particles: 60% pi+-, 25% gamma, 10% K0L, 2.5% e+-, 2.5% mu+-."""
    k = np.searchsorted(_SPECIES_CUM, rng.random(n), side="right").clip(0, 4)
    sign = np.where(rng.random(n) < 0.5, 1, -1)
    q = _SPECIES_CHG[k] * sign
    pid = _SPECIES_PID[k].copy()
    # pi+ = +211 (q=+1); e- = +11 (q=-1); mu- = +13 (q=-1); neutrals keep the positive code
    had = k == 0
    lep = k >= 3
    pid[had] = 211 * sign[had]
    pid[lep] = -_SPECIES_PID[k[lep]] * sign[lep]
    return pid, q, _SPECIES_MASS[k]


def _wrap_phi(phi):
    return (phi + np.pi) % (2.0 * np.pi) - np.pi


def _offsets(counts):
    off = np.zeros(counts.shape[0] + 1, dtype=np.int64)
    np.cumsum(counts, out=off[1:])
    return off


def _flat_kinematics(rng, n):
    """cfg0 kinematics: pT = 0.5 * 400^u, eta = -4 + 8u, phi = -pi + 2 pi u."""
    pt = 0.5 * np.power(400.0, rng.random(n))
    eta = -4.0 + 8.0 * rng.random(n)
    phi = -np.pi + 2.0 * np.pi * rng.random(n)
    return pt, eta, phi


def _gen_flat(card_cfg, n_events, seed, mean_mult):
    rng = np.random.Generator(np.random.PCG64(seed))
    counts = rng.poisson(mean_mult, n_events).astype(np.int64)
    off = _offsets(counts)
    n = int(off[-1])
    vz_ev = rng.normal(0.0, 0.05, n_events)
    pt, eta, phi = _flat_kinematics(rng, n)
    pid, q, m = _species(rng, n)
    vz = np.repeat(vz_ev, counts)
    z = np.zeros(n)
    return _finish(off, pid, q, pt, eta, phi, m, z, z, vz)


def _cone_constituents(rng, n_const_per_cone, eta_axis, phi_axis, e_cone, dr_sigma):
    """Constituents of cones: Dirichlet(0.3) shares of the cone energy taken as |p|,
    direction = axis + dR (cos psi, sin psi), dR = |N(0, dr_sigma)|.  Returns (|p|, eta, phi)."""
    n = int(n_const_per_cone.sum())
    g = rng.gamma(0.3, 1.0, n)
    starts = _offsets(n_const_per_cone)[:-1]
    nonempty = n_const_per_cone > 0
    sums = np.zeros(n_const_per_cone.shape[0])
    if n:
        red = np.add.reduceat(g, np.minimum(starts, n - 1))
        sums[nonempty] = red[nonempty]
    sums[~nonempty] = 1.0
    share = g / np.repeat(np.maximum(sums, 1e-300), n_const_per_cone)
    p = share * np.repeat(e_cone, n_const_per_cone)
    dr = np.abs(rng.normal(0.0, dr_sigma, n))
    psi = 2.0 * np.pi * rng.random(n)
    eta = np.repeat(eta_axis, n_const_per_cone) + dr * np.cos(psi)
    phi = _wrap_phi(np.repeat(phi_axis, n_const_per_cone) + dr * np.sin(psi))
    return p, eta, phi


def _gen_ttbar(n_events, seed):
    rng = np.random.Generator(np.random.PCG64(seed))
    counts = rng.poisson(250.0, n_events).astype(np.int64)
    vz_ev = rng.normal(0.0, 0.05, n_events)
    n_jets = rng.integers(4, 7, n_events)
    n_jet_part = rng.binomial(counts, 0.6)  # 60% of the event's particles are jet constituents
    n_soft = counts - n_jet_part
    # split the jet particles of each event over its jets with equal weights (multinomial)
    tot_jets = int(n_jets.sum())
    jet_event = np.repeat(np.arange(n_events), n_jets)
    jet_first = _offsets(n_jets)[:-1]
    which = rng.random(int(n_jet_part.sum()))
    part_event = np.repeat(np.arange(n_events), n_jet_part)
    jet_of_part = jet_first[part_event] + np.minimum((which * n_jets[part_event]).astype(np.int64), n_jets[part_event] - 1)
    n_const = np.bincount(jet_of_part, minlength=tot_jets).astype(np.int64)
    eta_axis = rng.uniform(-2.5, 2.5, tot_jets)
    phi_axis = rng.uniform(0.0, 2.0 * np.pi, tot_jets)
    e_jet = 30.0 * np.power(500.0 / 30.0, rng.random(tot_jets))
    p, eta_j, phi_j = _cone_constituents(rng, n_const, eta_axis, phi_axis, e_jet, 0.15)
    pt_j = np.maximum(p / np.cosh(eta_j), 0.1)
    ev_j = np.repeat(jet_event, n_const)
    ns = int(n_soft.sum())
    pt_s = np.maximum(rng.exponential(0.8, ns), 0.1)
    eta_s = rng.uniform(-4.0, 4.0, ns)
    phi_s = -np.pi + 2.0 * np.pi * rng.random(ns)
    ev_s = np.repeat(np.arange(n_events), n_soft)
    # event-major order: jet constituents (jet by jet), then the soft component
    ev = np.concatenate([ev_j, ev_s])
    order = np.argsort(ev, kind="stable")
    pt = np.concatenate([pt_j, pt_s])[order]
    eta = np.concatenate([eta_j, eta_s])[order]
    phi = np.concatenate([phi_j, phi_s])[order]
    off = _offsets(counts)
    n = int(off[-1])
    pid, q, m = _species(rng, n)
    vz = np.repeat(vz_ev, counts)
    z = np.zeros(n)
    return _finish(off, pid, q, pt, eta, phi, m, z, z, vz)


def _gen_pileup(n_events, seed):
    rng = np.random.Generator(np.random.PCG64(seed))
    n_soft = rng.poisson(4000.0, n_events).astype(np.int64)
    n_hard = 60
    counts = n_soft + n_hard
    off = _offsets(counts)
    n = int(off[-1])
    n_vtx = 200
    vz_tab = rng.normal(0.0, 0.05, (n_events, n_vtx))
    ns = int(n_soft.sum())
    pt_s = np.maximum(rng.exponential(0.6, ns), 0.1)
    eta_s = rng.uniform(-4.0, 4.0, ns)
    phi_s = -np.pi + 2.0 * np.pi * rng.random(ns)
    ev_s = np.repeat(np.arange(n_events), n_soft)
    vz_s = vz_tab[ev_s, rng.integers(0, n_vtx, ns)]
    # the hard dijet: two back-to-back cones of 200 GeV, 30 constituents each, at vertex 0
    eta_axis = rng.uniform(-2.5, 2.5, (n_events, 2))
    phi1 = rng.uniform(0.0, 2.0 * np.pi, n_events)
    phi_axis = np.stack([phi1, phi1 + np.pi], axis=1)
    n_const = np.full(2 * n_events, 30, dtype=np.int64)
    p, eta_h, phi_h = _cone_constituents(rng, n_const, eta_axis.ravel(), phi_axis.ravel(),
                                         np.full(2 * n_events, 200.0), 0.15)
    pt_h = np.maximum(p / np.cosh(eta_h), 0.1)
    ev_h = np.repeat(np.arange(n_events), n_hard)
    vz_h = vz_tab[ev_h, 0]
    # event-major order: soft component first, then the 60 dijet constituents
    ev = np.concatenate([ev_s, ev_h])
    order = np.argsort(ev, kind="stable")
    pt = np.concatenate([pt_s, pt_h])[order]
    eta = np.concatenate([eta_s, eta_h])[order]
    phi = np.concatenate([phi_s, phi_h])[order]
    vz = np.concatenate([vz_s, vz_h])[order]
    pid, q, m = _species(rng, n)
    z = np.zeros(n)
    return _finish(off, pid, q, pt, eta, phi, m, z, z, vz)


def _gen_zqq(n_events, seed):
    rng = np.random.Generator(np.random.PCG64(seed))
    counts = np.maximum(rng.poisson(30.0, n_events), 2).astype(np.int64)
    off = _offsets(counts)
    n = int(off[-1])
    # energies: 91.2 GeV x Dirichlet(1,...,1) taken as |p|
    g = rng.exponential(1.0, n)
    sums = np.add.reduceat(g, off[:-1])
    p = 91.2 * g / np.repeat(sums, counts)
    cos_t = rng.uniform(-0.95, 0.95, n_events)
    eta_ax = np.arctanh(cos_t)
    phi_ax = rng.uniform(0.0, 2.0 * np.pi, n_events)
    side = np.where(rng.random(n) < 0.5, 1.0, -1.0)
    dr = np.abs(rng.normal(0.0, 0.3, n))
    psi = 2.0 * np.pi * rng.random(n)
    eta = side * np.repeat(eta_ax, counts) + dr * np.cos(psi)
    phi = _wrap_phi(np.repeat(phi_ax, counts) + np.where(side > 0, 0.0, np.pi) + dr * np.sin(psi))
    pt = np.maximum(p / np.cosh(eta), 0.1)
    pid, q, m = _species(rng, n)
    z = np.zeros(n)
    return _finish(off, pid, q, pt, eta, phi, m, z, z, z)


def displaced(n_events: int, mean_mult: float, radius: float, half_length: float, seed: int, pt_lo: float = 0.15,
              pt_hi: float = 100.0, charged_frac: float = 0.75) -> Events:
    """Particles born anywhere inside a cylinder (r0 < 0.95 radius, |vz| < 0.95 half_length; uniform in volume), each with
    its own vertex: pT log-uniform in [pt_lo, pt_hi], eta ~ U(-3, 3), phi uniform; charges +-1 and +-2 (pions with twice
    the charge for |q| = 2), the rest photons and K0L.  For the chain's displaced-vertex branches."""
    rng = np.random.Generator(np.random.PCG64(seed))
    counts = rng.poisson(mean_mult, n_events).astype(np.int64)
    off = _offsets(counts)
    n = int(off[-1])
    r0 = 0.95 * radius * np.sqrt(rng.random(n))
    a = 2.0 * np.pi * rng.random(n)
    vx, vy = r0 * np.cos(a), r0 * np.sin(a)
    vz = 0.95 * half_length * (2.0 * rng.random(n) - 1.0)
    pt = pt_lo * np.power(pt_hi / pt_lo, rng.random(n))
    eta = -3.0 + 6.0 * rng.random(n)
    phi = -np.pi + 2.0 * np.pi * rng.random(n)
    u = rng.random(n)
    charged = u < charged_frac
    sign = np.where(rng.random(n) < 0.5, 1, -1)
    mag = np.where(rng.random(n) < 0.25, 2, 1)
    q = np.where(charged, sign * mag, 0)
    lepton = charged & (rng.random(n) < 0.1)
    pid = np.where(charged, 211 * sign, np.where(u < charged_frac + 0.15, 22, 130)).astype(np.int64)
    pid = np.where(lepton, np.where(rng.random(n) < 0.5, -11, -13) * sign, pid)
    m = np.where(pid == 22, 0.0, np.where(np.abs(pid) == 211, 0.13957039, np.where(pid == 130, 0.497611,
                 np.where(np.abs(pid) == 11, 0.00051099895, 0.1056584))))
    return _finish(off, pid, q, pt, eta, phi, m, vx, vy, vz)


def generate(cfg: int, n_events: int | None = None) -> Events:
    """Events of BASELINE.json configs[cfg]; `n_events` overrides the config's event count."""
    c = CONFIGS[cfg]
    ne = c["n_events"] if n_events is None else int(n_events)
    if cfg == 0:
        return _gen_flat(c["card"], ne, c["seed"], 60.0)
    if cfg == 1:
        return _gen_ttbar(ne, c["seed"])
    if cfg == 2:
        return _gen_pileup(ne, c["seed"])
    if cfg == 3:
        return _gen_flat(c["card"], ne, c["seed"], 40.0)
    if cfg == 4:
        return _gen_zqq(ne, c["seed"])
    raise KeyError(cfg)


def slice_events(ev: Events, e0: int, e1: int) -> Events:
    """Events [e0, e1) as a new CSR record (copies)."""
    i0, i1 = int(ev.offsets[e0]), int(ev.offsets[e1])
    kw = {k: np.ascontiguousarray(getattr(ev, k)[i0:i1]) for k in ("pid", "charge") + Events.FLOAT_FIELDS}
    return Events(offsets=np.ascontiguousarray(ev.offsets[e0:e1 + 1] - i0), **kw)


def concat_events(parts) -> Events:
    parts = list(parts)
    offs = [np.zeros(1, dtype=np.int64)]
    base = 0
    for p in parts:
        offs.append(p.offsets[1:] + base)
        base += p.n_particles
    kw = {k: np.concatenate([getattr(p, k) for p in parts]) for k in ("pid", "charge") + Events.FLOAT_FIELDS}
    return Events(offsets=np.concatenate(offs), **kw)


def from_lists(events) -> Events:
    """Build an Events record from python lists: events = [[(pid, q, px, py, pz, E, vx, vy, vz), ...], ...]."""
    counts = np.array([len(e) for e in events], dtype=np.int64)
    flat = [p for e in events for p in e]
    a = np.array(flat, dtype=np.float64).reshape(-1, 9)
    f = lambda k: np.ascontiguousarray(a[:, k], dtype=np.float32)  # noqa: E731
    return Events(offsets=_offsets(counts), pid=a[:, 0].astype(np.int32), charge=a[:, 1].astype(np.int8),
                  px=f(2), py=f(3), pz=f(4), E=f(5), vx=f(6), vy=f(7), vz=f(8))


def particle(pid, q, pt, eta, phi, mass=0.0, vx=0.0, vy=0.0, vz=0.0):
    """One particle tuple from (pT, eta, phi, m), fp64 (rounded to fp32 by from_lists)."""
    px, py, pz = pt * np.cos(phi), pt * np.sin(phi), pt * np.sinh(eta)
    return (pid, q, px, py, pz, float(np.sqrt(px * px + py * py + pz * pz + mass * mass)), vx, vy, vz)
