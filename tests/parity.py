"""Parity comparator: CUDA path (through the C ABI) versus the fp64 oracle, with the near-edge override
protocol of SURVEY.md 8c.6 / DESIGN.md "Comparison rule".

compare(card_name, ev, seed, gpu, event_base=0) -> report dict.  `gpu` is the dict of numpy arrays
returned by paper_2606_26089_b200.binding.DeviceOutputs.to_numpy() for a debug=True run on `ev`.

Rules (BASELINE.json north_star):
  * integers (status, accepted, tower id, class, src, counts, offsets, order): equal, except where the
    ORACLE flags the decision as near-edge (|x - edge| <= 1e-6 max(1,|edge|), D6: 1e-5 scale) and the
    GPU took the other allowed outcome; those are fed back to the oracle as overrides (it rejects an
    override it did not flag itself) and counted.
  * floats: |g - o| <= max(1e-5 |o|, 1e-6).  For the EFlow neutral energies N = E'' - T, a difference
    of two smeared quantities, the absolute term is 1e-5 max(|N|, E'', T).
"""
from __future__ import annotations

import numpy as np

from oracle import pdo

REL, ABS = 1e-5, 1e-6


def _close(g, o, scale=None):
    g = np.asarray(g, dtype=np.float64)
    o = np.asarray(o, dtype=np.float64)
    ref = np.abs(o) if scale is None else np.maximum(np.abs(o), scale)
    return np.abs(g - o) <= np.maximum(REL * ref, ABS)


def _phi_close(g, o):
    d = np.abs((np.asarray(g, dtype=np.float64) - o + np.pi) % (2 * np.pi) - np.pi)
    return d <= np.maximum(REL * np.abs(o), ABS)


def _event_of(offsets, idx):
    return np.searchsorted(offsets, idx, side="right") - 1


def _decisions_from_outputs(res, n_events, ev_idx, tw_id):
    """PD_DEC_* bits of each (event, tower) pair, derived from the Tower and EFlow collections."""
    big = np.int64(1) << 20
    key = ev_idx.astype(np.int64) * big + tw_id
    dec = np.zeros(key.shape[0], dtype=np.uint8)
    tow_ev = _event_of(res["tow_offsets"], np.arange(res["tow_tower"].shape[0]))
    tkey = tow_ev.astype(np.int64) * big + res["tow_tower"]
    pos = np.searchsorted(key, tkey)
    ok = (pos < key.shape[0])
    ok[ok] &= key[pos[ok]] == tkey[ok]
    if not ok.all():
        return None
    dec[pos[res["tow_Eem"] > 0]] |= 1
    dec[pos[res["tow_Ehad"] > 0]] |= 2
    efl_ev = _event_of(res["efl_offsets"], np.arange(res["efl_cls"].shape[0]))
    for cls, bit in ((4, 4), (3, 8)):
        sel = res["efl_cls"] == cls
        fkey = efl_ev[sel].astype(np.int64) * big + res["efl_src"][sel]
        p = np.searchsorted(key, fkey)
        ok = p < key.shape[0]
        ok[ok] &= key[p[ok]] == fkey[ok]
        if not ok.all():
            return None
        dec[p] |= bit
    return dec


def compare(card_name, ev, seed, gpu, event_base=0, max_rounds=6):
    card = pdo.Card(card_name)
    n = int(ev.offsets[-1])
    ne = int(ev.offsets.shape[0] - 1)
    rep = dict(n_particles=n, n_events=ne, flagged_particles=0, overridden_particles=0, flagged_towers=0,
               overridden_towers=0, unexcused=0, rounds=0, problems=[])
    ov_face = np.full(n, -1, dtype=np.int8)
    ov_tower = np.full(n, -2, dtype=np.int32)
    ov_row = np.full(n, -2, dtype=np.int8)
    tw_ov = {}  # (event, tower) -> [mask, value]
    g_status = gpu["dbg_status"]
    g_face = g_status & 3
    o = None
    for rnd in range(max_rounds):
        rep["rounds"] = rnd + 1
        ov = dict(face=ov_face, tower=ov_tower, eps_row=ov_row)
        if tw_ov:
            keys = sorted(tw_ov)
            ov.update(tw_event=np.array([k[0] for k in keys], dtype=np.int64), tw_id=np.array([k[1] for k in keys], dtype=np.int32),
                      tw_mask=np.array([tw_ov[k][0] for k in keys], dtype=np.uint8),
                      tw_value=np.array([tw_ov[k][1] for k in keys], dtype=np.uint8))
        try:
            o = pdo.simulate(card, ev, seed, event_base=event_base, overrides=ov, debug=True)
        except pdo.OracleError as exc:  # an override the oracle refuses = unexcused mismatch
            rep["problems"].append("oracle rejected overrides: %s" % exc)
            rep["unexcused"] += max(1, exc.n_rejected)
            return rep
        changed = False
        near = o["dbg_near"]
        # --- particle-level decisions
        o_face = o["dbg_status"] & 3
        d_stat = np.nonzero(g_status != o["dbg_status"])[0]
        for i in d_stat:
            if (near[i] & pdo.NEAR_FACE) and g_face[i] in (1, 2) and ov_face[i] == -1:
                # looper bit differs with same face: ENDCAP forces "does not reach", BARREL forces "reaches"
                want = g_face[i] if g_face[i] != o_face[i] else (2 if (g_status[i] & 4) else 1)
                ov_face[i] = want
                changed = True
            else:
                rep["unexcused"] += 1
                rep["problems"].append("status particle %d gpu %d oracle %d near %d" % (i, g_status[i], o["dbg_status"][i], near[i]))
        if not changed:
            d_row = np.nonzero(gpu["dbg_eps_row"] != o["dbg_eps_row"])[0]
            for i in d_row:
                if (near[i] & pdo.NEAR_EFF) and ov_row[i] == -2:
                    ov_row[i] = gpu["dbg_eps_row"][i]
                    changed = True
                else:
                    rep["unexcused"] += 1
                    rep["problems"].append("eps_row particle %d gpu %d oracle %d" % (i, gpu["dbg_eps_row"][i], o["dbg_eps_row"][i]))
            d_tow = np.nonzero(gpu["dbg_tower"] != o["dbg_tower"])[0]
            for i in d_tow:
                if (near[i] & (pdo.NEAR_ETA | pdo.NEAR_PHI)) and ov_tower[i] == -2:
                    ov_tower[i] = gpu["dbg_tower"][i]
                    changed = True
                else:
                    rep["unexcused"] += 1
                    rep["problems"].append("tower particle %d gpu %d oracle %d near %d eta %r phi %r" % (
                        i, gpu["dbg_tower"][i], o["dbg_tower"][i], near[i], o["dbg_eta_pos"][i], o["dbg_phi_pos"][i]))
        if rep["unexcused"]:
            return rep
        if changed:
            continue
        # --- accepted flags are never near-edge (D4)
        bad = np.nonzero(gpu["dbg_accepted"] != o["dbg_accepted"])[0]
        if bad.size:
            rep["unexcused"] += int(bad.size)
            rep["problems"].append("accepted differs at %s" % bad[:8])
            return rep
        # --- tower-level threshold decisions (D6)
        o_ev = _event_of(o["dtw_offsets"], np.arange(o["dtw_id"].shape[0]))
        first = np.nonzero(gpu["dbg_tw_first"] == 1)[0]
        g_ev = _event_of(ev.offsets, first)
        g_id = gpu["dbg_tower"][first]
        order = np.lexsort((g_id, g_ev))
        first, g_ev, g_id = first[order], g_ev[order], g_id[order]
        if g_ev.shape != o_ev.shape or not (np.array_equal(g_ev, o_ev) and np.array_equal(g_id, o["dtw_id"])):
            rep["unexcused"] += 1
            rep["problems"].append("deposited tower sets differ: gpu %d oracle %d" % (g_ev.shape[0], o_ev.shape[0]))
            return rep
        g_dec = gpu["dbg_tw_decisions"][first]
        o_dec = _decisions_from_outputs(o, ne, o_ev, o["dtw_id"])
        if o_dec is None:
            rep["unexcused"] += 1
            rep["problems"].append("oracle outputs reference towers that received no deposit")
            return rep
        diff = np.nonzero(g_dec != o_dec)[0]
        for t in diff:
            bits = int(g_dec[t] ^ o_dec[t])
            forcible = bits & int(o["dtw_near"][t])
            k = (int(o_ev[t]), int(o["dtw_id"][t]))
            cur = tw_ov.get(k, [0, 0])
            new = forcible & ~cur[0]
            if new == 0:
                rep["unexcused"] += 1
                rep["problems"].append("tower decision ev %d id %d gpu %d oracle %d near %d" % (k[0], k[1], g_dec[t], o_dec[t], o["dtw_near"][t]))
                continue
            cur[0] |= new
            cur[1] = (cur[1] & ~new) | (int(g_dec[t]) & new)
            tw_ov[k] = cur
            changed = True
        if rep["unexcused"]:
            return rep
        if not changed:
            break
    else:
        rep["unexcused"] += 1
        rep["problems"].append("override iteration did not converge")
        return rep

    near = o["dbg_near"]
    rep["flagged_particles"] = int(np.count_nonzero(near))
    rep["overridden_particles"] = int(np.count_nonzero((ov_face != -1) | (ov_tower != -2) | (ov_row != -2)))
    rep["flagged_towers"] = int(np.count_nonzero(o["dtw_near"]))
    rep["overridden_towers"] = len(tw_ov)

    def fail(msg):
        rep["unexcused"] += 1
        rep["problems"].append(msg)

    # --- integers: exact
    for name in ("trk_offsets", "tow_offsets", "efl_offsets", "trk_src", "trk_pid", "trk_charge", "tow_tower", "efl_cls", "efl_src"):
        if gpu[name].shape != o[name].shape or not np.array_equal(gpu[name], o[name]):
            fail("integer output %s differs" % name)
    if rep["unexcused"]:
        return rep
    # --- debug floats
    live = (o["dbg_status"] & 3) != 0
    errs = {}
    de = np.abs(gpu["dbg_eta_pos"][live].astype(np.float64) - o["dbg_eta_pos"][live])
    fin = np.isfinite(o["dbg_eta_pos"][live])
    dp = np.abs((gpu["dbg_phi_pos"][live].astype(np.float64) - o["dbg_phi_pos"][live] + np.pi) % (2 * np.pi) - np.pi)
    errs["max_abs_eta_pos"] = float(de[fin].max()) if fin.any() else 0.0
    errs["max_abs_phi_pos"] = float(dp.max()) if dp.size else 0.0
    band_e = 1e-6 * np.maximum(1.0, np.abs(o["dbg_eta_pos"][live][fin]))
    band_p = 1e-6 * np.maximum(1.0, np.abs(o["dbg_phi_pos"][live]))
    errs["eta_pos_outside_1e-6_band"] = int(np.count_nonzero(de[fin] > band_e))
    errs["phi_pos_outside_1e-6_band"] = int(np.count_nonzero(dp > band_p))
    rep["errors"] = errs
    if not _close(gpu["dbg_eta_pos"][live][fin], o["dbg_eta_pos"][live][fin]).all():
        fail("dbg_eta_pos beyond tolerance")
    if not _phi_close(gpu["dbg_phi_pos"][live], o["dbg_phi_pos"][live]).all():
        fail("dbg_phi_pos beyond tolerance")
    if not _close(gpu["dbg_pt_smeared"], o["dbg_pt_smeared"]).all():
        fail("dbg_pt_smeared beyond tolerance")
    # --- collections
    for name in ("trk_pt", "trk_eta", "trk_E", "trk_eta_out", "tow_eta", "tow_E", "tow_Eem", "tow_Ehad", "tow_ET", "efl_eta"):
        ok = _close(gpu[name], o[name])
        if not ok.all():
            i = int(np.nonzero(~ok)[0][0])
            fail("%s beyond tolerance at %d: gpu %r oracle %r (%d bad)" % (name, i, gpu[name][i], o[name][i], int((~ok).sum())))
    for name in ("trk_phi", "trk_phi_out", "tow_phi", "efl_phi"):
        ok = _phi_close(gpu[name], o[name])
        if not ok.all():
            i = int(np.nonzero(~ok)[0][0])
            fail("%s beyond tolerance at %d: gpu %r oracle %r" % (name, i, gpu[name][i], o[name][i]))
    # EFlow energies: tracks plain; neutrals with the operand-scaled absolute term
    cls = o["efl_cls"]
    scale = np.zeros(cls.shape[0])
    neutral = cls >= 3
    if neutral.any():
        big = np.int64(1) << 20
        o_ev = _event_of(o["dtw_offsets"], np.arange(o["dtw_id"].shape[0]))
        key = o_ev.astype(np.int64) * big + o["dtw_id"]
        efl_ev = _event_of(o["efl_offsets"], np.arange(cls.shape[0]))
        fk = efl_ev[neutral].astype(np.int64) * big + o["efl_src"][neutral]
        p = np.searchsorted(key, fk)
        is_ph = cls[neutral] == 4
        comp = np.where(is_ph, o["dtw_Eem_smeared"][p], o["dtw_Ehad_smeared"][p])
        trk = np.where(is_ph, o["dtw_Tem"][p], o["dtw_Thad"][p])
        scale[neutral] = np.maximum(comp, trk)
    okE = _close(gpu["efl_E"], o["efl_E"], scale)
    cosh = np.cosh(o["efl_eta"])
    okP = _close(gpu["efl_pt"], o["efl_pt"], scale / cosh)
    if not okE.all():
        i = int(np.nonzero(~okE)[0][0])
        fail("efl_E beyond tolerance at %d: gpu %r oracle %r scale %r" % (i, gpu["efl_E"][i], o["efl_E"][i], scale[i]))
    if not okP.all():
        fail("efl_pt beyond tolerance")
    # How many neutrals miss the PLAIN rule max(1e-5 |o|, 1e-6): reported by every test and bounded -- at most 1.5 % of
    # the neutrals (measured: 0-0.03 % on cfg1/2/4, 0.4 % on cfg0-like kinematics, ~1 % on the ATLAS-like card, whose
    # calorimeter resolution at high energy is comparable to the excess).  Closing the gap needs the smears of the tower
    # AND of its tracks in double: built and measured at +30 % of the chain's time on cfg2 with CUDA's double routines,
    # +5 % for the tower alone with short custom ones -- which left the count almost unchanged, because the fp32 track
    # energies dominate.
    n_out = int(np.count_nonzero(~_close(gpu["efl_E"], o["efl_E"])))
    n_neu = int(np.count_nonzero(neutral))
    errs["efl_neutral_E_outside_plain_tol"] = n_out
    errs["efl_neutrals"] = n_neu
    rep["neutral_outside_plain_tol"] = n_out
    rep["neutrals"] = n_neu
    if n_out > max(3, 0.015 * n_neu):
        fail("%d of %d neutrals outside the plain tolerance (bound: 1.5 %%)" % (n_out, n_neu))
    rel = np.abs(gpu["trk_pt"].astype(np.float64) - o["trk_pt"]) / np.maximum(np.abs(o["trk_pt"]), 1e-30)
    errs["max_rel_trk_pt"] = float(rel.max()) if rel.size else 0.0
    rel = np.abs(gpu["tow_E"].astype(np.float64) - o["tow_E"]) / np.maximum(np.abs(o["tow_E"]), 1e-30)
    errs["max_rel_tow_E"] = float(rel.max()) if rel.size else 0.0
    # invariant of north_star: every neutral has E > 0
    if neutral.any() and not (gpu["efl_E"][neutral] > 0).all():
        fail("neutral EFlow energy <= 0")
    return rep
