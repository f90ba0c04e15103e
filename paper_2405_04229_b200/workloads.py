"""Seeded synthetic workloads for the five BASELINE.json configs (cfg0..cfg4).

This module only *synthesises inputs*: fp32 segment arrays, atmosphere tables
(refractivity n-1 and vertical overburden X_v on a uniform height grid),
detector layouts and run parameters.  It holds none of the method's arithmetic
(no yield, no sampling, no tracing, no binning) and is the one module that both
the CPU oracle (``oracle/``) and the CUDA library binding consume, so that both
sides read identical fp32 bytes.

The recipes stand in for the thesis' CORSIKA showers ("1 TeV
vertical EM-Shower", "200 cascades of 500 GeV"), which are not
available; they take the shapes and value ranges of those workloads (Cherenkov
angle <= 1.4 deg PAPER.md:824; km-scale emission heights PAPER.md:450; metre
scale track segments PAPER.md:728).  The recipe is restated in DESIGN.md.

Everything is described with plain dicts / numpy arrays and symbolic strings;
each consumer maps them onto its own structs and flag values.
"""
from __future__ import annotations

import math
from typing import Optional

import numpy as np

# speed of light [m/ns]; used only to synthesise the segment clock t0
_C = 0.299792458

_SEG_FIELDS = ("x", "y", "z", "dx", "dy", "dz", "len", "beta", "t0", "charge", "edep")


# --------------------------------------------------------------------------
# atmosphere tables (inputs)
# --------------------------------------------------------------------------
def _five_layer_overburden(h: np.ndarray) -> np.ndarray:
    """Synthetic 5-layer vertical overburden X_v(h) [g/cm^2], h in metres.

    Four exponential layers X_v = a_i + b_i exp(-h/c_i) with boundaries
    0/4/10/40/100 km and scale heights 9.5/8.5/6.5/7.5 km, X_v(0) = 1030,
    rho(0) = 1.225e-3 g/cm^3, a_i and b_i from continuity of X_v and of the
    density; the fifth layer (h >= 100 km) falls linearly to zero with the
    density continuous at 100 km.  (A synthetic parameter set: the CORSIKA
    tables are not in the container.)
    """
    hb = np.array([0.0, 4e3, 10e3, 40e3, 100e3])
    c = np.array([9.5e3, 8.5e3, 6.5e3, 7.5e3])
    a = np.zeros(4)
    b = np.zeros(4)
    rho0 = 1.225e-3 * 100.0          # g/cm^3 -> g/cm^2 per metre
    b[0] = rho0 * c[0]
    a[0] = 1030.0 - b[0]
    for i in range(1, 4):
        rho_b = b[i - 1] / c[i - 1] * math.exp(-hb[i] / c[i - 1])
        b[i] = rho_b * c[i] * math.exp(hb[i] / c[i])
        x_b = a[i - 1] + b[i - 1] * math.exp(-hb[i] / c[i - 1])
        a[i] = x_b - b[i] * math.exp(-hb[i] / c[i])
    x100 = a[3] + b[3] * math.exp(-hb[4] / c[3])
    rho100 = b[3] / c[3] * math.exp(-hb[4] / c[3])
    if not (x100 > 0 and rho100 > 0):
        raise AssertionError("five-layer parameter set is not physical")
    out = np.empty_like(h, dtype=np.float64)
    for i in range(4):
        m = (h >= hb[i]) & (h <= hb[i + 1])
        out[m] = a[i] + b[i] * np.exp(-h[m] / c[i])
    m = h > hb[4]
    out[m] = np.maximum(0.0, x100 - rho100 * (h[m] - hb[4]))
    return out


def make_atmosphere(kind: str, h_obs: float = 0.0, rayleigh: bool = False,
                    aerosol: bool = False) -> dict:
    """kind: 'homogeneous' | 'planar_exp' | 'spherical_5layer'."""
    dh, n_nodes = 10.0, 10001
    h = np.arange(n_nodes, dtype=np.float64) * dh
    atm = dict(model=kind.split("_")[0], n_const_minus_1=np.float32(0.000293),
               h0=0.0, dh=dh, n_nodes=n_nodes, refractivity=None, overburden=None,
               earth_radius=6371000.0, h_obs=float(h_obs),
               rayleigh_X=0.0, rayleigh_lambda=400.0,
               aer_L=0.0, aer_H=1200.0, aer_lambda=350.0, aer_angstrom=1.0)
    if kind == "homogeneous":
        atm["refractivity"] = np.full(n_nodes, 0.000293, dtype=np.float32)
        atm["overburden"] = np.zeros(n_nodes, dtype=np.float32)
    else:
        atm["refractivity"] = (2.9e-4 * np.exp(-h / 8400.0)).astype(np.float32)
        if kind == "planar_exp":
            atm["overburden"] = (1030.0 * np.exp(-h / 8400.0)).astype(np.float32)
        elif kind == "spherical_5layer":
            atm["overburden"] = _five_layer_overburden(h).astype(np.float32)
        else:
            raise ValueError(kind)
    if rayleigh:
        atm["rayleigh_X"] = 2970.0       # g/cm^2 at 400 nm (parameter)
    if aerosol:
        atm["aer_L"] = 15000.0
    return atm


def _height_of_depth(atm: dict, xv: np.ndarray) -> np.ndarray:
    """Invert the (monotone) overburden table: height a.s.l. of vertical depth xv."""
    ob = atm["overburden"].astype(np.float64)
    h = atm["h0"] + atm["dh"] * np.arange(atm["n_nodes"])
    return np.interp(xv, ob[::-1], h[::-1])


# --------------------------------------------------------------------------
# shower-shaped segment sets (inputs)
# --------------------------------------------------------------------------
def _perp_basis(a: np.ndarray):
    t = np.array([1.0, 0.0, 0.0]) if abs(a[0]) < 0.9 else np.array([0.0, 1.0, 0.0])
    e1 = np.cross(a, t)
    e1 /= np.linalg.norm(e1)
    e2 = np.cross(a, e1)
    return e1, e2


def _tilt(axis: np.ndarray, polar: np.ndarray, azim: np.ndarray) -> np.ndarray:
    e1, e2 = _perp_basis(axis)
    sp, cp = np.sin(polar), np.cos(polar)
    d = (cp[:, None] * axis[None, :] + (sp * np.cos(azim))[:, None] * e1[None, :]
         + (sp * np.sin(azim))[:, None] * e2[None, :])
    return d / np.linalg.norm(d, axis=1, keepdims=True)


def _shower_segments(rng, n, atm, zenith_deg, azimuth_deg, xmax, lam_gh, r_moliere,
                     tilt_sigma_deg, len_lo, len_hi, lg_gamma_lo, lg_gamma_hi,
                     core=(0.0, 0.0)) -> dict:
    """Gaisser-Hillas depth (X0 = 0 => Gamma law), NKG-like lateral (beta-prime)."""
    zen, azi = math.radians(zenith_deg), math.radians(azimuth_deg)
    # unit vector along the direction of motion (downwards)
    axis = -np.array([math.sin(zen) * math.cos(azi), math.sin(zen) * math.sin(azi), math.cos(zen)])
    h_obs = atm["h_obs"]
    out = {k: np.empty(n, dtype=np.float32) for k in _SEG_FIELDS}
    filled = 0
    xv_ground = float(np.interp(h_obs, atm["h0"] + atm["dh"] * np.arange(atm["n_nodes"]),
                                atm["overburden"].astype(np.float64)))
    e1, e2 = _perp_basis(axis)
    while filled < n:
        m = int((n - filled) * 1.3) + 64
        X = rng.gamma(xmax / lam_gh + 1.0, lam_gh, m)          # slant depth [g/cm^2]
        xv = X * math.cos(zen)
        age = 3.0 * X / (X + 2.0 * xmax)
        age = np.clip(age, 0.2, 1.9)
        B = rng.beta(age, 4.5 - 2.0 * age)
        r = r_moliere * B / (1.0 - B)
        psi = rng.uniform(0.0, 2.0 * math.pi, m)
        L = rng.uniform(len_lo, len_hi, m)
        polar = np.abs(rng.normal(0.0, 1.0, m)) * math.radians(tilt_sigma_deg)
        az = rng.uniform(0.0, 2.0 * math.pi, m)
        lg = rng.uniform(lg_gamma_lo, lg_gamma_hi, m)
        q = rng.integers(0, 2, m) * 2 - 1
        h = _height_of_depth(atm, xv)
        ell = (h - h_obs) / math.cos(zen)                      # distance from the core along the axis
        pos = (-ell)[:, None] * axis[None, :] \
            + (r * np.cos(psi))[:, None] * e1[None, :] + (r * np.sin(psi))[:, None] * e2[None, :]
        pos[:, 0] += core[0]
        pos[:, 1] += core[1]
        d = _tilt(axis, polar, az)
        z_end = pos[:, 2] + L * d[:, 2]
        ok = (xv < xv_ground) & (pos[:, 2] > 1.0) & (z_end > 1.0) & (h < 99000.0) & np.isfinite(r) & (r < 5000.0)
        idx = np.nonzero(ok)[0][: n - filled]
        k = len(idx)
        sl = slice(filled, filled + k)
        out["x"][sl], out["y"][sl], out["z"][sl] = pos[idx, 0], pos[idx, 1], pos[idx, 2]
        out["dx"][sl], out["dy"][sl], out["dz"][sl] = d[idx, 0], d[idx, 1], d[idx, 2]
        out["len"][sl] = L[idx]
        gam = 10.0 ** lg[idx]
        out["beta"][sl] = np.sqrt(1.0 - 1.0 / (gam * gam))      # fp64, then rounded to fp32
        out["t0"][sl] = (120000.0 / math.cos(zen) - ell[idx]) / _C
        out["charge"][sl] = q[idx]
        out["edep"][sl] = 0.0
        filled += k
    return out


def _cfg0_segments(rng, n) -> dict:
    out = {k: np.empty(n, dtype=np.float32) for k in _SEG_FIELDS}
    out["x"][:] = rng.uniform(-50.0, 50.0, n)
    out["y"][:] = rng.uniform(-50.0, 50.0, n)
    z = rng.uniform(5000.0, 15000.0, n)
    out["z"][:] = z
    polar = np.abs(rng.normal(0.0, math.radians(3.0), n))
    az = rng.uniform(0.0, 2.0 * math.pi, n)
    d = _tilt(np.array([0.0, 0.0, -1.0]), polar, az)
    out["dx"][:], out["dy"][:], out["dz"][:] = d[:, 0], d[:, 1], d[:, 2]
    out["len"][:] = 10.0
    out["beta"][:] = rng.uniform(0.9999, 1.0, n)
    out["t0"][:] = z / _C
    out["charge"][:] = rng.integers(0, 2, n) * 2 - 1
    out["edep"][:] = 0.0
    return out


# --------------------------------------------------------------------------
# detectors (inputs)
# --------------------------------------------------------------------------
def _no_detector() -> dict:
    return dict(hist_nx=0, hist_ny=0, hist_x0=0.0, hist_y0=0.0, hist_cell=1.0,
                tel_xyzr=np.zeros((0, 4), dtype=np.float32),
                cam_enabled=False, cam_az_deg=0.0, cam_el_deg=0.0, cam_pix_deg=1.5,
                cam_rows=0, cam_cols=0, n_tbins=0, t_ref_ns=0.0, t_bin_ns=100.0)


def _grid(det: dict, n: int, cell: float) -> dict:
    det.update(hist_nx=n, hist_ny=n, hist_x0=-0.5 * n * cell, hist_y0=-0.5 * n * cell, hist_cell=cell)
    return det


def _square_lattice(nside: int, pitch: float, r: float) -> np.ndarray:
    c = (np.arange(nside) - 0.5 * (nside - 1)) * pitch
    xx, yy = np.meshgrid(c, c, indexing="xy")
    t = np.zeros((nside * nside, 4), dtype=np.float32)
    t[:, 0], t[:, 1], t[:, 3] = xx.ravel(), yy.ravel(), r
    return t


def _hex_lattice(nrow: int, ncol: int, pitch: float, r: float) -> np.ndarray:
    row_pitch = pitch * math.sqrt(3.0) / 2.0
    t = np.zeros((nrow * ncol, 4), dtype=np.float32)
    k = 0
    for ir in range(nrow):
        y = (ir - 0.5 * (nrow - 1)) * row_pitch
        shift = 0.5 * pitch if (ir % 2) else 0.0
        for ic in range(ncol):
            t[k, 0] = (ic - 0.5 * (ncol - 1)) * pitch + shift - 0.25 * pitch
            t[k, 1] = y
            t[k, 3] = r
            k += 1
    return t


def _default_params() -> dict:
    return dict(emit="cherenkov", trace="straight", trans="off",
                lv1=False, lv2=False, write="all",
                lambda_min_nm=300.0, lambda_max_nm=600.0, bunch_weight=1.0,
                lv1_margin_rad=0.0, lv2_margin_m=0.0, substeps=1,
                fluor_yield_per_MeV=4.0, line_nm=np.zeros(0, np.float32),
                line_cdf=np.zeros(0, np.float32), aim_factor=1.5,
                disp_b_nm2=0.0, disp_lambda0_nm=400.0)      # dispersion off (R13)


_TABLE = dict(n_h=512, n_zen=256, h_max=100000.0, zen_max_deg=89.0)

FULL_SEGMENTS = (1000, 100000, 1000000, 1000000, 10000000)


def make_config(k: int, n_segments: Optional[int] = None, rng_seed: Optional[int] = None) -> dict:
    """Build config k (0..4) of BASELINE.json; ``n_segments`` scales it down for tests.

    Returns dict(name, segments, atmosphere, detector, params, table, seed, seg_id_base).
    The numpy generator is ``default_rng(1000 + k)``; the kernel seed is 1.
    """
    n = FULL_SEGMENTS[k] if n_segments is None else int(n_segments)
    rng = np.random.default_rng(1000 + k if rng_seed is None else rng_seed)
    par = _default_params()
    det = _no_detector()
    table = None
    if k == 0:
        atm = make_atmosphere("homogeneous")
        seg = _cfg0_segments(rng, n)
        _grid(det, 200, 5.0)
    elif k == 1:
        atm = make_atmosphere("planar_exp", h_obs=2000.0, rayleigh=True)
        seg = _shower_segments(rng, n, atm, 0.0, 0.0, 330.0, 70.0, 80.0, 4.0, 5.0, 5.0, 2.0, 5.0)
        _grid(det, 400, 2.5)
        par.update(trace="numeric", trans="weight", write="all")
    elif k == 2:
        atm = make_atmosphere("spherical_5layer", h_obs=0.0, rayleigh=True)
        seg = _shower_segments(rng, n, atm, 60.0, 30.0, 650.0, 70.0, 80.0, 4.0, 10.0, 80.0, 1.5, 5.0)
        det["tel_xyzr"] = _square_lattice(10, 100.0, 6.0)
        table = dict(_TABLE)
        par.update(trace="table", trans="roulette", lv1=True, lv2=True, write="tel",
                   lambda_min_nm=250.0, lambda_max_nm=700.0, bunch_weight=5.0,
                   lv1_margin_rad=math.radians(1.0), lv2_margin_m=25.0)
    elif k == 3:
        atm = make_atmosphere("spherical_5layer", h_obs=0.0, rayleigh=True, aerosol=True)
        seg = _shower_segments(rng, n, atm, 30.0, 90.0, 750.0, 70.0, 80.0, 4.0, 10.0, 10.0, 2.0, 5.0)
        seg["edep"][:] = np.float32(0.9e13 / 1.0e6)             # MeV per segment at full size
        det["tel_xyzr"] = np.array([[20000.0, 0.0, 0.0, 1.9]], dtype=np.float32)
        det.update(cam_enabled=True, cam_az_deg=180.0, cam_el_deg=15.5, cam_pix_deg=1.5,
                   cam_rows=22, cam_cols=20, n_tbins=1000, t_bin_ns=100.0)
        lines = np.sort(rng.uniform(300.0, 430.0, 21)).astype(np.float32)
        inten = rng.uniform(0.0, 1.0, 21)
        cdf = np.cumsum(inten / inten.sum())
        cdf[-1] = 1.0
        table = dict(_TABLE)
        par.update(emit="fluorescence", trace="table", trans="roulette", write="tel",
                   line_nm=lines, line_cdf=cdf.astype(np.float32), lv2=True, lv2_margin_m=25.0)
        # time window (1000 x 100 ns): opens 2 us before the light of the earliest 5 % of the segments
        # can reach the aperture (segment clock + straight distance / c), so the bulk of the shower
        # falls inside it at any segment count
        tel0 = det["tel_xyzr"][0].astype(np.float64)
        dist = np.sqrt((seg["x"] - tel0[0]) ** 2 + (seg["y"] - tel0[1]) ** 2 + (seg["z"] - tel0[2]) ** 2)
        first = np.percentile(seg["t0"].astype(np.float64) + dist / _C, 5.0)
        det["t_ref_ns"] = float(np.floor((first - 2000.0) / 100.0) * 100.0)
    elif k == 4:
        atm = make_atmosphere("spherical_5layer", h_obs=0.0, rayleigh=True)
        seg = _shower_segments(rng, n, atm, 20.0, 0.0, 580.0, 70.0, 80.0, 4.0, 1.0, 20.0, 1.0, 6.0)
        det["tel_xyzr"] = _hex_lattice(100, 100, 50.0, 6.0)
        _grid(det, 1000, 1.0)
        table = dict(_TABLE)
        par.update(trace="table", trans="roulette", lv1=True, lv2=True, write="tel",
                   lambda_min_nm=250.0, lambda_max_nm=700.0, bunch_weight=1.0,
                   lv1_margin_rad=math.radians(1.0), lv2_margin_m=25.0)
    else:
        raise ValueError("config index must be 0..4")
    return dict(name=f"cfg{k}", index=k, segments=seg, atmosphere=atm, detector=det,
                params=par, table=table, seed=1, seg_id_base=0)


def slice_segments(seg: dict, lo: int, hi: int) -> dict:
    return {k: np.ascontiguousarray(v[lo:hi]) for k, v in seg.items()}
