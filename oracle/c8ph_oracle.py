"""ctypes front-end of the CPU oracle (``oracle/c8ph_oracle.c``).

TEST INFRASTRUCTURE ONLY: imported by tests/, ``__graft_entry__.smoke()`` and
``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs.  The product
package never imports this module.  It marshals the plain-dict workloads of
``paper_2405_04229_b200.workloads`` into the oracle's own C structs; all
arithmetic of the method lives in the C file.
"""
from __future__ import annotations

import ctypes as C
import math
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "c8ph_oracle.c")
# C8PH_ORACLE_SANITIZE=1 (set before the first call): the oracle is compiled with -fsanitize=address,undefined into its
# own file and loaded from there (the process needs libasan preloaded); used once by tests/test_oracle_pins.py.
_SAN = os.environ.get("C8PH_ORACLE_SANITIZE") == "1"
_LIB = os.path.join(_HERE, "libc8ph_oracle_san.so" if _SAN else "libc8ph_oracle.so")
_lock = threading.Lock()
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle (plain C, -O2, no fast-math, OpenMP over segments)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        san = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=all", "-fno-omit-frame-pointer"] if _SAN else ["-O2"]
        subprocess.check_call(["gcc", *san, "-std=c11", "-fPIC", "-shared", "-fopenmp",
                               "-fno-fast-math", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class Atmosphere(C.Structure):
    _fields_ = [("model", C.c_int32), ("n_nodes", C.c_int32), ("n_const_minus_1", C.c_double),
                ("h0", C.c_double), ("dh", C.c_double),
                ("refractivity", C.POINTER(C.c_float)), ("overburden", C.POINTER(C.c_float)),
                ("earth_radius", C.c_double), ("h_obs", C.c_double),
                ("rayleigh_X", C.c_double), ("rayleigh_lambda", C.c_double),
                ("aer_L", C.c_double), ("aer_H", C.c_double), ("aer_lambda", C.c_double),
                ("aer_angstrom", C.c_double),
                ("n_ext_lambda", C.c_int32), ("pad4", C.c_int32), ("ext_lambda0", C.c_double), ("ext_dlambda", C.c_double),
                ("ext_tau_v", C.POINTER(C.c_float))]


class Table(C.Structure):
    _fields_ = [("n_h", C.c_int32), ("n_zen", C.c_int32), ("n_ch", C.c_int32), ("pad", C.c_int32),
                ("h_max", C.c_double), ("zen_max_rad", C.c_double), ("data", C.POINTER(C.c_float)),
                ("n_rho", C.c_int32), ("pad3", C.c_int32), ("rho_max", C.c_double), ("data3", C.POINTER(C.c_float))]


class Segments(C.Structure):
    _fields_ = [(k, C.POINTER(C.c_float)) for k in
                ("x", "y", "z", "dx", "dy", "dz", "len", "beta", "t0", "charge", "edep")] + [("id", C.POINTER(C.c_uint64))]


class Detector(C.Structure):
    _fields_ = [("hist_nx", C.c_int32), ("hist_ny", C.c_int32),
                ("hist_x0", C.c_double), ("hist_y0", C.c_double), ("hist_cell", C.c_double),
                ("n_tel", C.c_int32), ("cam_enabled", C.c_int32), ("tel_xyzr", C.POINTER(C.c_float)),
                ("cam_az_deg", C.c_double), ("cam_el_deg", C.c_double), ("cam_pix_deg", C.c_double),
                ("cam_rows", C.c_int32), ("cam_cols", C.c_int32), ("n_tbins", C.c_int32), ("pad", C.c_int32),
                ("t_ref_ns", C.c_double), ("t_bin_ns", C.c_double),
                ("opt_enabled", C.c_int32), ("pad3", C.c_int32),
                ("opt_az_deg", C.c_double), ("opt_el_deg", C.c_double),
                ("opt_focal_m", C.c_double), ("opt_mirror_radius_m", C.c_double), ("opt_camera_radius_m", C.c_double),
                ("opt_kind", C.c_int32), ("opt_n_abs", C.c_int32),
                ("opt_lens_roc_m", C.c_double), ("opt_lens_thickness_m", C.c_double), ("opt_lens_index", C.c_double),
                ("opt_abs", (C.c_double * 7) * 8)]


class Params(C.Structure):
    _fields_ = [("emit", C.c_int32), ("trace", C.c_int32), ("trans", C.c_int32),
                ("lv1", C.c_int32), ("lv2", C.c_int32), ("substeps", C.c_int32),
                ("lambda_min_nm", C.c_double), ("lambda_max_nm", C.c_double), ("bunch_weight", C.c_double),
                ("lv1_margin_rad", C.c_double), ("lv2_margin_m", C.c_double),
                ("fluor_yield_per_MeV", C.c_double), ("aim_factor", C.c_double),
                ("n_lines", C.c_int32), ("pad", C.c_int32),
                ("line_nm", C.POINTER(C.c_float)), ("line_cdf", C.POINTER(C.c_float)),
                ("disp_b_nm2", C.c_double), ("disp_lambda0_nm", C.c_double),
                ("n_eff", C.c_int32), ("flat_plane", C.c_int32),
                ("eff_lambda0_nm", C.c_double), ("eff_dlambda_nm", C.c_double), ("eff", C.POINTER(C.c_float))]


PHOTON_DTYPE = np.dtype([("seg", "<i8"), ("j", "<i4"), ("status", "<i4"),
                         ("x", "<f8"), ("y", "<f8"), ("ux", "<f8"), ("uy", "<f8"), ("uz", "<f8"),
                         ("t", "<f8"), ("lambda_nm", "<f8"), ("T", "<f8"), ("weight", "<f8"),
                         ("x_line", "<f8"), ("y_line", "<f8"),
                         ("bin", "<i4"), ("tel", "<i4"), ("pix", "<i4"), ("tbin", "<i4")], align=True)

COUNTER_NAMES = ("segments", "seg_below_threshold", "seg_lv1", "seg_emitting", "emitted", "upgoing",
                 "lv2", "table_range", "roulette", "landed", "in_grid", "tel_hit", "cam_hit", "nonfinite")
ST_LANDED, ST_UPGOING, ST_LV2, ST_TABLE_RANGE, ST_ROULETTE = range(5)

_MODEL = {"homogeneous": 0, "planar": 1, "spherical": 2, "cylindrical": 3}
_EMIT = {"cherenkov": 0, "fluorescence": 1}
_TRACE = {"straight": 0, "numeric": 1, "table": 2}
_TRANS = {"off": 0, "weight": 1, "roulette": 2}


def _fp(a):
    return a.ctypes.data_as(C.POINTER(C.c_float))


def lib():
    global _lib
    with _lock:
        if _lib is None:
            build()
            L = C.CDLL(_LIB)
            L.orc_uniform.restype = C.c_double
            L.orc_uniform.argtypes = [C.c_uint32]
            L.orc_refractivity.restype = C.c_double
            L.orc_refractivity.argtypes = [C.POINTER(Atmosphere), C.c_double]
            L.orc_overburden.restype = C.c_double
            L.orc_overburden.argtypes = [C.POINTER(Atmosphere), C.c_double]
            L.orc_height.restype = C.c_double
            L.orc_cherenkov_yield.restype = C.c_double
            L.orc_cherenkov_yield.argtypes = [C.c_double] * 6
            L.orc_cherenkov_yield_dispersive.restype = C.c_double
            L.orc_cherenkov_yield_dispersive.argtypes = [C.c_double] * 8
            L.orc_dispersion_factor.restype = C.c_double
            L.orc_dispersion_factor.argtypes = [C.c_double] * 3
            L.orc_substep_track.restype = C.c_int32
            L.orc_substep_track.argtypes = [C.POINTER(C.c_double), C.POINTER(C.c_double)] + [C.c_double] * 5 + \
                                           [C.POINTER(C.c_double), C.c_double, C.c_int32, C.POINTER(C.c_float)]
            L.orc_highland_theta0.restype = C.c_double
            L.orc_highland_theta0.argtypes = [C.c_double] * 4
            L.orc_substep_track_ms.restype = C.c_int32
            L.orc_substep_track_ms.argtypes = [C.POINTER(Atmosphere), C.POINTER(C.c_double), C.POINTER(C.c_double)] + [C.c_double] * 5 + \
                                              [C.POINTER(C.c_double), C.c_double, C.c_double, C.c_double, C.c_uint64, C.c_uint64,
                                               C.c_int32, C.POINTER(C.c_float)]
            L.orc_last_mile.restype = C.c_int
            L.orc_last_mile.argtypes = [C.POINTER(Detector)] + [C.POINTER(C.c_double)] * 3 + [C.c_double, C.POINTER(C.c_double)]
            L.orc_refract.restype = C.c_int
            L.orc_refract.argtypes = [C.POINTER(C.c_double)] * 2 + [C.c_double, C.c_double, C.POINTER(C.c_double)]
            L.orc_segment_distance.restype = C.c_double
            L.orc_segment_distance.argtypes = [C.POINTER(C.c_double)] * 4
            L.orc_ext_tau_vertical.restype = C.c_double
            L.orc_ext_tau_vertical.argtypes = [C.POINTER(Atmosphere), C.c_double, C.c_double]
            L.orc_transmission_tabulated.restype = C.c_double
            L.orc_transmission_tabulated.argtypes = [C.POINTER(Atmosphere), C.c_double, C.c_double, C.c_double]
            L.orc_efficiency.restype = C.c_double
            L.orc_efficiency.argtypes = [C.POINTER(Params), C.c_double]
            L.orc_straight_line.restype = C.c_double
            L.orc_trace.restype = C.c_int
            L.orc_trace.argtypes = [C.POINTER(Atmosphere), C.c_int, C.c_double, C.c_double, C.c_double,
                                    C.c_double, C.c_int, C.POINTER(C.c_double)]
            L.orc_build_table.restype = None
            L.orc_build_table.argtypes = [C.POINTER(Atmosphere), C.c_int, C.c_int, C.c_double, C.c_double,
                                          C.c_int, C.POINTER(C.c_float)]
            L.orc_build_table_flat.restype = None
            L.orc_build_table_flat.argtypes = [C.POINTER(Atmosphere), C.c_int, C.c_int, C.c_int, C.c_double, C.c_double,
                                               C.c_double, C.c_int, C.POINTER(C.c_float)]
            L.orc_table_flat_lookup.restype = C.c_int
            L.orc_table_flat_lookup.argtypes = [C.POINTER(Table), C.c_double, C.c_double, C.c_double, C.c_double, C.POINTER(C.c_double),
                                                C.POINTER(C.c_double)]
            L.orc_trace_cyl.restype = C.c_int
            L.orc_trace_cyl.argtypes = [C.POINTER(Atmosphere)] + [C.c_double] * 5 + [C.c_int, C.POINTER(C.c_double)]
            L.orc_cyl_correction.restype = C.c_int
            L.orc_cyl_correction.argtypes = [C.POINTER(Atmosphere)] + [C.c_double] * 4 + [C.c_int, C.POINTER(C.c_double)]
            L.orc_build_table_cyl.restype = None
            L.orc_build_table_cyl.argtypes = [C.POINTER(Atmosphere), C.c_int, C.c_int, C.c_int, C.c_double, C.c_double,
                                              C.c_int, C.POINTER(C.c_float)]
            L.orc_table_cyl_lookup.restype = C.c_int
            L.orc_table_cyl_lookup.argtypes = [C.POINTER(Table), C.c_double, C.c_double, C.c_double, C.POINTER(C.c_double)]
            L.orc_table_lookup.restype = C.c_int
            L.orc_table_lookup.argtypes = [C.POINTER(Table), C.c_double, C.c_double, C.POINTER(C.c_double)]
            L.orc_transmission.restype = C.c_double
            L.orc_transmission.argtypes = [C.POINTER(Atmosphere), C.c_double, C.c_double, C.c_double]
            L.orc_ray_sphere.restype = C.c_int
            L.orc_camera_pixel.restype = C.c_int
            L.orc_count.restype = C.c_int64
            L.orc_run.restype = C.c_int
            assert L.orc_sizeof_photon() == PHOTON_DTYPE.itemsize, (L.orc_sizeof_photon(), PHOTON_DTYPE.itemsize)
            assert L.orc_n_counters() == len(COUNTER_NAMES)
            _lib = L
    return _lib


# ------------------------------------------------------------------ marshalling
class _Keep:
    """Holds the numpy arrays a C struct points into."""

    def __init__(self):
        self.refs = []

    def f32(self, a):
        a = np.ascontiguousarray(a, dtype=np.float32)
        self.refs.append(a)
        return _fp(a)


def atmosphere_struct(atm: dict, keep: _Keep) -> Atmosphere:
    s = Atmosphere()
    s.model = _MODEL[atm["model"]]
    s.n_nodes = int(atm["n_nodes"])
    s.n_const_minus_1 = float(np.float32(atm["n_const_minus_1"]))
    s.h0, s.dh = float(atm["h0"]), float(atm["dh"])
    s.refractivity = keep.f32(atm["refractivity"])
    s.overburden = keep.f32(atm["overburden"]) if atm.get("overburden") is not None else None
    s.earth_radius, s.h_obs = float(atm["earth_radius"]), float(atm["h_obs"])
    for k in ("rayleigh_X", "rayleigh_lambda", "aer_L", "aer_H", "aer_lambda", "aer_angstrom"):
        setattr(s, k, float(np.float32(atm[k])))
    ext = atm.get("ext_tau_v")
    s.n_ext_lambda = 0 if ext is None else int(np.asarray(ext).shape[0])
    s.ext_tau_v = keep.f32(np.asarray(ext).reshape(-1)) if s.n_ext_lambda else None
    s.ext_lambda0 = float(np.float32(atm.get("ext_lambda0_nm", 0.0)))
    s.ext_dlambda = float(np.float32(atm.get("ext_dlambda_nm", 1.0)))
    return s


def detector_struct(det: dict, keep: _Keep) -> Detector:
    s = Detector()
    s.hist_nx, s.hist_ny = int(det["hist_nx"]), int(det["hist_ny"])
    s.hist_x0, s.hist_y0, s.hist_cell = (float(np.float32(det[k])) for k in ("hist_x0", "hist_y0", "hist_cell"))
    tel = np.ascontiguousarray(det["tel_xyzr"], dtype=np.float32).reshape(-1, 4)
    s.n_tel = tel.shape[0]
    s.tel_xyzr = keep.f32(tel) if tel.shape[0] else None
    s.cam_enabled = int(bool(det["cam_enabled"]))
    s.cam_az_deg, s.cam_el_deg, s.cam_pix_deg = (float(np.float32(det[k])) for k in ("cam_az_deg", "cam_el_deg", "cam_pix_deg"))
    s.cam_rows, s.cam_cols, s.n_tbins = int(det["cam_rows"]), int(det["cam_cols"]), int(det["n_tbins"])
    s.t_ref_ns, s.t_bin_ns = float(det["t_ref_ns"]), float(np.float32(det["t_bin_ns"]))
    s.opt_enabled = int(bool(det.get("opt_enabled", False)))
    s.opt_az_deg, s.opt_el_deg = float(np.float32(det.get("opt_az_deg", 0.0))), float(np.float32(det.get("opt_el_deg", 90.0)))
    s.opt_focal_m = float(np.float32(det.get("opt_focal_m", 1.0)))
    s.opt_mirror_radius_m = float(np.float32(det.get("opt_mirror_radius_m", 0.0)))
    s.opt_camera_radius_m = float(np.float32(det.get("opt_camera_radius_m", 0.0)))
    s.opt_kind = int(det.get("opt_kind", 0))
    s.opt_lens_roc_m = float(np.float32(det.get("opt_lens_roc_m", 0.0)))
    s.opt_lens_thickness_m = float(np.float32(det.get("opt_lens_thickness_m", 0.0)))
    s.opt_lens_index = float(np.float32(det.get("opt_lens_index", 1.0)))
    absb = np.asarray(det.get("opt_absorbers", np.zeros((0, 7))), dtype=np.float32).reshape(-1, 7)
    s.opt_n_abs = len(absb)
    assert len(absb) <= 8
    for k, row in enumerate(absb):
        for j in range(7):
            s.opt_abs[k][j] = float(row[j])
    return s


def params_struct(par: dict, keep: _Keep) -> Params:
    s = Params()
    s.emit, s.trace, s.trans = _EMIT[par["emit"]], _TRACE[par["trace"]], _TRANS[par["trans"]]
    s.lv1, s.lv2, s.substeps = int(bool(par["lv1"])), int(bool(par["lv2"])), int(par.get("substeps", 1))
    for k in ("lambda_min_nm", "lambda_max_nm", "bunch_weight", "lv1_margin_rad", "lv2_margin_m",
              "fluor_yield_per_MeV", "aim_factor"):
        setattr(s, k, float(np.float32(par[k])))
    s.n_lines = len(par["line_nm"])
    s.line_nm = keep.f32(par["line_nm"]) if s.n_lines else None
    s.line_cdf = keep.f32(par["line_cdf"]) if s.n_lines else None
    s.disp_b_nm2 = float(np.float32(par.get("disp_b_nm2", 0.0)))
    s.disp_lambda0_nm = float(np.float32(par.get("disp_lambda0_nm", 400.0)))
    eff = par.get("eff")
    s.n_eff = 0 if eff is None else len(eff)
    s.flat_plane = int(par.get("flat_plane", 0))       # 0: off, 1 / True: analytic step (R19), 2: 3-D table (R21)
    s.eff = keep.f32(eff) if s.n_eff else None
    s.eff_lambda0_nm = float(np.float32(par.get("eff_lambda0_nm", 0.0)))
    s.eff_dlambda_nm = float(np.float32(par.get("eff_dlambda_nm", 1.0)))
    return s


def segments_struct(seg: dict, keep: _Keep) -> Segments:
    s = Segments()
    for k, _ in Segments._fields_:
        if k != "id":
            setattr(s, k, keep.f32(seg[k]))
    if seg.get("id") is not None:                       # explicit global segment ids (else seg_id_base + i)
        ids = np.ascontiguousarray(seg["id"], dtype=np.uint64)
        keep.refs.append(ids)
        s.id = ids.ctypes.data_as(C.POINTER(C.c_uint64))
    return s


# ------------------------------------------------------------------ step-level entry points (pins)
def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*[int(v) & 0xFFFFFFFF for v in ctr])
    k = (C.c_uint32 * 2)(*[int(v) & 0xFFFFFFFF for v in key])
    o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return [int(v) for v in o]


def uniform(r: int) -> float:
    return lib().orc_uniform(int(r))


def refractivity(atm: dict, h: float) -> float:
    keep = _Keep()
    return lib().orc_refractivity(C.byref(atmosphere_struct(atm, keep)), float(h))


def overburden(atm: dict, h: float) -> float:
    keep = _Keep()
    return lib().orc_overburden(C.byref(atmosphere_struct(atm, keep)), float(h))


def height(atm: dict, A) -> float:
    keep = _Keep()
    a = (C.c_double * 3)(*A)
    return lib().orc_height(C.byref(atmosphere_struct(atm, keep)), a)


def cherenkov_yield(charge, length, beta, n, lam1, lam2) -> float:
    return lib().orc_cherenkov_yield(charge, length, beta, n, lam1, lam2)


def rodrigues(P):
    p = (C.c_double * 3)(*P)
    m = (C.c_double * 9)()
    lib().orc_rodrigues(p, m)
    return np.array(m[:]).reshape(3, 3)


def cone_direction(M, cos_th, sin_th, phi):
    m = (C.c_double * 9)(*np.asarray(M, dtype=np.float64).ravel())
    u = (C.c_double * 3)()
    lib().orc_cone_direction(m, C.c_double(cos_th), C.c_double(sin_th), C.c_double(phi), u)
    return np.array(u[:])


def straight_line(A, u):
    a = (C.c_double * 3)(*A)
    d = (C.c_double * 3)(*u)
    i = (C.c_double * 3)()
    t = lib().orc_straight_line(a, d, i)
    return np.array(i[:]), t


def trace(atm: dict, spherical: bool, h_e, zen_rad, h_g, sub=1):
    """-> None (no-ground) or dict(disp, S, cT, X, tau_aer, sin_arr)."""
    keep = _Keep()
    out = (C.c_double * 6)()
    rc = lib().orc_trace(C.byref(atmosphere_struct(atm, keep)), int(spherical), float(h_e),
                         math.sin(zen_rad), math.cos(zen_rad), float(h_g), int(sub), out)
    if rc:
        return None
    return dict(disp=out[0], S=out[1], cT=out[2], X=out[3], tau_aer=out[4], sin_arr=out[5])


def build_table(atm: dict, table: dict, sub: int = 1) -> np.ndarray:
    keep = _Keep()
    out = np.empty((table["n_h"], table["n_zen"], 5), dtype=np.float32)
    lib().orc_build_table(C.byref(atmosphere_struct(atm, keep)), table["n_h"], table["n_zen"],
                          float(table["h_max"]), math.radians(float(np.float32(table["zen_max_deg"]))), int(sub), _fp(out))
    return out


def build_table_flat(atm: dict, table: dict, sub: int = 1) -> np.ndarray:
    """R21: [2 (even, odd in the pointing angle)][n_rho][n_h][n_zen][5], the correction relative to the flat plane."""
    keep = _Keep()
    out = np.empty((2, table["n_rho"], table["n_h"], table["n_zen"], 5), dtype=np.float32)
    lib().orc_build_table_flat(C.byref(atmosphere_struct(atm, keep)), table["n_h"], table["n_zen"], table["n_rho"],
                           float(table["h_max"]), math.radians(float(np.float32(table["zen_max_deg"]))),
                           float(np.float32(table["rho_max_m"])), int(sub), _fp(out))
    return out


def trace_cyl(atm: dict, h_e, zen_rad, psi_rad, h_g, sub=1):
    """R24: the layered ray in the cylindrical model; returns (no_ground, [central angle, S, cT, X, tau, y', ux', uy', uz'])."""
    keep = _Keep()
    out = (C.c_double * 9)()
    bad = lib().orc_trace_cyl(C.byref(atmosphere_struct(atm, keep)), float(h_e), math.sin(zen_rad), math.cos(zen_rad),
                              float(psi_rad), float(h_g), int(sub), out)
    return bool(bad), list(out)


def cyl_correction(atm: dict, h_e, zen_rad, psi_rad, sub=1):
    """R24: (bad, [along, across, dt_ns, X_slant, tau_aer]) of the cylindrical ray against the straight line."""
    keep = _Keep()
    out = (C.c_double * 5)()
    bad = lib().orc_cyl_correction(C.byref(atmosphere_struct(atm, keep)), float(h_e), math.sin(zen_rad), math.cos(zen_rad),
                                   float(psi_rad), int(sub), out)
    return bool(bad), list(out)


def build_table_cyl(atm: dict, table: dict, sub: int = 1) -> np.ndarray:
    """R24: [n_c][n_h][n_zen][5], third axis c = cos^2(psi); ch1 = across displacement / (sin psi cos psi)."""
    keep = _Keep()
    out = np.empty((table["n_c"], table["n_h"], table["n_zen"], 5), dtype=np.float32)
    lib().orc_build_table_cyl(C.byref(atmosphere_struct(atm, keep)), table["n_h"], table["n_zen"], table["n_c"],
                              float(table["h_max"]), math.radians(float(np.float32(table["zen_max_deg"]))), int(sub), _fp(out))
    return out


def table_struct(table: dict, data: np.ndarray, keep: _Keep, data3: np.ndarray | None = None) -> Table:
    t = Table()
    t.n_h, t.n_zen, t.n_ch = int(table["n_h"]), int(table["n_zen"]), int(data.shape[-1])
    t.h_max = float(table["h_max"])
    t.zen_max_rad = math.radians(float(np.float32(table["zen_max_deg"])))
    t.data = keep.f32(data)
    if data3 is not None:
        if data3.ndim == 4:                                 # cylindrical model: [n_c][n_h][n_zen][5], third axis c in [0, 1]
            t.n_rho, t.rho_max = int(table["n_c"]), 1.0
        else:
            t.n_rho, t.rho_max = int(table["n_rho"]), float(np.float32(table["rho_max_m"]))
        t.data3 = keep.f32(data3)
    return t


def table_flat_lookup(table: dict, data: np.ndarray, data3: np.ndarray, h: float, zen_rad: float, rho: float, cos_chi: float):
    keep = _Keep()
    t = table_struct(table, data, keep, data3)
    out = (C.c_double * 5)()
    perp = C.c_double(0.0)
    bad = lib().orc_table_flat_lookup(C.byref(t), float(h), float(zen_rad), float(rho), float(cos_chi), out, C.byref(perp))
    return bool(bad), list(out), perp.value


def table_lookup(table: dict, data: np.ndarray, h: float, zen_rad: float):
    keep = _Keep()
    out = (C.c_double * 5)()
    rc = lib().orc_table_lookup(C.byref(table_struct(table, data, keep)), float(h), float(zen_rad), out)
    return None if rc else np.array(out[:])


def transmission(atm: dict, x_slant, tau_aer, lambda_nm) -> float:
    keep = _Keep()
    return lib().orc_transmission(C.byref(atmosphere_struct(atm, keep)), x_slant, tau_aer, lambda_nm)


def ray_sphere(I, u, c, r):
    s = C.c_double()
    hit = lib().orc_ray_sphere((C.c_double * 3)(*I), (C.c_double * 3)(*u), (C.c_double * 3)(*c),
                               C.c_double(r), C.byref(s))
    return (bool(hit), s.value if hit else None)


def camera_pixel(det: dict, u_arr) -> int:
    keep = _Keep()
    return lib().orc_camera_pixel(C.byref(detector_struct(det, keep)), (C.c_double * 3)(*u_arr))


# ------------------------------------------------------------------ whole path
_table_cache = {}


def _table_key(cfg: dict, sub: int):
    atm = cfg["atmosphere"]
    return (atm["model"], atm["h_obs"], atm["refractivity"].tobytes()[:4096], atm["overburden"].tobytes()[:4096],
            atm["aer_L"], atm["aer_H"], tuple(sorted(cfg["table"].items())), sub)


def table_for(cfg: dict, sub: int = 1) -> np.ndarray | None:
    if cfg.get("table") is None:
        return None
    key = _table_key(cfg, sub)
    if key not in _table_cache:
        _table_cache[key] = build_table(cfg["atmosphere"], cfg["table"], sub)
    return _table_cache[key]


def table_cyl_for(cfg: dict, sub: int = 1) -> np.ndarray | None:
    """The cylindrical model's table (R24) if the config's table has the third axis (n_c)."""
    if cfg.get("table") is None or not cfg["table"].get("n_c"):
        return None
    key = ("cyl",) + _table_key(cfg, sub)
    if key not in _table_cache:
        _table_cache[key] = build_table_cyl(cfg["atmosphere"], cfg["table"], sub)
    return _table_cache[key]


def table_flat_for(cfg: dict, sub: int = 1) -> np.ndarray | None:
    """The flat-plane table of R21 if the config's table has the extra axes (n_rho, rho_max_m)."""
    if cfg.get("table") is None or not cfg["table"].get("n_rho"):
        return None
    key = ("t3",) + _table_key(cfg, sub)
    if key not in _table_cache:
        _table_cache[key] = build_table_flat(cfg["atmosphere"], cfg["table"], sub)
    return _table_cache[key]


def run(cfg: dict, record: bool = True, table_data: np.ndarray | None = None, threads: int | None = None) -> dict:
    """Run the whole path on cfg['segments'].

    Returns dict(hist, tel_counts, counters{name: int}, n_bunch, photons (structured array, every
    emitted photon with its status; only if record)).
    """
    L = lib()
    L.orc_set_threads.argtypes = [C.c_int]
    L.orc_set_threads.restype = C.c_int
    L.orc_set_threads(int(threads) if threads is not None else 0)
    keep = _Keep()
    atm = atmosphere_struct(cfg["atmosphere"], keep)
    det = detector_struct(cfg["detector"], keep)
    par = params_struct(cfg["params"], keep)
    seg = segments_struct(cfg["segments"], keep)
    n_seg = len(cfg["segments"]["x"])
    tab_ptr = None
    if cfg.get("table") is not None and cfg["params"]["trace"] == "table":
        cyl = cfg["atmosphere"]["model"] == "cylindrical"
        if table_data is None:
            table_data = table_for(cfg) if not cyl else np.zeros((cfg["table"]["n_h"], cfg["table"]["n_zen"], 5), np.float32)
        data3 = table_cyl_for(cfg) if cyl else (table_flat_for(cfg) if int(cfg["params"].get("flat_plane", 0)) == 2 else None)
        tab = table_struct(cfg["table"], table_data, keep, data3)
        tab_ptr = C.byref(tab)
    dd = cfg["detector"]
    n_hist = dd["n_tbins"] * dd["cam_rows"] * dd["cam_cols"] if dd["cam_enabled"] else dd["hist_nx"] * dd["hist_ny"]
    hist = np.zeros(max(n_hist, 1), dtype=np.float64)
    tel = np.zeros(max(det.n_tel, 1), dtype=np.float64)
    cnt = np.zeros(len(COUNTER_NAMES), dtype=np.uint64)
    seed, base = int(cfg["seed"]), int(cfg["seg_id_base"])
    n_bunch = np.zeros(n_seg, dtype=np.int64)
    total = L.orc_count(C.byref(atm), C.byref(det), C.byref(par), tab_ptr, C.byref(seg), C.c_int64(n_seg),
                        C.c_int64(base), C.c_uint64(seed), n_bunch.ctypes.data_as(C.POINTER(C.c_int64)))
    photons, offs_p, ph_p = None, None, None
    if record:
        offsets = np.zeros(n_seg, dtype=np.int64)
        np.cumsum(n_bunch[:-1], out=offsets[1:])
        photons = np.zeros(int(total), dtype=PHOTON_DTYPE)
        offs_p = offsets.ctypes.data_as(C.POINTER(C.c_int64))
        ph_p = photons.ctypes.data_as(C.c_void_p)
    rc = L.orc_run(C.byref(atm), C.byref(det), C.byref(par), tab_ptr, C.byref(seg), C.c_int64(n_seg),
                   C.c_int64(base), C.c_uint64(seed),
                   hist.ctypes.data_as(C.POINTER(C.c_double)), tel.ctypes.data_as(C.POINTER(C.c_double)),
                   cnt.ctypes.data_as(C.POINTER(C.c_uint64)), C.c_int(1 if record else 0), offs_p, ph_p)
    if rc:
        raise RuntimeError(f"orc_run failed: {rc}")
    return dict(hist=hist[:n_hist], tel_counts=tel[:det.n_tel], n_bunch=n_bunch, total_bunches=int(total),
                counters={k: int(v) for k, v in zip(COUNTER_NAMES, cnt)}, photons=photons)


def substep_tracks(tracks: dict, B, tol_m: float, max_sub: int = 4096) -> dict:
    """R16: cut helical tracks (dict of float32 arrays x,y,z,dx,dy,dz,len,beta,t0,charge,p_GeV) into chords.
    Returns dict(segments={x..charge,edep}, offsets=int64[n+1])."""
    L = lib()
    n = len(tracks["x"])
    Bd = (C.c_double * 3)(*[float(np.float32(b)) for b in B])
    counts = np.zeros(n, dtype=np.int64)
    arr = lambda v: (C.c_double * 3)(*[float(x) for x in v])
    args = []
    for i in range(n):
        a = (arr([tracks[k][i] for k in ("x", "y", "z")]), arr([tracks[k][i] for k in ("dx", "dy", "dz")]),
             float(tracks["len"][i]), float(tracks["beta"][i]), float(tracks["t0"][i]), float(tracks["charge"][i]),
             float(tracks["p_GeV"][i]))
        args.append(a)
        counts[i] = L.orc_substep_track(a[0], a[1], a[2], a[3], a[4], a[5], a[6], Bd, float(np.float32(tol_m)), int(max_sub), None)
    offsets = np.concatenate([[0], np.cumsum(counts)]).astype(np.int64)
    out = np.zeros((int(offsets[-1]), 10), dtype=np.float32)
    for i, a in enumerate(args):
        L.orc_substep_track(a[0], a[1], a[2], a[3], a[4], a[5], a[6], Bd, float(np.float32(tol_m)), int(max_sub),
                            out[offsets[i]:].ctypes.data_as(C.POINTER(C.c_float)))
    names = ("x", "y", "z", "dx", "dy", "dz", "len", "beta", "t0", "charge")
    seg = {k: np.ascontiguousarray(out[:, j]) for j, k in enumerate(names)}
    seg["edep"] = np.zeros(len(out), dtype=np.float32)
    return dict(segments=seg, offsets=offsets)


def substep_tracks_ms(atm: dict, tracks: dict, B, tol_m: float, ms_max_step_m: float, ms_X0: float = 36.62,
                      seed: int = 1, track_id_base: int = 0, max_sub: int = 4096) -> dict:
    """R18: R16's magnetic pieces plus Highland multiple scattering per piece (sequential random walk)."""
    L = lib()
    keep = _Keep()
    a_s = atmosphere_struct(atm, keep)
    n = len(tracks["x"])
    Bd = (C.c_double * 3)(*[float(np.float32(b)) for b in B])
    arr = lambda v: (C.c_double * 3)(*[float(x) for x in v])
    counts = np.zeros(n, dtype=np.int64)
    calls = []
    for i in range(n):
        a = (arr([tracks[k][i] for k in ("x", "y", "z")]), arr([tracks[k][i] for k in ("dx", "dy", "dz")]),
             float(tracks["len"][i]), float(tracks["beta"][i]), float(tracks["t0"][i]), float(tracks["charge"][i]),
             float(tracks["p_GeV"][i]))
        calls.append(a)
        counts[i] = L.orc_substep_track_ms(C.byref(a_s), a[0], a[1], a[2], a[3], a[4], a[5], a[6], Bd, float(np.float32(tol_m)),
                                           float(np.float32(ms_max_step_m)), float(np.float32(ms_X0)), C.c_uint64(seed),
                                           C.c_uint64(track_id_base + i), int(max_sub), None)
    offsets = np.concatenate([[0], np.cumsum(counts)]).astype(np.int64)
    out = np.zeros((int(offsets[-1]), 10), dtype=np.float32)
    for i, a in enumerate(calls):
        L.orc_substep_track_ms(C.byref(a_s), a[0], a[1], a[2], a[3], a[4], a[5], a[6], Bd, float(np.float32(tol_m)),
                               float(np.float32(ms_max_step_m)), float(np.float32(ms_X0)), C.c_uint64(seed),
                               C.c_uint64(track_id_base + i), int(max_sub),
                               out[offsets[i]:].ctypes.data_as(C.POINTER(C.c_float)))
    names = ("x", "y", "z", "dx", "dy", "dz", "len", "beta", "t0", "charge")
    seg = {k: np.ascontiguousarray(out[:, j]) for j, k in enumerate(names)}
    seg["edep"] = np.zeros(len(out), dtype=np.float32)
    return dict(segments=seg, offsets=offsets)
