"""Thin Python binding over the C-ABI of ``libc8ph.so`` (include/c8ph.h).

Argument marshalling only: every step of the hot path runs in the CUDA kernels of the library.
PyTorch is used for device memory and streams.  There is no CPU fallback: if the shared library
is missing or cannot be loaded, importing a symbol raises.
"""
from __future__ import annotations

import ctypes as C
import math
import os
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# C8PH_LIB selects another build of the same library (an A/B build made with `build.py --define ... --out ...`)
LIB_PATH = os.environ.get("C8PH_LIB") or os.path.join(_HERE, "libc8ph.so")

OK, E_ARG, E_STATE, E_CUDA, E_NOMEM = 0, -1, -2, -3, -4
ATM = {"homogeneous": 0, "planar": 1, "spherical": 2, "cylindrical": 3}
EMIT = {"cherenkov": 0, "fluorescence": 1}
TRACE = {"straight": 0, "numeric": 1, "table": 2}
TRANS = {"off": 0, "weight": 1, "roulette": 2}
WRITE = {"none": 0, "all": 1, "tel": 2}
TABLE_CHANNELS = 5
TEL_NONE = 0x3FFF
COUNTER_NAMES = ("segments", "seg_below_threshold", "seg_lv1", "seg_emitting", "emitted", "upgoing", "lv2",
                 "table_range", "roulette", "landed", "in_grid", "tel_hit", "cam_hit", "written", "overflow",
                 "clipped", "nonfinite")
N_COUNTERS = len(COUNTER_NAMES)

EXPORTS = ("c8ph_create", "c8ph_destroy", "c8ph_last_error", "c8ph_version", "c8ph_init_atmosphere",
           "c8ph_build_trace_table", "c8ph_get_trace_table", "c8ph_set_trace_table", "c8ph_set_detector",
           "c8ph_emit_propagate", "c8ph_emit_propagate_host", "c8ph_last_kernel_ms", "c8ph_launch_count",
           "c8ph_counter_name", "c8ph_substep_plan", "c8ph_substep_fill", "c8ph_set_line_spectrum", "c8ph_set_efficiency",
           "c8ph_get_trace_table_flat", "c8ph_get_trace_table_cyl", "c8ph_substep_plan_static", "c8ph_substep_plan_static_error")
SUBSTEP_STATIC_MAX_TRACKS = 4194304      # C8PH_SUBSTEP_STATIC_MAX_TRACKS

PHOTON_DTYPE = np.dtype([("x", "<f4"), ("y", "<f4"), ("ux", "<f4"), ("uy", "<f4"), ("t_ns", "<f4"),
                         ("lambda_nm", "<f4"), ("seg", "<u4"), ("j_tel", "<u4")])
assert PHOTON_DTYPE.itemsize == 32

_fp = C.POINTER(C.c_float)


class AtmosphereDesc(C.Structure):
    _fields_ = [("size", C.c_uint32), ("model", C.c_int32), ("n_const_minus_1", C.c_float),
                ("h0_m", C.c_float), ("dh_m", C.c_float), ("n_nodes", C.c_int32),
                ("refractivity", _fp), ("overburden_gcm2", _fp),
                ("earth_radius_m", C.c_float), ("h_obs_m", C.c_float),
                ("rayleigh_X_gcm2", C.c_float), ("rayleigh_lambda_nm", C.c_float),
                ("aer_L_m", C.c_float), ("aer_H_m", C.c_float), ("aer_lambda_nm", C.c_float),
                ("aer_angstrom", C.c_float),
                ("n_ext_lambda", C.c_int32), ("ext_lambda0_nm", C.c_float), ("ext_dlambda_nm", C.c_float), ("ext_tau_v", _fp)]


class TableDesc(C.Structure):
    _fields_ = [("size", C.c_uint32), ("n_h", C.c_int32), ("n_zen", C.c_int32),
                ("h_max_m", C.c_float), ("zen_max_deg", C.c_float), ("substeps", C.c_int32),
                ("n_rho", C.c_int32), ("rho_max_m", C.c_float), ("n_c", C.c_int32)]


class Detector(C.Structure):
    _fields_ = [("size", C.c_uint32), ("hist_nx", C.c_int32), ("hist_ny", C.c_int32),
                ("hist_x0", C.c_float), ("hist_y0", C.c_float), ("hist_cell", C.c_float),
                ("n_tel", C.c_int32), ("tel_xyzr", _fp), ("cam_enabled", C.c_int32),
                ("cam_axis_az_deg", C.c_float), ("cam_axis_el_deg", C.c_float), ("cam_pix_deg", C.c_float),
                ("cam_rows", C.c_int32), ("cam_cols", C.c_int32), ("n_tbins", C.c_int32),
                ("t_ref_ns", C.c_double), ("t_bin_ns", C.c_float),
                ("opt_enabled", C.c_int32), ("opt_az_deg", C.c_float), ("opt_el_deg", C.c_float),
                ("opt_focal_m", C.c_float), ("opt_mirror_radius_m", C.c_float), ("opt_camera_radius_m", C.c_float),
                ("opt_kind", C.c_int32), ("opt_lens_roc_m", C.c_float), ("opt_lens_thickness_m", C.c_float),
                ("opt_lens_index", C.c_float), ("opt_n_abs", C.c_int32), ("opt_abs", (C.c_float * 7) * 8)]


class Params(C.Structure):
    _fields_ = [("size", C.c_uint32), ("emit", C.c_int32), ("trace", C.c_int32), ("trans", C.c_int32),
                ("write", C.c_int32), ("filter_lv1", C.c_int32), ("filter_lv2", C.c_int32),
                ("lambda_min_nm", C.c_float), ("lambda_max_nm", C.c_float), ("bunch_weight", C.c_float),
                ("lv1_margin_rad", C.c_float), ("lv2_margin_m", C.c_float),
                ("fluor_yield_per_MeV", C.c_float), ("aim_factor", C.c_float),
                ("disp_b_nm2", C.c_float), ("disp_lambda0_nm", C.c_float),
                ("use_efficiency", C.c_int32), ("flat_plane", C.c_int32)]


class Segments(C.Structure):
    _fields_ = [("size", C.c_uint32)] + [(k, C.c_void_p) for k in
                                          ("x", "y", "z", "dx", "dy", "dz", "len", "beta", "t0", "charge", "edep", "id")]


class SegmentsOut(C.Structure):
    _fields_ = [("size", C.c_uint32)] + [(k, C.c_void_p) for k in
                                          ("x", "y", "z", "dx", "dy", "dz", "len", "beta", "t0", "charge", "edep")]


class SubstepDesc(C.Structure):
    _fields_ = [("size", C.c_uint32), ("B_tesla", C.c_float * 3), ("tol_m", C.c_float), ("max_sub", C.c_int32),
                ("ms_enabled", C.c_int32), ("ms_max_step_m", C.c_float), ("ms_X0_gcm2", C.c_float),
                ("seed", C.c_uint64), ("track_id_base", C.c_int64), ("clipped", C.c_void_p)]


class Outputs(C.Structure):
    _fields_ = [("size", C.c_uint32), ("hist", C.c_void_p), ("tel_counts", C.c_void_p), ("photons", C.c_void_p),
                ("photon_weight", C.c_void_p), ("photon_capacity", C.c_int64), ("counters", C.c_void_p)]


SEG_FIELDS = ("x", "y", "z", "dx", "dy", "dz", "len", "beta", "t0", "charge", "edep")

_lib = None


def load_library():
    """dlopen libc8ph.so; raises if it is missing (there is no fallback path)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2405_04229_b200.build` "
                               "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        L.c8ph_create.argtypes = [C.POINTER(C.c_void_p), C.c_int]
        L.c8ph_destroy.argtypes = [C.c_void_p]
        L.c8ph_last_error.argtypes = [C.c_void_p]
        L.c8ph_last_error.restype = C.c_char_p
        L.c8ph_init_atmosphere.argtypes = [C.c_void_p, C.POINTER(AtmosphereDesc)]
        L.c8ph_build_trace_table.argtypes = [C.c_void_p, C.POINTER(TableDesc), C.c_void_p]
        L.c8ph_get_trace_table.argtypes = [C.c_void_p, _fp, C.c_int64]
        L.c8ph_set_trace_table.argtypes = [C.c_void_p, C.POINTER(TableDesc), _fp]
        L.c8ph_get_trace_table_flat.argtypes = [C.c_void_p, _fp, C.c_int64]
        L.c8ph_get_trace_table_cyl.argtypes = [C.c_void_p, _fp, C.c_int64]
        L.c8ph_set_detector.argtypes = [C.c_void_p, C.POINTER(Detector)]
        L.c8ph_emit_propagate.argtypes = [C.c_void_p, C.POINTER(Segments), C.c_int64, C.c_int64,
                                          C.POINTER(Params), C.c_uint64, C.POINTER(Outputs), C.c_void_p]
        L.c8ph_emit_propagate_host.argtypes = [C.c_void_p, C.POINTER(Segments), C.c_int64, C.c_int64,
                                               C.POINTER(Params), C.c_uint64, C.POINTER(Outputs)]
        L.c8ph_last_kernel_ms.argtypes = [C.c_void_p]
        L.c8ph_last_kernel_ms.restype = C.c_float
        L.c8ph_launch_count.argtypes = [C.c_void_p]
        L.c8ph_launch_count.restype = C.c_int64
        L.c8ph_substep_plan.argtypes = [C.c_void_p, C.POINTER(Segments), C.c_void_p, C.c_int64, C.POINTER(SubstepDesc),
                                        C.c_void_p, C.c_void_p]
        L.c8ph_substep_fill.argtypes = [C.c_void_p, C.POINTER(Segments), C.c_void_p, C.c_int64, C.POINTER(SubstepDesc),
                                        C.c_void_p, C.POINTER(SegmentsOut), C.c_void_p]
        L.c8ph_substep_plan_static.argtypes = [C.POINTER(Segments), C.c_void_p, C.c_int64, C.POINTER(SubstepDesc), C.c_void_p, C.c_void_p]
        L.c8ph_substep_plan_static_error.restype = C.c_char_p
        L.c8ph_set_line_spectrum.argtypes = [C.c_void_p, C.c_int32, _fp, _fp]
        L.c8ph_set_efficiency.argtypes = [C.c_void_p, C.c_int32, C.c_float, C.c_float, _fp]
        L.c8ph_counter_name.argtypes = [C.c_int]
        L.c8ph_counter_name.restype = C.c_char_p
        _lib = L
    return _lib


class C8phError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libc8ph error {code}: {msg}")
        self.code = code


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


class Context:
    """One libc8ph context on one CUDA device.  Method names follow the C entry points."""

    def __init__(self, device: int = 0):
        self.lib = load_library()
        self._h = C.c_void_p()
        rc = self.lib.c8ph_create(C.byref(self._h), int(device))
        if rc:
            raise C8phError(rc, self.lib.c8ph_last_error(None).decode())
        self.device = int(device)
        self._det = None
        self._keep = []

    def close(self):
        if self._h:
            self.lib.c8ph_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc):
        if rc:
            raise C8phError(rc, self.lib.c8ph_last_error(self._h).decode())

    # ---- setup ---------------------------------------------------------------------------------
    def init_atmosphere(self, atm: dict):
        d = AtmosphereDesc()
        d.size = C.sizeof(AtmosphereDesc)
        d.model = ATM[atm["model"]]
        d.n_const_minus_1 = float(atm["n_const_minus_1"])
        d.h0_m, d.dh_m, d.n_nodes = float(atm["h0"]), float(atm["dh"]), int(atm["n_nodes"])
        eta = _f32(atm["refractivity"])
        d.refractivity = eta.ctypes.data_as(_fp)
        xv = None
        if atm.get("overburden") is not None:
            xv = _f32(atm["overburden"])
            d.overburden_gcm2 = xv.ctypes.data_as(_fp)
        d.earth_radius_m, d.h_obs_m = float(atm["earth_radius"]), float(atm["h_obs"])
        d.rayleigh_X_gcm2, d.rayleigh_lambda_nm = float(atm["rayleigh_X"]), float(atm["rayleigh_lambda"])
        d.aer_L_m, d.aer_H_m = float(atm["aer_L"]), float(atm["aer_H"])
        d.aer_lambda_nm, d.aer_angstrom = float(atm["aer_lambda"]), float(atm["aer_angstrom"])
        ext = atm.get("ext_tau_v")
        if ext is not None:
            ext = _f32(np.asarray(ext))
            d.n_ext_lambda = ext.shape[0]
            d.ext_tau_v = ext.ctypes.data_as(_fp)
            d.ext_lambda0_nm, d.ext_dlambda_nm = float(atm["ext_lambda0_nm"]), float(atm["ext_dlambda_nm"])
        self._check(self.lib.c8ph_init_atmosphere(self._h, C.byref(d)))

    @staticmethod
    def _table_desc(table: dict) -> TableDesc:
        t = TableDesc()
        t.size = C.sizeof(TableDesc)
        t.n_h, t.n_zen = int(table["n_h"]), int(table["n_zen"])
        t.h_max_m, t.zen_max_deg = float(table["h_max"]), float(table["zen_max_deg"])
        t.substeps = int(table.get("substeps", 1))
        t.n_rho, t.rho_max_m = int(table.get("n_rho", 0) or 0), float(table.get("rho_max_m", 0.0) or 0.0)
        t.n_c = int(table.get("n_c", 0) or 0)
        return t

    def get_trace_table_cyl(self) -> np.ndarray:
        """[n_c][n_h][n_zen][4] texels of the cylindrical model's table (R24)."""
        t = self._table
        out = np.empty((t["n_c"], t["n_h"], t["n_zen"], 4), dtype=np.float32)
        self._check(self.lib.c8ph_get_trace_table_cyl(self._h, out.ctypes.data_as(_fp), out.size))
        return out

    def get_trace_table_flat(self) -> np.ndarray:
        """[2 (even, odd)][n_rho][n_h][n_zen][4] texels of the flat-plane table (R21)."""
        t = self._table
        out = np.empty((2, t["n_rho"], t["n_h"], t["n_zen"], 4), dtype=np.float32)
        self._check(self.lib.c8ph_get_trace_table_flat(self._h, out.ctypes.data_as(_fp), out.size))
        return out

    def build_trace_table(self, table: dict, stream=None):
        self._table = dict(table)
        self._check(self.lib.c8ph_build_trace_table(self._h, C.byref(self._table_desc(table)), _stream_ptr(stream)))

    def get_trace_table(self) -> np.ndarray:
        t = self._table
        out = np.empty((t["n_h"], t["n_zen"], TABLE_CHANNELS), dtype=np.float32)
        self._check(self.lib.c8ph_get_trace_table(self._h, out.ctypes.data_as(_fp), out.size))
        return out

    def set_trace_table(self, table: dict, data: np.ndarray):
        self._table = dict(table)
        data = _f32(data)
        assert data.shape == (table["n_h"], table["n_zen"], TABLE_CHANNELS)
        self._check(self.lib.c8ph_set_trace_table(self._h, C.byref(self._table_desc(dict(table, n_rho=0, n_c=0))), data.ctypes.data_as(_fp)))

    def set_detector(self, det: dict):
        d = Detector()
        d.size = C.sizeof(Detector)
        d.hist_nx, d.hist_ny = int(det["hist_nx"]), int(det["hist_ny"])
        d.hist_x0, d.hist_y0, d.hist_cell = float(det["hist_x0"]), float(det["hist_y0"]), float(det["hist_cell"])
        tel = _f32(det["tel_xyzr"]).reshape(-1, 4)
        d.n_tel = tel.shape[0]
        d.tel_xyzr = tel.ctypes.data_as(_fp) if tel.shape[0] else None
        d.cam_enabled = int(bool(det["cam_enabled"]))
        d.cam_axis_az_deg, d.cam_axis_el_deg = float(det["cam_az_deg"]), float(det["cam_el_deg"])
        d.cam_pix_deg = float(det["cam_pix_deg"])
        d.cam_rows, d.cam_cols, d.n_tbins = int(det["cam_rows"]), int(det["cam_cols"]), int(det["n_tbins"])
        d.t_ref_ns, d.t_bin_ns = float(det["t_ref_ns"]), float(det["t_bin_ns"])
        d.opt_enabled = int(bool(det.get("opt_enabled", False)))
        d.opt_az_deg, d.opt_el_deg = float(det.get("opt_az_deg", 0.0)), float(det.get("opt_el_deg", 90.0))
        d.opt_focal_m = float(det.get("opt_focal_m", 1.0))
        d.opt_mirror_radius_m, d.opt_camera_radius_m = float(det.get("opt_mirror_radius_m", 0.0)), float(det.get("opt_camera_radius_m", 0.0))
        d.opt_kind = int(det.get("opt_kind", 0))
        d.opt_lens_roc_m, d.opt_lens_thickness_m = float(det.get("opt_lens_roc_m", 0.0)), float(det.get("opt_lens_thickness_m", 0.0))
        d.opt_lens_index = float(det.get("opt_lens_index", 1.0))
        absb = _f32(det.get("opt_absorbers", np.zeros((0, 7), np.float32))).reshape(-1, 7)
        d.opt_n_abs = len(absb)
        for k, row in enumerate(absb[:8]):
            for j in range(7):
                d.opt_abs[k][j] = float(row[j])
        self._check(self.lib.c8ph_set_detector(self._h, C.byref(d)))
        self._det = dict(det)
        self._n_tel = tel.shape[0]

    def n_hist(self) -> int:
        d = self._det
        if d["cam_enabled"]:
            return d["cam_rows"] * d["cam_cols"] * d["n_tbins"]
        return d["hist_nx"] * d["hist_ny"]

    def _params(self, par: dict):
        p = Params()
        p.size = C.sizeof(Params)
        p.emit, p.trace, p.trans = EMIT[par["emit"]], TRACE[par["trace"]], TRANS[par["trans"]]
        p.write = WRITE[par["write"]]
        p.filter_lv1, p.filter_lv2 = int(bool(par["lv1"])), int(bool(par["lv2"]))
        p.lambda_min_nm, p.lambda_max_nm = float(par["lambda_min_nm"]), float(par["lambda_max_nm"])
        p.bunch_weight = float(par["bunch_weight"])
        p.lv1_margin_rad, p.lv2_margin_m = float(par["lv1_margin_rad"]), float(par["lv2_margin_m"])
        p.fluor_yield_per_MeV, p.aim_factor = float(par["fluor_yield_per_MeV"]), float(par["aim_factor"])
        p.disp_b_nm2, p.disp_lambda0_nm = float(par.get("disp_b_nm2", 0.0)), float(par.get("disp_lambda0_nm", 400.0))
        p.use_efficiency = int(par.get("eff") is not None and len(par["eff"]) > 0)
        p.flat_plane = int(par.get("flat_plane", 0))                   # 0 off, 1 / True analytic step (R19), 2 table (R21)
        self._sync_spectra(par)
        return p, None

    # ---- wavelength tables of the context (set-up calls; the hot call copies nothing) ------------
    def set_line_spectrum(self, line_nm, line_cdf):
        ln, lc = _f32(line_nm), _f32(line_cdf)
        self._check(self.lib.c8ph_set_line_spectrum(self._h, len(ln), ln.ctypes.data_as(_fp), lc.ctypes.data_as(_fp)))
        self._lines_key = (ln.tobytes(), lc.tobytes())

    def set_efficiency(self, eff, lambda0_nm: float, dlambda_nm: float):
        ef = _f32(eff if eff is not None else [])
        self._check(self.lib.c8ph_set_efficiency(self._h, len(ef), float(lambda0_nm), float(dlambda_nm),
                                                 ef.ctypes.data_as(_fp) if len(ef) else None))
        self._eff_key = (ef.tobytes(), float(lambda0_nm), float(dlambda_nm))

    def _sync_spectra(self, par: dict):
        """Convenience of this binding (marshalling only): a run-parameter dict may carry the line spectrum and the
        efficiency table; they are handed to the library's set-up calls when they differ from what the context holds."""
        if par["emit"] == "fluorescence" and len(par["line_nm"]):
            key = (_f32(par["line_nm"]).tobytes(), _f32(par["line_cdf"]).tobytes())
            if getattr(self, "_lines_key", None) != key:
                self.set_line_spectrum(par["line_nm"], par["line_cdf"])
        eff = par.get("eff")
        if eff is not None and len(eff):
            key = (_f32(eff).tobytes(), float(par.get("eff_lambda0_nm", 0.0)), float(par.get("eff_dlambda_nm", 1.0)))
            if getattr(self, "_eff_key", None) != key:
                self.set_efficiency(eff, key[1], key[2])

    # ---- the hot call, DEVICE buffers ------------------------------------------------------------
    def emit_propagate(self, seg_dev: dict, n_segments: int, seg_id_base: int, par: dict, seed: int,
                       out: dict, stream=None):
        """seg_dev: dict of torch CUDA float32 tensors (SoA); out: dict with torch CUDA tensors
        'hist' (f32), 'tel_counts' (f32), 'photons' (uint8, 32 B/record), 'photon_weight' (f32),
        'counters' (int64[N_COUNTERS]); any but 'counters' may be None.  Asynchronous."""
        s = Segments()
        s.size = C.sizeof(Segments)
        for k in SEG_FIELDS:
            t = seg_dev.get(k)
            setattr(s, k, _dev_ptr(t, "float32", n_segments) if t is not None else None)
        if seg_dev.get("id") is not None:                                # explicit global segment ids (int64 tensor)
            s.id = _dev_ptr(seg_dev["id"], "int64", n_segments)
        o = Outputs()
        o.size = C.sizeof(Outputs)
        o.hist = _dev_ptr(out.get("hist"), "float32", self.n_hist())
        o.tel_counts = _dev_ptr(out.get("tel_counts"), "float32", self._n_tel)
        ph = out.get("photons")
        cap = 0
        if ph is not None:
            cap = ph.numel() * ph.element_size() // 32
            o.photons = _dev_ptr(ph, None, 0)
        pw = out.get("photon_weight")
        o.photon_weight = _dev_ptr(pw, "float32", cap) if pw is not None else None
        o.photon_capacity = cap
        o.counters = _dev_ptr(out["counters"], "int64", N_COUNTERS)
        p, keep = self._params(par)
        self._check(self.lib.c8ph_emit_propagate(self._h, C.byref(s), int(n_segments), int(seg_id_base),
                                                 C.byref(p), C.c_uint64(int(seed)), C.byref(o), _stream_ptr(stream)))
        del keep

    # ---- the same call with HOST buffers (end-to-end path) ---------------------------------------
    def emit_propagate_host(self, seg_host: dict, n_segments: int, seg_id_base: int, par: dict, seed: int,
                            photon_capacity: int = 0, want_weight: bool = False, out: Optional[dict] = None) -> dict:
        """seg_host: dict of numpy float32 arrays (or pinned torch CPU tensors).  Returns a dict of
        numpy arrays: hist, tel_counts, counters{name: int}, photons (structured), photon_weight."""
        s = Segments()
        s.size = C.sizeof(Segments)
        keep = []
        for k in SEG_FIELDS:
            a = seg_host.get(k)
            if a is None:
                continue
            if hasattr(a, "data_ptr"):
                assert str(a.dtype) == "torch.float32" and a.is_contiguous() and a.numel() >= n_segments
                setattr(s, k, a.data_ptr())
                keep.append(a)
            else:
                a = _f32(a)
                assert a.size >= n_segments
                keep.append(a)
                setattr(s, k, a.ctypes.data)
        if seg_host.get("id") is not None:
            ids = seg_host["id"]
            if hasattr(ids, "data_ptr"):
                assert str(ids.dtype) in ("torch.int64", "torch.uint64") and ids.is_contiguous() and ids.numel() >= n_segments
                s.id = ids.data_ptr()
            else:
                ids = np.ascontiguousarray(ids, dtype=np.uint64)
                s.id = ids.ctypes.data
            keep.append(ids)
        if out is None:
            out = self.alloc_host_outputs(photon_capacity, want_weight)
        o = Outputs()
        o.size = C.sizeof(Outputs)
        o.hist = out["hist"].ctypes.data if out["hist"].size else None
        o.tel_counts = out["tel_counts"].ctypes.data if out["tel_counts"].size else None
        o.photons = out["photons"].ctypes.data if len(out["photons"]) else None
        o.photon_weight = out["photon_weight"].ctypes.data if out.get("photon_weight") is not None and len(out["photon_weight"]) else None
        o.photon_capacity = len(out["photons"])
        o.counters = out["counters_raw"].ctypes.data
        p, keep2 = self._params(par)
        self._check(self.lib.c8ph_emit_propagate_host(self._h, C.byref(s), int(n_segments), int(seg_id_base),
                                                      C.byref(p), C.c_uint64(int(seed)), C.byref(o)))
        del keep, keep2
        cnt = out["counters_raw"]
        res = dict(out)
        res["counters"] = {k: int(v) for k, v in zip(COUNTER_NAMES, cnt)}
        n = min(res["counters"]["written"], len(out["photons"]))
        res["photons"] = out["photons"][:n]
        if res.get("photon_weight") is not None:
            res["photon_weight"] = out["photon_weight"][:n]
        return res

    def alloc_host_outputs(self, photon_capacity: int = 0, want_weight: bool = False) -> dict:
        return dict(hist=np.zeros(self.n_hist(), dtype=np.float32),
                    tel_counts=np.zeros(self._n_tel, dtype=np.float32),
                    photons=np.zeros(int(photon_capacity), dtype=PHOTON_DTYPE),
                    photon_weight=np.zeros(int(photon_capacity), dtype=np.float32) if want_weight else None,
                    counters_raw=np.zeros(N_COUNTERS, dtype=np.uint64))

    # ---- sub-stepping (the step before the hot path) ---------------------------------------------
    def substep_tracks(self, trk_dev: dict, n_tracks: int, B_tesla, tol_m: float, max_sub: int = 4096, stream=None,
                       ms_max_step_m=None, ms_X0_gcm2: float = 36.62, seed: int = 1, track_id_base: int = 0):
        """trk_dev: dict of torch CUDA float32 tensors x,y,z,dx,dy,dz,len,beta,t0,charge,p_GeV.
        Returns (segments dict of torch CUDA tensors incl. edep = 0, offsets int64[n+1] CUDA tensor).
        ms_max_step_m is not None: multiple-scattering pieces (0 = no cap on the piece length).
        c8ph_substep_plan -> read offsets[n] (one 8-byte D2H) -> allocate -> c8ph_substep_fill."""
        import torch
        dev = trk_dev["x"].device
        t = Segments()
        t.size = C.sizeof(Segments)
        for k in SEG_FIELDS:
            v = trk_dev.get(k)
            setattr(t, k, _dev_ptr(v, "float32", n_tracks) if (v is not None and k != "edep") else None)
        p = _dev_ptr(trk_dev["p_GeV"], "float32", n_tracks)
        d = SubstepDesc()
        d.size = C.sizeof(SubstepDesc)
        d.B_tesla = (C.c_float * 3)(*[float(b) for b in B_tesla])
        d.tol_m, d.max_sub = float(tol_m), int(max_sub)
        d.ms_enabled = 0 if ms_max_step_m is None else 1
        d.ms_max_step_m = 0.0 if ms_max_step_m is None else float(ms_max_step_m)
        d.ms_X0_gcm2, d.seed, d.track_id_base = float(ms_X0_gcm2), int(seed), int(track_id_base)
        offsets = torch.zeros(n_tracks + 1, dtype=torch.int64, device=dev)
        clipped = torch.zeros(1, dtype=torch.int64, device=dev)          # tracks clipped to max_sub pieces (read via .clipped_tracks)
        d.clipped = clipped.data_ptr()
        self.clipped_tracks = clipped
        self._check(self.lib.c8ph_substep_plan(self._h, C.byref(t), p, int(n_tracks), C.byref(d),
                                               offsets.data_ptr(), _stream_ptr(stream)))
        total = int(offsets[-1].item())
        seg = {k: torch.empty(max(total, 1), dtype=torch.float32, device=dev) for k in SEG_FIELDS}
        o = SegmentsOut()
        o.size = C.sizeof(SegmentsOut)
        for k in SEG_FIELDS:
            setattr(o, k, seg[k].data_ptr())
        self._check(self.lib.c8ph_substep_fill(self._h, C.byref(t), p, int(n_tracks), C.byref(d),
                                               offsets.data_ptr(), C.byref(o), _stream_ptr(stream)))
        return {k: v[:total] for k, v in seg.items()}, offsets

    def last_kernel_ms(self) -> float:
        return float(self.lib.c8ph_last_kernel_ms(self._h))

    def launch_count(self) -> int:
        return int(self.lib.c8ph_launch_count(self._h))


def _stream_ptr(stream):
    if stream is None:
        import torch
        return C.c_void_p(torch.cuda.current_stream().cuda_stream)
    if hasattr(stream, "cuda_stream"):
        return C.c_void_p(stream.cuda_stream)
    return C.c_void_p(int(stream))


def _dev_ptr(t, dtype, min_elems):
    if t is None:
        return None
    assert t.is_cuda and t.is_contiguous(), "device tensors must be contiguous CUDA tensors"
    if dtype is not None:
        assert str(t.dtype) == "torch." + dtype, (t.dtype, dtype)
        assert t.numel() >= min_elems, (t.numel(), min_elems)
    return t.data_ptr()


def substep_plan_static(trk_dev: dict, n_tracks: int, B_tesla, tol_m: float, offsets, max_sub: int = 4096, stream=None,
                        ms_max_step_m=None, clipped=None) -> None:
    """c8ph_substep_plan_static: the piece-count scan without a context and without any allocation (scratch = a
    static device array inside the library, at most SUBSTEP_STATIC_MAX_TRACKS tracks).  trk_dev as in
    Context.substep_tracks; offsets: caller's int64[n_tracks + 1] CUDA tensor (written); clipped: optional int64[1]
    CUDA tensor (incremented).  Runs on the current device and stream; argument marshalling only."""
    lib = load_library()
    need = n_tracks if n_tracks <= SUBSTEP_STATIC_MAX_TRACKS else 0     # beyond the limit the library refuses: no size check here
    t = Segments()
    t.size = C.sizeof(Segments)
    for k in SEG_FIELDS:
        v = trk_dev.get(k)
        setattr(t, k, _dev_ptr(v, "float32", need) if (v is not None and k != "edep") else None)
    d = SubstepDesc()
    d.size = C.sizeof(SubstepDesc)
    d.B_tesla = (C.c_float * 3)(*[float(b) for b in B_tesla])
    d.tol_m, d.max_sub = float(tol_m), int(max_sub)
    d.ms_enabled = 0 if ms_max_step_m is None else 1
    d.ms_max_step_m = 0.0 if ms_max_step_m is None else float(ms_max_step_m)
    d.ms_X0_gcm2, d.seed, d.track_id_base = 36.62, 1, 0
    d.clipped = clipped.data_ptr() if clipped is not None else None
    rc = lib.c8ph_substep_plan_static(C.byref(t), _dev_ptr(trk_dev.get("p_GeV"), "float32", need), int(n_tracks), C.byref(d),
                                      _dev_ptr(offsets, "int64", need + 1), _stream_ptr(stream))
    if rc:
        raise C8phError(rc, lib.c8ph_substep_plan_static_error().decode())


# ---- convenience: run a whole workload dict on the device -----------------------------------------
def setup_context(cfg: dict, device: int = 0, ctx: Optional[Context] = None) -> Context:
    """create -> init_atmosphere -> set_detector -> build_trace_table for a workloads.make_config dict."""
    ctx = ctx or Context(device)
    ctx.init_atmosphere(cfg["atmosphere"])
    ctx.set_detector(cfg["detector"])
    if cfg.get("table") is not None:
        ctx.build_trace_table(cfg["table"])
    return ctx


def segments_to_device(seg: dict, device: int = 0) -> dict:
    import torch
    out = {k: torch.from_numpy(_f32(v)).to(f"cuda:{device}") for k, v in seg.items() if k != "id"}
    if seg.get("id") is not None:                                      # explicit global segment ids
        out["id"] = torch.from_numpy(np.ascontiguousarray(seg["id"], dtype=np.uint64).view(np.int64)).to(f"cuda:{device}")
    return out


def alloc_device_outputs(ctx: Context, photon_capacity: int, want_weight: bool = False, device: int = 0) -> dict:
    import torch
    dev = f"cuda:{device}"
    return dict(hist=torch.zeros(max(ctx.n_hist(), 1), dtype=torch.float32, device=dev),
                tel_counts=torch.zeros(max(ctx._n_tel, 1), dtype=torch.float32, device=dev),
                photons=torch.zeros((max(int(photon_capacity), 1), 32), dtype=torch.uint8, device=dev) if photon_capacity else None,
                photon_weight=torch.zeros(max(int(photon_capacity), 1), dtype=torch.float32, device=dev) if (want_weight and photon_capacity) else None,
                counters=torch.zeros(N_COUNTERS, dtype=torch.int64, device=dev))


def outputs_to_host(ctx: Context, out: dict) -> dict:
    """Synchronising copy of device outputs into numpy (tests / examples)."""
    cnt = out["counters"].cpu().numpy().astype(np.uint64)
    res = dict(counters={k: int(v) for k, v in zip(COUNTER_NAMES, cnt)})
    res["hist"] = out["hist"].cpu().numpy()[:ctx.n_hist()]
    res["tel_counts"] = out["tel_counts"].cpu().numpy()[:ctx._n_tel]
    if out.get("photons") is not None:
        n = min(res["counters"]["written"], out["photons"].shape[0])
        res["photons"] = out["photons"][:n].cpu().numpy().view(PHOTON_DTYPE).reshape(-1)
        if out.get("photon_weight") is not None:
            res["photon_weight"] = out["photon_weight"][:n].cpu().numpy()
    else:
        res["photons"] = np.zeros(0, dtype=PHOTON_DTYPE)
    return res


def run_config(cfg: dict, ctx: Optional[Context] = None, photon_capacity: Optional[int] = None,
               want_weight: bool = True, device: int = 0) -> dict:
    """One pass of the whole path over cfg['segments'] with device-resident inputs (tests / smoke)."""
    import torch
    ctx = ctx or setup_context(cfg, device)
    seg = segments_to_device(cfg["segments"], device)
    n = len(cfg["segments"]["x"])
    if photon_capacity is None:
        photon_capacity = 1 << 22
    out = alloc_device_outputs(ctx, photon_capacity, want_weight, device)
    ctx.emit_propagate(seg, n, cfg["seg_id_base"], cfg["params"], cfg["seed"], out)
    torch.cuda.synchronize()
    res = outputs_to_host(ctx, out)
    res["kernel_ms"] = ctx.last_kernel_ms()
    return res
