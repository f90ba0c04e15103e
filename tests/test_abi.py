"""The C-ABI boundary (-m "not gpu"): libc8ph.so builds for sm_100a, loads without a GPU, exports
every symbol include/c8ph.h declares, and the Python structs mirror the C layouts.  No compute
calls are made here."""
import ctypes as C
import os
import re
import subprocess

import pytest

from paper_2405_04229_b200 import api, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "c8ph.h")


@pytest.fixture(scope="module")
def lib():
    build.build()
    return api.load_library()


def _declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(c8ph_[a-z_0-9]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lib):
    names = _declared_functions()
    assert len(names) >= 14 and "c8ph_emit_propagate" in names and "c8ph_build_trace_table" in names
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(api.EXPORTS) == names


def test_version_and_counter_names(lib):
    assert lib.c8ph_version() == 200
    got = [lib.c8ph_counter_name(i).decode() for i in range(api.N_COUNTERS)]
    assert tuple(got) == api.COUNTER_NAMES
    assert lib.c8ph_counter_name(api.N_COUNTERS) == b""


def test_struct_layouts_match_the_header(tmp_path):
    """sizeof/offsetof from a C compile of the header against the ctypes mirrors."""
    fields = {
        "c8ph_atmosphere_desc": (api.AtmosphereDesc, ["size", "refractivity", "earth_radius_m", "aer_angstrom", "n_ext_lambda", "ext_tau_v"]),
        "c8ph_table_desc": (api.TableDesc, ["size", "h_max_m", "substeps", "n_rho", "rho_max_m", "n_c"]),
        "c8ph_detector": (api.Detector, ["size", "tel_xyzr", "cam_enabled", "t_ref_ns", "t_bin_ns", "opt_enabled", "opt_camera_radius_m", "opt_kind", "opt_lens_index", "opt_n_abs", "opt_abs"]),
        "c8ph_params": (api.Params, ["size", "write", "bunch_weight", "aim_factor", "disp_lambda0_nm", "use_efficiency", "flat_plane"]),
        "c8ph_segments": (api.Segments, ["size", "x", "edep", "id"]),
        "c8ph_outputs": (api.Outputs, ["size", "hist", "photon_capacity", "counters"]),
        "c8ph_substep_desc": (api.SubstepDesc, ["size", "B_tesla", "tol_m", "ms_enabled", "ms_X0_gcm2", "seed", "track_id_base", "clipped"]),
        "c8ph_segments_out": (api.SegmentsOut, ["size", "x", "edep"]),
    }
    lines = ['#include <stdio.h>', '#include <stddef.h>', f'#include "{HEADER}"', "int main(void){"]
    for s, (_, fs) in fields.items():
        lines.append(f'printf("{s} %zu\\n", sizeof({s}));')
        for f in fs:
            lines.append(f'printf("{s}.{f} %zu\\n", offsetof({s}, {f}));')
    lines.append('printf("c8ph_photon %zu\\n", sizeof(c8ph_photon)); printf("N %d\\n", (int)C8PH_N_COUNTERS); return 0;}')
    src = tmp_path / "layout.c"
    src.write_text("\n".join(lines))
    exe = tmp_path / "layout"
    subprocess.check_call(["gcc", "-std=c99", "-o", str(exe), str(src)])
    out = dict(l.split() for l in subprocess.check_output([str(exe)], text=True).splitlines())
    for s, (cls, fs) in fields.items():
        assert int(out[s]) == C.sizeof(cls), s
        for f in fs:
            assert int(out[f"{s}.{f}"]) == getattr(cls, f).offset, (s, f)
    assert int(out["c8ph_photon"]) == api.PHOTON_DTYPE.itemsize == 32
    assert int(out["N"]) == api.N_COUNTERS


def test_create_fails_loudly_without_a_gpu(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    h = C.c_void_p()
    rc = lib.c8ph_create(C.byref(h), 0)
    assert rc == api.E_CUDA and not h.value
    assert b"no CUDA device" in lib.c8ph_last_error(None)
    with pytest.raises(api.C8phError):
        api.Context(0)


def test_product_does_not_import_the_oracle():
    """The product path must not route through oracle/ (no CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_2405_04229_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "c8ph_oracle" not in txt, f
    otxt = open(os.path.join(ROOT, "oracle", "c8ph_oracle.c")).read()
    assert "#include \"" not in otxt                       # the oracle includes no project header


def test_missing_library_fails_loudly(monkeypatch, tmp_path):
    """No silent fallback: without libc8ph.so the binding raises and names the build step."""
    monkeypatch.setattr(api, "_lib", None)
    monkeypatch.setattr(api, "LIB_PATH", str(tmp_path / "libc8ph.so"))
    with pytest.raises(RuntimeError) as e:
        api.load_library()
    assert "no CPU fallback" in str(e.value) and "build" in str(e.value)
    with pytest.raises(RuntimeError):
        api.Context(0)
