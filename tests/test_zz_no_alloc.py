"""c8ph_substep_plan_static (include/c8ph.h): the allocation-free variant of the sub-stepping plan - scan scratch in a
static device array inside the library, no context - against the existing path c8ph_substep_plan (context-owned
scratch) and the oracle's piece counts.  The offsets are integers: bit-exact.  Two calls in a row on different inputs
(the scratch keeps the first call's block totals: the second must not see them), then the size limit.
Collected last (file name) so that a failure here cannot hide another test under `pytest -x`."""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu
if not torch.cuda.is_available():                                     # pragma: no cover
    pytest.skip("no CUDA device", allow_module_level=True)

from oracle import c8ph_oracle as O                                    # noqa: E402
from paper_2405_04229_b200 import api, workloads as W                 # noqa: E402


def _tracks(n, seed):
    rng = np.random.default_rng(seed)
    cfg = W.make_config(4, n_segments=n)
    trk = {k: v.copy() for k, v in cfg["segments"].items() if k != "edep"}
    trk["len"] = rng.uniform(0.5, 600.0, n).astype(np.float32)
    trk["p_GeV"] = (10 ** rng.uniform(-2.2, 1.3, n)).astype(np.float32)
    trk["charge"] = rng.choice([-1.0, 1.0, 2.0, 0.0], n).astype(np.float32)
    return cfg, trk


def test_static_plan_matches_the_context_path_on_two_calls_in_a_row():
    B, tol = (2.0e-5, -0.5e-5, -4.3e-5), 0.01
    # first call: several scan blocks and a ragged tail; second call: fewer tracks, other momenta, multiple scattering
    cases = [dict(n=70001, seed=5, max_sub=4096, ms=None), dict(n=2049, seed=6, max_sub=16, ms=10.0)]
    ctx = api.Context()
    for c in cases:
        cfg, trk = _tracks(c["n"], c["seed"])
        dev = {k: torch.from_numpy(v).cuda() for k, v in trk.items()}
        if c["ms"] is not None:
            ctx.init_atmosphere(cfg["atmosphere"])                      # the context path wants it for ms_enabled
        _, want = ctx.substep_tracks(dev, c["n"], B, tol, c["max_sub"], ms_max_step_m=c["ms"])
        want_clipped = int(ctx.clipped_tracks.item())
        got = torch.full((c["n"] + 1,), -7, dtype=torch.int64, device="cuda")
        clipped = torch.zeros(1, dtype=torch.int64, device="cuda")
        api.substep_plan_static(dev, c["n"], B, tol, got, c["max_sub"], ms_max_step_m=c["ms"], clipped=clipped)
        torch.cuda.synchronize()
        assert torch.equal(got, want), c
        assert int(clipped.item()) == want_clipped
        if c["ms"] is None:
            ora = O.substep_tracks(trk, B, tol, c["max_sub"])
        else:
            ora = O.substep_tracks_ms(cfg["atmosphere"], trk, B, tol, c["ms"], max_sub=c["max_sub"])
        assert np.array_equal(got.cpu().numpy(), ora["offsets"])
    assert int(got[-1]) > 2049 and want_clipped > 0
    ctx.close()


def test_static_plan_edges_and_limit():
    _, trk = _tracks(64, 9)
    dev = {k: torch.from_numpy(v).cuda() for k, v in trk.items()}
    off = torch.full((65,), -7, dtype=torch.int64, device="cuda")
    api.substep_plan_static(dev, 0, (0.0, 0.0, 0.0), 0.01, off)          # empty input: offsets[0] = 0, nothing else touched
    torch.cuda.synchronize()
    assert int(off[0]) == 0 and int(off[1]) == -7
    api.substep_plan_static(dev, 64, (0.0, 0.0, 0.0), 0.01, off)         # no field: one piece per track
    torch.cuda.synchronize()
    assert torch.equal(off, torch.arange(65, dtype=torch.int64, device="cuda"))
    # beyond the static scratch: refused with a clear error before anything is launched
    with pytest.raises(api.C8phError) as e:
        api.substep_plan_static(dev, api.SUBSTEP_STATIC_MAX_TRACKS + 1, (0.0, 0.0, 0.0), 0.01, off)
    assert e.value.code == api.E_ARG and "C8PH_SUBSTEP_STATIC_MAX_TRACKS" in str(e.value)
    with pytest.raises(api.C8phError) as e:
        api.substep_plan_static(dev, 64, (0.0, 0.0, 0.0), -1.0, off)
    assert e.value.code == api.E_ARG
    torch.cuda.synchronize()
    assert torch.equal(off, torch.arange(65, dtype=torch.int64, device="cuda"))
