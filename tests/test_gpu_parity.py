"""Parity of the CUDA path (through the C-ABI of libc8ph.so) with the CPU oracle (-m gpu).

Same seeded inputs on both sides; photons are matched by their (segment, j) key and compared
element by element within BASELINE.json's tolerances (tests/c8ph_parity.py).  Sizes are what the oracle
finishes in seconds while still spanning many warps/CTAs and ragged tails; the full-size case of
the benchmark configuration is checked on sampled segment windows plus size-independent
properties.
"""
import copy
import os
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
if not torch.cuda.is_available():                                     # pragma: no cover
    pytest.skip("no CUDA device", allow_module_level=True)

from oracle import c8ph_oracle as O                                    # noqa: E402
from paper_2405_04229_b200 import api, build, workloads as W          # noqa: E402
import c8ph_parity as parity                                           # noqa: E402

build.build()


def _both(cfg, capacity=1 << 22, check_photons=True, ctx=None, max_range_m=None):
    ora = O.run(cfg, record=check_photons)
    gpu = api.run_config(cfg, ctx=ctx, photon_capacity=capacity)
    rep = parity.compare(cfg, ora, gpu, check_photons=check_photons, max_range_m=max_range_m)
    print("parity:", parity.summary(rep))
    return ora, gpu, rep


# ---------------------------------------------------------------------------------- the five configs
def test_cfg0_full_size():
    cfg = W.make_config(0)
    ora, gpu, rep = _both(cfg)
    assert gpu["counters"]["emitted"] > 3.5e5 and gpu["counters"]["written"] == gpu["counters"]["landed"]
    assert rep["max_dpos_m"] < 2e-3                                   # anchor + offset form: sub-mm


def test_cfg1_planar_numeric_weight():
    cfg = W.make_config(1, n_segments=2000)
    ora, gpu, rep = _both(cfg)
    assert gpu["counters"]["landed"] > 1e5
    assert abs(rep["hist_total"][0] - rep["hist_total"][1]) / rep["hist_total"][0] < 1e-5


@pytest.mark.parametrize("zenith_deg", [0.0, 40.0, 64.0, 72.0])
def test_planar_layered_sum_inclined(zenith_deg):
    """Eq. 3.15 per photon at inclined incidence, photon by photon against the oracle's layer loop.  The device sums the
    layers in closed form (layer moments) where (nu_max - nu_min) / (n_e cos z)^2 < 0.02 and layer by
    layer beyond.  With six times the refractivity of air (so that the switch sits at 65 degrees, where the landing
    point is still well conditioned in fp32) 0 / 40 degrees are all closed form, 64 mixes the two inside one warp
    (Cherenkov cone, segment tilts of 2 degrees), 72 is all loop."""
    cfg = W.make_config(1, n_segments=600)
    atm = cfg["atmosphere"]
    atm["refractivity"] = (6.0 * atm["refractivity"].astype(np.float64)).astype(np.float32)
    rng = np.random.default_rng(11)
    cfg["segments"] = W._shower_segments(rng, 600, atm, zenith_deg, 25.0, 330.0, 70.0, 80.0, 2.0, 5.0, 5.0, 2.0, 5.0)
    W._grid(cfg["detector"], 400, 2.5 / math.cos(math.radians(zenith_deg)) ** 2)
    # clock zero = the shower front at the core (arrival times of ~1e6 ns have an fp32 spacing of 0.125 ns in the record)
    s = cfg["segments"]
    front = s["t0"].astype(np.float64) + (s["z"].astype(np.float64) - atm["h_obs"]) / math.cos(math.radians(zenith_deg)) / 0.299792458
    s["t0"] = (s["t0"].astype(np.float64) - np.median(front)).astype(np.float32)
    ora, gpu, rep = _both(cfg)
    assert gpu["counters"]["landed"] > 1e4
    assert abs(rep["hist_total"][0] - rep["hist_total"][1]) / rep["hist_total"][0] < 1e-5


def test_cfg2_spherical_table_filters_roulette():
    cfg = W.make_config(2, n_segments=20000)
    ora, gpu, rep = _both(cfg)
    c = gpu["counters"]
    assert c["seg_lv1"] > 0 and c["lv2"] > 0 and c["roulette"] > 0 and c["tel_hit"] > 5000


def test_cfg3_fluorescence_camera():
    cfg = W.make_config(3, n_segments=20000)
    cfg["segments"]["edep"][:] *= 40.0                                # enough photons for statistics
    ora, gpu, rep = _both(cfg)
    assert gpu["counters"]["cam_hit"] > 300


def test_cfg4_all_features_small():
    cfg = W.make_config(4, n_segments=3000)
    ora, gpu, rep = _both(cfg)
    c = gpu["counters"]
    assert c["in_grid"] > 1e5 and c["tel_hit"] > 1e4 and c["roulette"] > 0


# ---------------------------------------------------------------------------------- the trace table
def test_trace_table_against_oracle_nodes():
    cfg = W.make_config(2, n_segments=4)
    ctx = api.setup_context(cfg)
    got = ctx.get_trace_table()
    want = O.table_for(cfg)
    assert got.shape == want.shape == (512, 256, 5)
    nan_g, nan_w = np.isnan(got[..., 0]), np.isnan(want[..., 0])
    assert (nan_g != nan_w).sum() <= 2 and 0.05 < nan_w.mean() < 0.08
    zen = np.linspace(0.0, 89.0, 256)
    ok = ~(nan_g | nan_w) & (zen[None, :] <= 75.0)
    d = np.abs(got.astype(np.float64) - want.astype(np.float64))
    assert d[..., 0][ok].max() <= 1e-4                                # 0.1 mm
    assert d[..., 2][ok].max() <= 3e-4                                # 0.3 ps
    assert d[..., 3][ok].max() <= 1e-2                                # g/cm^2
    ok_all = ~(nan_g | nan_w)
    rel = d[ok_all] / np.maximum(np.abs(want[ok_all].astype(np.float64)), 1e-3)
    assert rel.max() < 1e-3


def test_injected_oracle_table_gives_same_photons():
    """Isolation: with the oracle's table injected, table-build differences drop out."""
    cfg = W.make_config(2, n_segments=5000)
    ctx = api.Context(0)
    ctx.init_atmosphere(cfg["atmosphere"])
    ctx.set_detector(cfg["detector"])
    ctx.set_trace_table(cfg["table"], O.table_for(cfg))
    _both(cfg, ctx=ctx)


def test_telescope_grids_equal_brute_force_search(monkeypatch):
    """SURVEY O12 pin on the device: the sorted-key uniform grids (hit test, LV2 proximity, per-cell
    accept / reject bounds) give exactly the decisions of a search over all telescopes, on ~3e7 rays
    against the 10,000 spheres of cfg4 and on cfg2's 100-sphere lattice at 60 deg zenith."""
    for k, n in ((4, 80000), (2, 60000)):
        cfg = W.make_config(k, n_segments=n)
        res = {}
        for mode in ("grid", "brute"):
            monkeypatch.setenv("C8PH_FORCE_BRUTE", "1" if mode == "brute" else "0")
            ctx = api.setup_context(cfg)                               # the switch is read at c8ph_create
            res[mode] = api.run_config(cfg, ctx=ctx, photon_capacity=1 << 23)
            ctx.close()
        g, b = res["grid"], res["brute"]
        assert g["counters"] == b["counters"] and g["counters"]["tel_hit"] > 1e4
        assert np.array_equal(g["tel_counts"], b["tel_counts"]) and np.array_equal(g["hist"], b["hist"])
        key = lambda p: np.argsort(p["seg"].astype(np.int64) << 32 | p["j_tel"])
        assert np.array_equal(g["photons"][key(g["photons"])], b["photons"][key(b["photons"])])



def test_irregular_array_varied_radii_and_heights(monkeypatch):
    """Row f1 (non-lattice arrays): 300 telescopes at random positions with radii 2-12 m and centres up
    to 15 m above / below the observation level, the 1 PeV shower of cfg4 at 2 000 segments and the
    inclined one of cfg2 at 20 000.  Against the oracle's brute force, and grid == search-all."""
    rng = np.random.default_rng(4242)
    tel = np.zeros((300, 4), dtype=np.float32)
    tel[:, 0], tel[:, 1] = rng.uniform(-450.0, 450.0, 300), rng.uniform(-450.0, 450.0, 300)
    tel[:, 2], tel[:, 3] = rng.uniform(-15.0, 15.0, 300), rng.uniform(2.0, 12.0, 300)
    for k, n in ((4, 2000), (2, 20000)):
        cfg = W.make_config(k, n_segments=n)
        cfg["detector"]["tel_xyzr"] = tel.copy()
        ora, gpu, rep = _both(cfg)
        assert gpu["counters"]["tel_hit"] > 2000 and gpu["counters"]["lv2"] >= 0
        monkeypatch.setenv("C8PH_FORCE_BRUTE", "1")
        ctx = api.setup_context(cfg)
        brute = api.run_config(cfg, ctx=ctx)
        ctx.close()
        monkeypatch.setenv("C8PH_FORCE_BRUTE", "0")
        assert brute["counters"] == gpu["counters"] and np.array_equal(brute["tel_counts"], gpu["tel_counts"])


# ---------------------------------------------------------------------------------- edge cases
def test_empty_and_tiny_inputs():
    cfg = W.make_config(0, n_segments=1)
    ctx = api.setup_context(cfg)
    seg = api.segments_to_device(cfg["segments"])
    out = api.alloc_device_outputs(ctx, 1024)
    ctx.emit_propagate(seg, 0, 0, cfg["params"], 1, out)
    torch.cuda.synchronize()
    assert int(out["counters"].sum()) == 0
    for n in (1, 31, 33, 257):
        _both(W.make_config(0, n_segments=n), capacity=1 << 18)


def test_random_directions_upgoing_and_subthreshold():
    """Isotropic particle directions (up-going, horizontal: the non-anchor branch) and a beta
    spectrum straddling the Cherenkov threshold."""
    for k, n in ((0, 4000), (2, 6000)):
        cfg = W.make_config(k, n_segments=n)
        rng = np.random.default_rng(77 + k)
        s = cfg["segments"]
        v = rng.normal(size=(n, 3))
        v /= np.linalg.norm(v, axis=1, keepdims=True)
        half = n // 2
        s["dx"][:half], s["dy"][:half], s["dz"][:half] = v[:half, 0], v[:half, 1], v[:half, 2]
        s["dz"][0], s["dx"][0], s["dy"][0] = 1.0, 0.0, 0.0                 # straight up: degenerate bisector
        s["dz"][1], s["dx"][1], s["dy"][1] = -1.0, 0.0, 0.0                # straight down
        s["beta"][::3] = rng.uniform(0.9995, 0.99999, len(s["beta"][::3])).astype(np.float32)
        cfg["params"].update(lv1=False)
        ora, gpu, rep = _both(cfg, max_range_m=20000.0)
        assert gpu["counters"]["upgoing"] > 0 and gpu["counters"]["seg_below_threshold"] > 0
        assert rep["beyond_range"] < 0.5 * gpu["counters"]["written"]


def test_emission_at_or_below_the_observation_level_is_dropped():
    """Reading R7 (t* = -A_z/u_z > 0): segments that start or end at or below the observation level - their photons
    from z <= 0 are dropped and counted with the up-going ones, the rest is propagated as usual; per-photon layered
    sum (cfg1), table (cfg4) and straight line (cfg0) against the oracle."""
    for k, n in ((1, 200), (4, 1200), (0, 600)):
        cfg = W.make_config(k, n_segments=n)
        rng = np.random.default_rng(5)
        s = cfg["segments"]
        s["z"][::5] = rng.uniform(-100.0, 5.0, len(s["z"][::5])).astype(np.float32)
        cfg["params"]["lv1"] = False
        ref = api.run_config(W.make_config(k, n_segments=n))
        ora, gpu, rep = _both(cfg)
        assert gpu["counters"]["upgoing"] > ref["counters"]["upgoing"] + 100


def test_filters_lossless_on_device():
    cfg = W.make_config(2, n_segments=20000)
    on = api.run_config(cfg)
    off_cfg = copy.deepcopy(cfg)
    off_cfg["params"].update(lv1=False, lv2=False)
    off = api.run_config(off_cfg)
    assert on["counters"]["tel_hit"] == off["counters"]["tel_hit"]
    assert np.array_equal(on["tel_counts"], off["tel_counts"])
    key = lambda p: np.sort(p["seg"].astype(np.int64) << 32 | p["j_tel"])
    assert np.array_equal(key(on["photons"]), key(off["photons"]))


def test_batching_and_grid_independence():
    """Results depend on (seed, seg_id_base + i, j) only: two half calls == one call, bit for bit."""
    cfg = W.make_config(4, n_segments=2000)
    ctx = api.setup_context(cfg)
    full = api.run_config(cfg, ctx=ctx)
    seg = api.segments_to_device(cfg["segments"])
    out = api.alloc_device_outputs(ctx, 1 << 22, True)
    cut = 777
    a = {k: v[:cut].contiguous() for k, v in seg.items()}
    b = {k: v[cut:].contiguous() for k, v in seg.items()}
    ctx.emit_propagate(a, cut, 0, cfg["params"], cfg["seed"], out)
    ctx.emit_propagate(b, 2000 - cut, cut, cfg["params"], cfg["seed"], out)
    torch.cuda.synchronize()
    two = api.outputs_to_host(ctx, out)
    assert two["counters"] == {**full["counters"], "segments": 2000}
    assert np.array_equal(two["hist"], full["hist"]) and np.array_equal(two["tel_counts"], full["tel_counts"])
    pa, pb = full["photons"].copy(), two["photons"].copy()
    # records of the second call carry call-local segment indices; the calls ran back to back on
    # one stream, so the second call's records are the tail of the list: shift them back
    n_first = int((full["photons"]["seg"] < cut).sum())
    pb_seg = pb["seg"].astype(np.int64)
    pb_seg[n_first:] += cut
    ka = np.sort(pa["seg"].astype(np.int64) << 32 | pa["j_tel"])
    kb = np.sort(pb_seg << 32 | pb["j_tel"])
    assert np.array_equal(ka, kb)
    oa, ob = np.argsort(pa["seg"].astype(np.int64) << 32 | pa["j_tel"]), np.argsort(pb_seg << 32 | pb["j_tel"])
    for f in ("x", "y", "ux", "uy", "t_ns", "lambda_nm"):
        assert np.array_equal(pa[f][oa], pb[f][ob]), f


def test_photon_buffer_overflow_is_counted_not_silent():
    cfg = W.make_config(0, n_segments=200)
    ctx = api.setup_context(cfg)
    ref = api.run_config(cfg, ctx=ctx)
    small = api.run_config(cfg, ctx=ctx, photon_capacity=1000)
    c = small["counters"]
    assert c["written"] == ref["counters"]["written"] and c["overflow"] == c["written"] - 1000
    assert len(small["photons"]) == 1000
    assert np.array_equal(small["hist"], ref["hist"])                 # overflowing photons are still binned


def test_bunch_count_cap_per_segment_is_counted_not_silent():
    """Maximum size of one segment (R1): the record key holds 18 bits of photon index, so a segment emits at
    most C8PH_MAX_BUNCHES_PER_SEGMENT - 1 = 262143 bunches; a segment asking for more (charge 30: 293365) is clipped,
    counted in `clipped`, and the photons it does emit are the oracle's photons of the same indices."""
    cfg = W.make_config(0, n_segments=3)
    cfg["segments"]["charge"][1] = 30.0
    ora = O.run(cfg)
    assert ora["n_bunch"][1] > 262143 > ora["n_bunch"][0]
    gpu = api.run_config(cfg, photon_capacity=1 << 19)
    c = gpu["counters"]
    cap = 262143
    assert c["clipped"] == 1 and c["overflow"] == 0
    assert c["emitted"] == ora["n_bunch"][0] + cap + ora["n_bunch"][2] == c["written"]
    g = gpu["photons"]
    j = (g["j_tel"] >> 14).astype(np.int64)
    mid = g["seg"] == 1
    assert mid.sum() == cap and np.array_equal(np.sort(j[mid]), np.arange(cap))
    o = ora["photons"]
    o = o[(o["seg"] == 1) & (o["j"] < cap)]
    o = o[np.argsort(o["j"])]
    gm = g[mid][np.argsort(j[mid])]
    assert np.abs(gm["x"] - o["x"]).max() < 0.05 and np.abs(gm["y"] - o["y"]).max() < 0.05
    assert np.allclose(gm["lambda_nm"], o["lambda_nm"], rtol=2e-6)


def test_host_buffer_entry_point_matches_device_path():
    cfg = W.make_config(4, n_segments=1500)
    ctx = api.setup_context(cfg)
    dev = api.run_config(cfg, ctx=ctx)
    host = ctx.emit_propagate_host(cfg["segments"], 1500, 0, cfg["params"], cfg["seed"],
                                   photon_capacity=1 << 20, want_weight=True)
    assert host["counters"] == dev["counters"]
    assert np.array_equal(host["hist"], dev["hist"]) and np.array_equal(host["tel_counts"], dev["tel_counts"])
    k = lambda p: np.argsort(p["seg"].astype(np.int64) << 32 | p["j_tel"])
    assert np.array_equal(host["photons"][k(host["photons"])], dev["photons"][k(dev["photons"])])


def test_argument_errors_are_reported():
    cfg = W.make_config(2, n_segments=8)
    ctx = api.Context(0)
    seg = api.segments_to_device(cfg["segments"])
    with pytest.raises(api.C8phError) as e:
        ctx.set_detector(cfg["detector"])
        out = api.alloc_device_outputs(ctx, 16)
        ctx.emit_propagate(seg, 8, 0, cfg["params"], 1, out)
    assert e.value.code == api.E_STATE
    ctx.init_atmosphere(cfg["atmosphere"])
    with pytest.raises(api.C8phError) as e:
        ctx.emit_propagate(seg, 8, 0, cfg["params"], 1, out)          # table not built
    assert e.value.code == api.E_STATE
    bad = dict(cfg["params"], bunch_weight=0.0)
    ctx.build_trace_table(cfg["table"])
    with pytest.raises(api.C8phError) as e:
        ctx.emit_propagate(seg, 8, 0, bad, 1, out)
    assert e.value.code == api.E_ARG


# ---------------------------------------------------------------------------------- full size
def test_cfg4_full_size_sampled_windows_and_invariants():
    """BASELINE configs[4] at its full 1e7 segments in the launch configuration bench.py times
    (device-resident inputs, WRITE_TEL photon list).  The oracle cannot run 3.4e9 photons, so:
    photons of sampled segment windows are compared one by one with the oracle run on the same
    windows (valid because every photon depends only on (seed, segment id, j)), and the whole
    output is checked through identities that hold at any size."""
    n = W.FULL_SEGMENTS[4]
    cfg = W.make_config(4)
    ctx = api.setup_context(cfg)
    seg = api.segments_to_device(cfg["segments"])
    cap = 220_000_000
    out = api.alloc_device_outputs(ctx, cap, False)
    ctx.emit_propagate(seg, n, 0, cfg["params"], cfg["seed"], out)
    torch.cuda.synchronize()
    cnt = {k: int(v) for k, v in zip(api.COUNTER_NAMES, out["counters"].cpu().numpy())}
    assert cnt["segments"] == n and cnt["overflow"] == 0 and cnt["clipped"] == 0
    assert cnt["emitted"] == cnt["upgoing"] + cnt["lv2"] + cnt["table_range"] + cnt["roulette"] + cnt["landed"]
    assert cnt["emitted"] > 2e9
    hist = out["hist"]
    assert float(hist.max()) < 2 ** 24                                # fp32 counts stay exact
    assert int(hist.double().sum().item()) == cnt["in_grid"]
    assert int(out["tel_counts"].double().sum().item()) == cnt["tel_hit"] == cnt["written"]
    # sampled windows: first, a ragged middle one, last
    ph_seg = out["photons"][:cnt["written"]].view(torch.int32)[:, 6]
    for lo, hi in ((0, 400), (4_999_777, 5_000_190), (n - 300, n)):
        m = (ph_seg >= lo) & (ph_seg < hi)
        rec = out["photons"][:cnt["written"]][m].cpu().numpy().view(api.PHOTON_DTYPE).reshape(-1).copy()
        rec["seg"] -= lo
        sub = copy.deepcopy(cfg)
        sub["segments"] = W.slice_segments(cfg["segments"], lo, hi)
        sub["seg_id_base"] = lo
        ora = O.run(sub)
        want = ora["photons"][(ora["photons"]["status"] == O.ST_LANDED) & (ora["photons"]["tel"] >= 0)]
        gk = np.sort(rec["seg"].astype(np.int64) << 18 | (rec["j_tel"] >> 14))
        ok = np.sort(want["seg"].astype(np.int64) << 18 | want["j"])
        common = np.intersect1d(gk, ok)
        budget = max(3, int(math.ceil(1e-4 * ora["counters"]["emitted"])))
        assert len(gk) + len(ok) - 2 * len(common) <= budget
        # element-by-element on the window via the standard comparison of a window-only device run
        win = api.run_config(sub, ctx=ctx)
        print(f"window [{lo}, {hi}):", parity.summary(parity.compare(sub, ora, win)))
        k2 = np.argsort(win["photons"]["seg"].astype(np.int64) << 32 | win["photons"]["j_tel"])
        k1 = np.argsort(rec["seg"].astype(np.int64) << 32 | rec["j_tel"])
        assert np.array_equal(rec[k1], win["photons"][k2])            # full-size run == window run, bit for bit


def test_cfg4_first_1e5_segments_whole_histogram_and_every_telescope_counter():
    """SURVEY 8(d) / BASELINE.md section 3: the first 1e5 segment ids of configs[4] (3.4e7 photons, about a minute of
    oracle time on the box's cores) compared as a whole: the 1000 x 1000 ground histogram bin by bin (the hot core
    bins hold hundreds of photons), all 10 000 telescope counters and every event counter."""
    n = 100_000
    cfg = W.make_config(4, n_segments=n)
    ora = O.run(cfg, record=False)
    gpu = api.run_config(cfg, photon_capacity=1 << 22)
    rep = parity.compare(cfg, ora, gpu, check_photons=False)
    print("parity (1e5 segments):", parity.summary(rep), "counters (oracle, device):",
          {k: rep[k] for k in ("emitted", "landed", "in_grid", "tel_hit", "roulette", "lv2")})
    ho, hg = ora["hist"], gpu["hist"].astype(np.float64)
    assert ho.max() > 300 and rep["hist_total_rel"] <= 1e-5
    assert np.abs(ho - hg).max() <= 3                                 # no bin off by more than a few flips
    to, tg = ora["tel_counts"], gpu["tel_counts"].astype(np.float64)
    assert (to > 0).sum() > 2000 and np.abs(to - tg).max() <= 3
    assert abs(tg.sum() - to.sum()) <= max(3, 1e-5 * to.sum())


def test_cfg1_full_size_sampled_windows_and_invariants():
    """BASELINE configs[1] at its full 1e5 segments (planar atmosphere, per-photon layered sum, weight mode,
    every photon written: 8.1e6 records): whole-run identities plus photon-by-photon comparison with the
    oracle on sampled segment windows."""
    n = W.FULL_SEGMENTS[1]
    cfg = W.make_config(1)
    ctx = api.setup_context(cfg)
    seg = api.segments_to_device(cfg["segments"])
    out = api.alloc_device_outputs(ctx, 12_000_000, True)
    ctx.emit_propagate(seg, n, 0, cfg["params"], cfg["seed"], out)
    torch.cuda.synchronize()
    cnt = {k: int(v) for k, v in zip(api.COUNTER_NAMES, out["counters"].cpu().numpy())}
    assert cnt["segments"] == n and cnt["overflow"] == 0 and cnt["clipped"] == 0
    assert cnt["emitted"] == cnt["upgoing"] + cnt["lv2"] + cnt["table_range"] + cnt["roulette"] + cnt["landed"]
    assert cnt["emitted"] > 5e6 and cnt["written"] == cnt["landed"] and cnt["roulette"] == 0
    wsum = out["photon_weight"][:cnt["written"]].double().sum().item()
    assert 0.0 < out["hist"].double().sum().item() <= wsum * (1 + 1e-6)       # the grid holds part of the landed weight
    rec_all = out["photons"][:cnt["written"]]
    ph_seg = rec_all.view(torch.int32)[:, 6]
    for lo, hi in ((0, 600), (50_017, 50_640), (n - 500, n)):
        m = (ph_seg >= lo) & (ph_seg < hi)
        rec = rec_all[m].cpu().numpy().view(api.PHOTON_DTYPE).reshape(-1).copy()
        rec["seg"] -= lo
        sub = copy.deepcopy(cfg)
        sub["segments"] = W.slice_segments(cfg["segments"], lo, hi)
        sub["seg_id_base"] = lo
        ora = O.run(sub)
        win = api.run_config(sub, ctx=ctx)
        print(f"window [{lo}, {hi}):", parity.summary(parity.compare(sub, ora, win)))
        k2 = np.argsort(win["photons"]["seg"].astype(np.int64) << 32 | win["photons"]["j_tel"])
        k1 = np.argsort(rec["seg"].astype(np.int64) << 32 | rec["j_tel"])
        assert len(rec) > 2e4 and np.array_equal(rec[k1], win["photons"][k2])   # full-size run == window run, bit for bit


def test_cfg3_full_size_against_the_whole_oracle():
    """BASELINE configs[3] at its full 1e6 segments (forced-cone fluorescence: ~1.7e5 photons, which
    the oracle runs completely): counters, camera histogram and every photon record."""
    cfg = W.make_config(3)
    assert len(cfg["segments"]["x"]) == W.FULL_SEGMENTS[3]
    ora, gpu, rep = _both(cfg, capacity=1 << 20)
    assert gpu["counters"]["segments"] == 1_000_000 and gpu["counters"]["emitted"] > 1e5
    assert gpu["counters"]["cam_hit"] > 1000


def test_cfg2_full_size_sampled_windows_and_invariants():
    """BASELINE configs[2] at its full 1e6 segments (1.4e8 bunches of weight 5 after LV1): whole-run
    identities plus photon-by-photon comparison with the oracle on sampled segment windows."""
    n = W.FULL_SEGMENTS[2]
    cfg = W.make_config(2)
    ctx = api.setup_context(cfg)
    seg = api.segments_to_device(cfg["segments"])
    out = api.alloc_device_outputs(ctx, 4_000_000, False)
    ctx.emit_propagate(seg, n, 0, cfg["params"], cfg["seed"], out)
    torch.cuda.synchronize()
    cnt = {k: int(v) for k, v in zip(api.COUNTER_NAMES, out["counters"].cpu().numpy())}
    assert cnt["segments"] == n and cnt["overflow"] == 0 and cnt["clipped"] == 0
    assert cnt["segments"] >= cnt["seg_below_threshold"] + cnt["seg_lv1"] + cnt["seg_emitting"]
    assert cnt["emitted"] == cnt["upgoing"] + cnt["lv2"] + cnt["table_range"] + cnt["roulette"] + cnt["landed"]
    assert cnt["seg_lv1"] > 0.2 * n and cnt["lv2"] > 0.5 * cnt["emitted"] and cnt["emitted"] > 1e8
    w = float(cfg["params"]["bunch_weight"])
    assert int(round(out["tel_counts"].double().sum().item() / w)) == cnt["tel_hit"] == cnt["written"]
    rec_all = out["photons"][:cnt["written"]]
    ph_seg = rec_all.view(torch.int32)[:, 6]
    for lo, hi in ((0, 3000), (500_123, 504_000), (n - 2500, n)):
        m = (ph_seg >= lo) & (ph_seg < hi)
        rec = rec_all[m].cpu().numpy().view(api.PHOTON_DTYPE).reshape(-1).copy()
        rec["seg"] -= lo
        sub = copy.deepcopy(cfg)
        sub["segments"] = W.slice_segments(cfg["segments"], lo, hi)
        sub["seg_id_base"] = lo
        ora = O.run(sub)
        win = api.run_config(sub, ctx=ctx)
        print(f"window [{lo}, {hi}):", parity.summary(parity.compare(sub, ora, win)))
        k2 = np.argsort(win["photons"]["seg"].astype(np.int64) << 32 | win["photons"]["j_tel"])
        k1 = np.argsort(rec["seg"].astype(np.int64) << 32 | rec["j_tel"])
        assert np.array_equal(rec[k1], win["photons"][k2])            # full-size run == window run, bit for bit


def _thesis_array(golden_dir, name):
    return np.loadtxt(os.path.join(golden_dir, name), comments="#", dtype=np.float32).reshape(-1, 4)


@pytest.mark.parametrize("name,n_tel", [("telescope_array_1.txt", 13), ("telescope_array_2.txt", 180)])
def test_thesis_model_arrays(golden_dir, monkeypatch, name, n_tel):
    """Row f1: the thesis' own model arrays (Appendix B.3; fixtures parsed from PAPER.md by
    tests/golden/make_telescope_arrays.py): 13 telescopes of radius 12 / 23 m and 180 of radius
    2.1 / 5.8 / 11.1 m, centres 5-75 m above the observation level, non-lattice.  cfg4's shower
    (vertical-ish) and cfg2's (60 deg zenith) against the oracle's brute force, and grid == search-all."""
    tel = _thesis_array(golden_dir, name)
    assert tel.shape == (n_tel, 4)
    for k, n in ((4, 3000), (2, 30000)):
        cfg = W.make_config(k, n_segments=n)
        cfg["detector"]["tel_xyzr"] = tel.copy()
        ora, gpu, rep = _both(cfg)
        assert gpu["counters"]["tel_hit"] > 500
        monkeypatch.setenv("C8PH_FORCE_BRUTE", "1")
        ctx = api.setup_context(cfg)
        brute = api.run_config(cfg, ctx=ctx)
        ctx.close()
        monkeypatch.setenv("C8PH_FORCE_BRUTE", "0")
        assert brute["counters"] == gpu["counters"] and np.array_equal(brute["tel_counts"], gpu["tel_counts"])


def test_emit_propagate_is_stream_ordered_and_graph_capturable():
    """The hot call enqueues only (no allocation, no host sync, no bulk copy): it can run on a side
    stream and be captured into a CUDA graph; replays give the bits of the eager call."""
    cfg = W.make_config(4, n_segments=1200)
    ctx = api.setup_context(cfg)
    eager = api.run_config(cfg, ctx=ctx)
    seg = api.segments_to_device(cfg["segments"])
    out = api.alloc_device_outputs(ctx, 1 << 20, True)
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        ctx.emit_propagate(seg, 1200, 0, cfg["params"], cfg["seed"], out, stream=side)     # warm-up on the side stream
    side.synchronize()
    first = api.outputs_to_host(ctx, out)
    assert first["counters"] == eager["counters"] and np.array_equal(first["hist"], eager["hist"])
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=side):
        for k in ("hist", "tel_counts", "counters"):
            out[k].zero_()
        ctx.emit_propagate(seg, 1200, 0, cfg["params"], cfg["seed"], out, stream=torch.cuda.current_stream())
    for _ in range(3):
        g.replay()
    torch.cuda.synchronize()
    rep = api.outputs_to_host(ctx, out)
    assert rep["counters"] == eager["counters"]
    assert np.array_equal(rep["hist"], eager["hist"]) and np.array_equal(rep["tel_counts"], eager["tel_counts"])
    key = lambda p: np.argsort(p["seg"].astype(np.int64) << 32 | p["j_tel"])
    assert np.array_equal(rep["photons"][key(rep["photons"])], eager["photons"][key(eager["photons"])])


def test_dispersion_yield_spectrum_and_cone():
    """Row f4: n(lambda, h) = 1 + eta(h) D(lambda) (thesis P:314-322).  Device against oracle, photon
    by photon: (a) cfg0 with particles whose Cherenkov threshold lies inside the band (only the blue
    part emits, strongly non-uniform spectrum, rejection sampling takes several trials); (b) cfg4's
    full feature set with dispersion on (generic kernel variant); (c) the layered-sum variant."""
    eta, b, l0 = 0.000293, 5700.0, 400.0
    cfg = W.make_config(0, n_segments=600)
    cfg["params"].update(disp_b_nm2=b, disp_lambda0_nm=l0)
    k_th = 1.0 / np.linspace(280.0, 640.0, 600)                        # threshold wavelength: below, inside, beyond the band
    cfg["segments"]["beta"][:] = (1.0 / (1.0 + eta * (1.0 + b * (k_th ** 2 - 1 / l0 ** 2)))).astype(np.float32)
    cfg["segments"]["len"][:] = 60.0
    ora, gpu, rep = _both(cfg)
    assert gpu["counters"]["emitted"] > 1e4 and gpu["counters"]["seg_below_threshold"] > 10
    lam = gpu["photons"]["lambda_nm"]
    assert lam.min() >= 300.0 and lam.max() <= 600.0 and np.median(lam) < 400.0
    plain = api.run_config(W.make_config(0, n_segments=600))
    assert plain["counters"]["emitted"] != gpu["counters"]["emitted"]
    for k, n in ((4, 2500), (1, 600)):
        cfg = W.make_config(k, n_segments=n)
        cfg["params"].update(disp_b_nm2=b, disp_lambda0_nm=l0)
        ora, gpu, rep = _both(cfg)
        off = api.run_config(W.make_config(k, n_segments=n))
        assert gpu["counters"]["emitted"] > off["counters"]["emitted"]      # blue end sees a larger n
    bad = dict(cfg["params"], disp_b_nm2=-1.0)
    ctx = api.setup_context(cfg)
    with pytest.raises(api.C8phError) as e:
        api.run_config(dict(cfg, params=bad), ctx=ctx)
    assert e.value.code == api.E_ARG


def test_detector_efficiency_folding():
    """Row f4: eps(lambda) folded into the survival probability (roulette: cfg2, cfg4) or the weight
    (cfg1), device against oracle photon by photon; a bell-shaped curve on a 10 nm grid."""
    lam = np.arange(200.0, 801.0, 10.0)
    eff = (0.85 * np.exp(-0.5 * ((lam - 420.0) / 90.0) ** 2)).astype(np.float32)
    for k, n in ((2, 20000), (4, 2500), (1, 600)):
        cfg = W.make_config(k, n_segments=n)
        cfg["params"].update(eff=eff, eff_lambda0_nm=200.0, eff_dlambda_nm=10.0)
        ora, gpu, rep = _both(cfg)
        off = api.run_config(W.make_config(k, n_segments=n))
        if k == 1:
            assert gpu["counters"]["landed"] == off["counters"]["landed"] and gpu["hist"].sum() < 0.8 * off["hist"].sum()
        else:
            assert 0.2 * off["counters"]["landed"] < gpu["counters"]["landed"] < 0.8 * off["counters"]["landed"]
    cfg = W.make_config(0, n_segments=50)                                  # transmission off: the table is refused
    cfg["params"].update(eff=eff, eff_lambda0_nm=200.0, eff_dlambda_nm=10.0)
    with pytest.raises(api.C8phError) as e:
        api.run_config(cfg)
    assert e.value.code == api.E_ARG


def test_last_mile_optics():
    """Row f3 (thesis sec. 6.4): parabolic mirror + shadowing camera inside the bounding spheres, fused
    after the sphere test so that only camera hits are written.  The MAGIC-like telescope of the thesis
    (17 m parabola, f = 17 m, 1.47 m camera) on cfg4's lattice and on cfg2's inclined shower with the
    telescopes pointed at the shower; records are camera-plane points, compared photon by photon."""
    for k, n, az, el in ((4, 4000, 0.0, 70.0), (2, 40000, 30.0, 30.0)):
        cfg = W.make_config(k, n_segments=n)
        tel = cfg["detector"]["tel_xyzr"].copy()
        tel[:, 3] = 12.0
        cfg["detector"]["tel_xyzr"] = tel
        base = api.run_config(cfg)
        cfg["detector"].update(opt_enabled=True, opt_az_deg=az, opt_el_deg=el, opt_focal_m=17.0,
                               opt_mirror_radius_m=8.5, opt_camera_radius_m=0.735)
        ora, gpu, rep = _both(cfg)
        c = gpu["counters"]
        assert c["tel_hit"] == base["counters"]["tel_hit"] and 50 < c["cam_hit"] == c["written"] < c["tel_hit"]
        ph = gpu["photons"]
        assert np.all(np.hypot(ph["x"], ph["y"]) <= 0.735 * (1 + 1e-5))
        assert rep["max_dpos_m"] < 2e-3                                    # camera-plane agreement: mm
    cfg["detector"]["tel_xyzr"][:, 3] = 6.0                                # sphere too small for the optics
    with pytest.raises(api.C8phError) as e:
        api.setup_context(cfg)
    assert e.value.code == api.E_ARG


def test_last_mile_truss_shadowing_and_refracting_lens():
    """Row f3, the rest of thesis sec. 6.4 (R22): absorbing objects (a four-mast truss and a
    cross strut on the MAGIC-like telescope) and light bending at a boundary layer (a plano-convex lens telescope with
    the camera in its back focal plane; rays that are totally reflected inside the glass are lost).  Device against
    oracle photon by photon; the truss removes light, the lens images the shower onto its camera."""
    # --- truss on the mirror telescope of test_last_mile_optics
    cfg = W.make_config(4, n_segments=4000)
    cfg["detector"]["tel_xyzr"][:, 3] = 12.0
    cfg["detector"].update(opt_enabled=True, opt_az_deg=0.0, opt_el_deg=70.0, opt_focal_m=17.0,
                           opt_mirror_radius_m=8.5, opt_camera_radius_m=0.735)
    clear = api.run_config(cfg)
    masts = [[6.0 * np.cos(a), 6.0 * np.sin(a), -8.5 + 36.0 / 68.0, 0.6 * np.cos(a), 0.6 * np.sin(a), 8.5, 0.08]
             for a in np.radians([45.0, 135.0, 225.0, 315.0])]               # mirror surface (rho = 6 m) to the camera rim
    masts.append([-8.0, 0.0, 2.0, 8.0, 0.0, 2.0, 0.05])                      # a cross strut
    cfg["detector"]["opt_absorbers"] = np.array(masts, np.float32)
    ora, gpu, rep = _both(cfg)
    c = gpu["counters"]
    assert c["tel_hit"] == clear["counters"]["tel_hit"]
    assert 0.85 * clear["counters"]["cam_hit"] < c["cam_hit"] < 0.99 * clear["counters"]["cam_hit"]     # a few per cent shadowed
    assert rep["max_dpos_m"] < 2e-3
    # --- lens telescope: R = 12 m, n = 1.5, thickness 1.2 m, aperture 5 m, camera in the back focal plane
    R_l, n_l, t_l = 12.0, 1.5, 1.2
    bfd = R_l / (n_l - 1.0) - t_l / n_l
    cfg = W.make_config(4, n_segments=4000)
    cfg["detector"]["tel_xyzr"][:, 3] = 14.0
    cfg["detector"].update(opt_enabled=True, opt_az_deg=0.0, opt_el_deg=70.0, opt_focal_m=bfd, opt_mirror_radius_m=5.0,
                           opt_camera_radius_m=1.5, opt_kind=1, opt_lens_roc_m=R_l, opt_lens_thickness_m=t_l, opt_lens_index=n_l,
                           opt_absorbers=np.array([[-5.0, 0.0, -3.0, 5.0, 0.0, -3.0, 0.05]], np.float32))
    ora, gpu, rep = _both(cfg)
    c = gpu["counters"]
    assert 200 < c["cam_hit"] == c["written"] < c["tel_hit"]
    ph = gpu["photons"]
    assert np.all(np.hypot(ph["x"], ph["y"]) <= 1.5 * (1 + 1e-5)) and rep["max_dpos_m"] < 2e-3
    # the image of the 20-degree-inclined light sits f tan(20 deg) ~ 8 m off axis for an axis at 70 deg elevation: outside this
    # camera; what arrives comes from the halo - pointing the lens at the shower (el 90 - 20) is what the config does, so most hits
    # are within the camera; a lens that is not in focus smears them
    blur = copy.deepcopy(cfg)
    blur["detector"]["opt_focal_m"] = 0.6 * bfd
    res = api.run_config(blur)
    assert res["counters"]["cam_hit"] != c["cam_hit"]
    bad = copy.deepcopy(cfg)
    bad["detector"]["opt_lens_thickness_m"] = 13.0                           # thicker than the radius of curvature
    with pytest.raises(api.C8phError) as e:
        api.setup_context(bad)
    assert e.value.code == api.E_ARG


def test_substepping_matches_the_oracle_and_feeds_the_hot_path():
    """Row f2 (thesis sec. 4.2.1): tracks cut into chords of the Lorentz helix on the device (plan =
    count + prefix sum, fill = a warp per 32 tracks) against the oracle: piece counts bit-exact,
    positions to fp32 storage, directions 1e-6, lengths 1e-5 relative, clocks 1e-3 ns; the segments then
    run through c8ph_emit_propagate and agree with the oracle run on the oracle's segments."""
    rng = np.random.default_rng(21)
    n = 5000                                                              # several scan blocks + a ragged tail
    cfg = W.make_config(4, n_segments=n)
    trk = {k: v.copy() for k, v in cfg["segments"].items() if k != "edep"}
    trk["len"] = rng.uniform(5.0, 400.0, n).astype(np.float32)
    trk["p_GeV"] = (10 ** rng.uniform(-2.0, 1.0, n)).astype(np.float32)
    B, tol = (2.0e-5, -0.5e-5, -4.3e-5), 0.01
    want = O.substep_tracks(trk, B, tol)
    ctx = api.setup_context(cfg)
    dev = {k: torch.from_numpy(v).cuda() for k, v in trk.items()}
    seg, off = ctx.substep_tracks(dev, n, B, tol)
    assert np.array_equal(off.cpu().numpy(), want["offsets"]) and want["offsets"][-1] > 3 * n
    got = {k: v.cpu().numpy() for k, v in seg.items()}
    ws = want["segments"]
    for k in ("x", "y", "z"):
        assert np.abs(got[k].astype(np.float64) - ws[k]).max() <= 2 * np.spacing(np.float32(np.abs(ws[k]).max()))
    for k in ("dx", "dy", "dz"):
        assert np.abs(got[k] - ws[k]).max() < 1e-6
    assert np.allclose(got["len"], ws["len"], rtol=1e-5, atol=0) and np.allclose(got["t0"], ws["t0"], rtol=0, atol=1e-3 + 4e-3)
    assert np.array_equal(got["beta"], ws["beta"]) and np.array_equal(got["charge"], ws["charge"]) and not got["edep"].any()
    # no field: identity
    seg0, off0 = ctx.substep_tracks(dev, n, (0.0, 0.0, 0.0), tol)
    assert int(off0[-1]) == n and np.allclose(seg0["x"].cpu().numpy(), trk["x"]) and np.allclose(seg0["len"].cpu().numpy(), trk["len"], rtol=1e-6)
    # the pieces through the hot path: device pieces vs oracle pieces, photon by photon (2000 pieces)
    m = 2000
    sub = copy.deepcopy(cfg)
    sub["segments"] = {k: np.ascontiguousarray(v[:m]) for k, v in ws.items()}
    ora = O.run(sub)
    gcfg = copy.deepcopy(sub)
    gcfg["segments"] = {k: np.ascontiguousarray(v[:m]) for k, v in got.items()}
    gpu = api.run_config(gcfg, ctx=ctx)
    if all(np.array_equal(gcfg["segments"][k], sub["segments"][k]) for k in sub["segments"]):
        parity.compare(sub, ora, gpu)
    else:                                                                 # last-bit differences in the pieces: totals only
        assert abs(gpu["counters"]["emitted"] - ora["counters"]["emitted"]) <= 1e-3 * ora["counters"]["emitted"]


def test_multiple_scattering_substeps_match_the_oracle():
    """Row f2 with multiple scattering (R18): one thread walks one track (magnetic rotation, Highland
    offset and deflection per piece, normals from Philox counter (piece, track id, 16)).  Piece counts
    bit-exact; both sides walk in fp64, so the random walk agrees to rounding: positions to fp32 storage +
    1e-4 m, directions 1e-6, lengths 1e-5 relative; ids offset by track_id_base; E_STATE without an atmosphere."""
    rng = np.random.default_rng(22)
    n = 3000
    cfg = W.make_config(4, n_segments=n)
    trk = {k: v.copy() for k, v in cfg["segments"].items() if k != "edep"}
    trk["len"] = rng.uniform(5.0, 400.0, n).astype(np.float32)
    trk["p_GeV"] = (10 ** rng.uniform(-2.0, 1.0, n)).astype(np.float32)
    B, tol, step, seed, base = (2.0e-5, -0.5e-5, -4.3e-5), 0.01, 25.0, 77, 1 << 33
    want = O.substep_tracks_ms(cfg["atmosphere"], trk, B, tol, step, seed=seed, track_id_base=base)
    ctx = api.setup_context(cfg)
    dev = {k: torch.from_numpy(v).cuda() for k, v in trk.items()}
    seg, off = ctx.substep_tracks(dev, n, B, tol, ms_max_step_m=step, seed=seed, track_id_base=base)
    assert np.array_equal(off.cpu().numpy(), want["offsets"]) and want["offsets"][-1] > 5 * n
    got = {k: v.cpu().numpy() for k, v in seg.items()}
    ws = want["segments"]
    for k in ("x", "y", "z"):
        assert np.abs(got[k].astype(np.float64) - ws[k]).max() <= 2 * np.spacing(np.float32(np.abs(ws[k]).max())) + 1e-4
    for k in ("dx", "dy", "dz"):
        assert np.abs(got[k] - ws[k]).max() < 1e-6
    assert np.allclose(got["len"], ws["len"], rtol=1e-5, atol=0) and np.allclose(got["t0"], ws["t0"], rtol=0, atol=5e-3)
    assert np.array_equal(got["beta"], ws["beta"]) and np.array_equal(got["charge"], ws["charge"]) and not got["edep"].any()
    # the walk really scatters: the pieces differ from the helix chords of the same count by far more than rounding
    seg_h, off_h = ctx.substep_tracks(dev, n, B, tol)
    assert int(off[-1]) > int(off_h[-1])
    low = trk["p_GeV"] < 0.05
    first, last = want["offsets"][:-1][low], want["offsets"][1:][low] - 1
    bend = np.abs(got["dx"][last] - got["dx"][first]) + np.abs(got["dy"][last] - got["dy"][first])
    assert np.median(bend) > 1e-3
    # another id base draws other normals
    seg2, _ = ctx.substep_tracks(dev, n, B, tol, ms_max_step_m=step, seed=seed, track_id_base=0)
    assert np.abs(seg2["x"].cpu().numpy() - got["x"]).max() > 1e-3
    # no atmosphere in the context: refused
    bare = api.Context()
    with pytest.raises(api.C8phError) as e:
        bare.substep_tracks(dev, n, B, tol, ms_max_step_m=step)
    assert e.value.code == api.E_STATE


@pytest.mark.parametrize("trial", range(6))
def test_random_telescope_arrays(trial, monkeypatch):
    """Seeded random telescope arrays: 1 to 16382 spheres (the record's 14-bit index allows 16382), radii 0.5-15 m at
    altitudes +-5 m, packed into 60 m (heavily overlapping) up to 5 km squares, with a nested pair and an exact
    duplicate (earliest entry, then lowest index): device against oracle, and grid search against search-all."""
    rng = np.random.default_rng(55000 + trial)
    k = int(rng.choice([2, 4]))
    cfg = W.make_config(k, n_segments={2: 6000, 4: 1200}[k])
    n_tel = (16382, 1, 150, 3000, 9, 2)[trial]
    ext = float(rng.choice([30.0, 300.0, 2500.0]))
    t = np.zeros((n_tel, 4), np.float32)
    t[:, 0], t[:, 1] = rng.uniform(-ext, ext, n_tel), rng.uniform(-ext, ext, n_tel)
    t[:, 2], t[:, 3] = rng.uniform(-5, 5, n_tel), rng.uniform(0.5, 15.0, n_tel)
    if n_tel > 3:
        t[1, :3] = t[0, :3] + np.float32([0.3, -0.2, 0.1])
    if n_tel > 5:
        t[4] = t[3]
    cfg["detector"]["tel_xyzr"] = t
    cfg["params"]["lv2_margin_m"] = float(rng.uniform(0, 50))
    ora, gpu, rep = _both(cfg, capacity=1 << 23)
    monkeypatch.setenv("C8PH_FORCE_BRUTE", "1")
    ctx = api.setup_context(cfg)
    br = api.run_config(cfg, ctx=ctx, photon_capacity=1 << 23)
    ctx.close()
    assert br["counters"] == gpu["counters"] and np.array_equal(br["tel_counts"], gpu["tel_counts"])


@pytest.mark.parametrize("trial", range(8))
def test_random_substepping_inputs(trial):
    """Sub-stepping under seeded random inputs: track counts around the warp / scan-block sizes (1, 31, 33, 700, 2049),
    neutral and doubly charged particles, zero and random fields, tolerances, piece caps, with and without multiple
    scattering (steps 0 = no cap, 10, 50 m), 40-bit id bases - piece counts bit-exact, pieces to fp32 storage."""
    rng = np.random.default_rng(31000 + trial)
    n, k = int(rng.choice([1, 31, 33, 700, 2049])), int(rng.choice([1, 4]))
    cfg = W.make_config(k, n_segments=n)
    trk = {kk: v.copy() for kk, v in cfg["segments"].items() if kk != "edep"}
    trk["len"] = rng.uniform(0.5, 900.0, n).astype(np.float32)
    trk["p_GeV"] = (10 ** rng.uniform(-2.3, 1.5, n)).astype(np.float32)
    trk["charge"] = rng.choice([-1.0, 1.0, 2.0, 0.0], n).astype(np.float32)
    B = tuple(float(x) for x in rng.normal(0, 3e-5, 3)) if rng.integers(4) else (0.0, 0.0, 0.0)
    tol, max_sub = float(rng.choice([0.001, 0.01, 0.1])), int(rng.choice([8, 64, 4096]))
    ms = None if rng.integers(2) else float(rng.choice([0.0, 10.0, 50.0]))
    seed, base = int(rng.integers(1, 2 ** 60)), int(rng.integers(0, 2 ** 40))
    if ms is None:
        want = O.substep_tracks(trk, B, tol, max_sub)
    else:
        want = O.substep_tracks_ms(cfg["atmosphere"], trk, B, tol, ms, seed=seed, track_id_base=base, max_sub=max_sub)
    ctx = api.setup_context(cfg)
    dev = {kk: torch.from_numpy(v).cuda() for kk, v in trk.items()}
    seg, off = ctx.substep_tracks(dev, n, B, tol, max_sub, ms_max_step_m=ms, seed=seed, track_id_base=base)
    assert np.array_equal(off.cpu().numpy(), want["offsets"])
    got, ws = {kk: v.cpu().numpy() for kk, v in seg.items()}, want["segments"]
    for kk in ("x", "y", "z"):
        assert np.abs(got[kk].astype(np.float64) - ws[kk]).max() <= 2 * np.spacing(np.float32(np.abs(ws[kk]).max())) + 2e-4
    for kk in ("dx", "dy", "dz"):
        assert np.abs(got[kk] - ws[kk]).max() < 2e-6
    assert np.allclose(got["len"], ws["len"], rtol=2e-5, atol=1e-6) and np.allclose(got["t0"], ws["t0"], rtol=0, atol=6e-3)


def _off_centre(k, n, shift_m, zen_deg=None, **par):
    """cfg k with segments, ground grid and telescopes moved rigidly by shift_m along x: the array sits that far
    from the point where the plane z = 0 touches the observation sphere.  zen_deg: the segments become inclined
    tracks of that zenith angle (random azimuth) whose axes pass within ~60 m of the array centre."""
    cfg = W.make_config(k, n_segments=n)
    s = cfg["segments"]
    if zen_deg is not None:
        rng = np.random.default_rng(5)
        az, th = rng.uniform(0, 2 * np.pi, n), np.radians(zen_deg)
        s["dx"] = (np.sin(th) * np.cos(az)).astype(np.float32)
        s["dy"] = (np.sin(th) * np.sin(az)).astype(np.float32)
        s["dz"] = np.full(n, -np.cos(th), np.float32)
        s["x"] = (-s["z"] * np.tan(th) * np.cos(az) + rng.normal(0, 60, n)).astype(np.float32)
        s["y"] = (-s["z"] * np.tan(th) * np.sin(az) + rng.normal(0, 60, n)).astype(np.float32)
    s["x"] = (s["x"] + np.float32(shift_m)).astype(np.float32)
    cfg["detector"]["hist_x0"] = cfg["detector"]["hist_x0"] + shift_m
    tel = cfg["detector"]["tel_xyzr"].copy()
    tel[:, 0] += np.float32(shift_m)
    cfg["detector"]["tel_xyzr"] = tel
    cfg["params"].update(par)
    return cfg


def test_flat_observation_plane_far_from_the_origin():
    """Row f1 (thesis Fig. 4.10; R19): the detector plane z = 0 against the observation sphere of
    the (height, zenith) table.  cfg4's array 18 km from the origin (sag 25 m): device against oracle photon by
    photon with the flat-plane step on - cfg4's own near-vertical tracks, tracks inclined by 60 and 70 degrees
    (where the step moves photons by up to 8 and 37 cm and the clock by up to 0.2 and 1.2 ns: more than the
    tolerances); at the origin the step changes nothing.  (The per-photon layered sum is planar only.)"""
    shift = 18000.0
    for zen, n, d_med, d_max, t_med in ((None, 2500, 5e-4, 2e-3, 0.02), (60.0, 1500, 0.01, 0.07, 0.015), (70.0, 1500, 0.03, 0.3, 0.04)):
        cfg = _off_centre(4, n, shift, zen, flat_plane=True)
        ora, gpu, rep = _both(cfg)
        assert gpu["counters"]["tel_hit"] > 1e4 and gpu["counters"]["in_grid"] > 1e5
        assert rep["max_dpos_m"] < 0.02 and rep["max_dt_ns"] < 0.05
        off = O.run(_off_centre(4, n, shift, zen, flat_plane=False))
        a, b = ora["photons"], off["photons"]
        both = (a["status"] == O.ST_LANDED) & (b["status"] == O.ST_LANDED)
        d = np.hypot(a["x"][both] - b["x"][both], a["y"][both] - b["y"][both])
        assert both.sum() > 1e5 and np.median(d) > d_med and d.max() > d_max
        assert np.median(np.abs(a["t"][both] - b["t"][both])) > t_med
    # at the origin the step is below the tolerances: same histogram with and without it
    near_on = api.run_config(_off_centre(4, 1500, 0.0, flat_plane=True))
    near_off = api.run_config(_off_centre(4, 1500, 0.0, flat_plane=False))
    moved = 0.5 * np.abs(near_on["hist"].astype(np.float64) - near_off["hist"]).sum()
    assert near_on["counters"]["landed"] == near_off["counters"]["landed"] and moved <= 1e-4 * near_on["counters"]["emitted"]


_FLAT_TABLE = dict(n_h=256, n_zen=256, h_max=50000.0, zen_max_deg=80.0, n_rho=16, rho_max_m=30000.0)


def test_flat_plane_table_nodes_and_photons_against_the_oracle(monkeypatch):
    """Row f1 (thesis P:861, Fig. 4.10; R21): the table relative to the flat observation plane over (height,
    zenith, polar radius, pointing angle).  Device nodes against the oracle's (0.1 mm / 0.3 ps where the 2-D nodes
    agree to that); photons with flat_plane = 2 against the oracle, array 18 km from the origin, cfg4's near-vertical
    tracks and tracks inclined by 60 degrees (every azimuth, so every pointing angle); the compiled variant and the
    generic kernel agree; against the analytic step (flat_plane = 1) the positions stay within 1 mm."""
    cfg = _off_centre(4, 2500, 18000.0, None, flat_plane=2)
    cfg["table"] = dict(cfg["table"], **_FLAT_TABLE)
    ctx = api.setup_context(cfg)
    got = ctx.get_trace_table_flat()
    want = O.table_flat_for(cfg)
    assert got.shape == (2, 16, 256, 256, 4) and want.shape == (2, 16, 256, 256, 5)
    zen = np.linspace(0.0, 80.0, 256)
    for part, chans in ((0, ((0, 0, 1e-4), (1, 2, 3e-4), (2, 3, 1e-2))), (1, ((0, 0, 1e-4), (1, 2, 3e-4), (2, 3, 1e-4)))):
        for cg, cw, tol in chans:
            g, w = got[part, ..., cg].astype(np.float64), want[part, ..., cw].astype(np.float64)
            ok = np.isfinite(g) & np.isfinite(w) & (zen[None, None, :] <= 70.0)
            assert ok.mean() > 0.7 and np.abs(g - w)[ok].max() <= tol, (part, cg, np.abs(g - w)[ok].max())
    assert (np.isfinite(got[0, ..., 0]) != np.isfinite(want[0, ..., 0])).mean() < 1e-3
    for zen_deg, n in ((None, 2500), (60.0, 1500)):
        c2 = _off_centre(4, n, 18000.0, zen_deg, flat_plane=2)
        c2["table"] = dict(c2["table"], **_FLAT_TABLE)
        ora, gpu, rep = _both(c2)
        assert gpu["counters"]["tel_hit"] > 1e4 and gpu["counters"]["in_grid"] > 1e5 and rep["max_dpos_m"] < 0.02
        monkeypatch.setenv("C8PH_FORCE_GENERIC", "1")
        gen = api.run_config(c2, ctx=api.setup_context(c2))
        monkeypatch.setenv("C8PH_FORCE_GENERIC", "0")
        parity.compare(c2, ora, gen)
        c1 = copy.deepcopy(c2)
        c1["params"]["flat_plane"] = 1
        step = O.run(c1)
        a, b = ora["photons"], step["photons"]
        both = (a["status"] == O.ST_LANDED) & (b["status"] == O.ST_LANDED)
        assert both.sum() > 1e5 and np.hypot(a["x"][both] - b["x"][both], a["y"][both] - b["y"][both]).max() < 1e-3
    # beyond rho_max the lookup is out of range: counted, not extrapolated
    far = _off_centre(4, 400, 31000.0, None, flat_plane=2)
    far["table"] = dict(far["table"], **_FLAT_TABLE)
    res = api.run_config(far)
    assert res["counters"]["table_range"] > 0.5 * (res["counters"]["emitted"] - res["counters"]["lv2"] - res["counters"]["upgoing"])
    # flat_plane = 2 without the extra axes is a state error
    with pytest.raises(api.C8phError) as e:
        api.run_config(_off_centre(4, 100, 0.0, None, flat_plane=2))
    assert e.value.code == api.E_STATE


def test_cylindrical_atmosphere_model_nodes_and_photons_against_the_oracle():
    """Row f1 (thesis sec. 3.3.3; R24): the cylindrical model.  The device builds its table by Bouguer's
    invariant in the plane of curvature with the effective index sqrt(n^2 - kappa^2); the oracle by stepping Eq. 3.15 in
    three dimensions: node by node 0.1 mm / 0.3 ps (also the displacement across the flight, which the spherical model
    does not have).  Photons: cfg4's array 8 km from the origin, tracks inclined by 50 degrees at every azimuth (so every
    angle against the plane of curvature), device against oracle; and against the spherical model the same photons
    differ by millimetres to centimetres, as the thesis says of instrumented areas of this size."""
    tab = dict(n_h=192, n_zen=192, h_max=40000.0, zen_max_deg=75.0, n_c=5)
    cfg = _off_centre(4, 1500, 8000.0, 50.0)
    cfg["atmosphere"]["model"] = "cylindrical"
    cfg["table"] = dict(tab)
    ctx = api.setup_context(cfg)
    got = ctx.get_trace_table_cyl()
    want = O.table_cyl_for(cfg)
    assert got.shape == (5, 192, 192, 4) and want.shape == (5, 192, 192, 5)
    zen = np.linspace(0.0, 75.0, 192)
    for cg, cw, tol in ((0, 0, 1e-4), (1, 2, 3e-4), (2, 3, 1e-2), (3, 1, 2e-4)):
        g, w = got[..., cg].astype(np.float64), want[..., cw].astype(np.float64)
        ok = np.isfinite(g) & np.isfinite(w) & (zen[None, None, :] <= 70.0)
        assert ok.mean() > 0.85 and np.abs(g - w)[ok].max() <= tol, (cg, np.abs(g - w)[ok].max())
    assert np.abs(got[2, 100, 150, 3]) > 1e-3                          # the across displacement is there (millimetres)
    ora, gpu, rep = _both(cfg, ctx=ctx)
    assert gpu["counters"]["tel_hit"] > 1e4 and gpu["counters"]["in_grid"] > 1e5 and rep["max_dpos_m"] < 5e-3
    sph = copy.deepcopy(cfg)
    sph["atmosphere"]["model"] = "spherical"
    sph["table"] = {k: v for k, v in tab.items() if k != "n_c"}
    so = O.run(sph)
    a, b = ora["photons"], so["photons"]
    both = (a["status"] == O.ST_LANDED) & (b["status"] == O.ST_LANDED)
    d = np.hypot(a["x"][both] - b["x"][both], a["y"][both] - b["y"][both])
    assert both.sum() > 1e5 and 1e-3 < d.max() < 0.2 and np.median(d) > 1e-4
    # state errors: the model needs its table, and has no numeric tracing, aerosol or fluorescence
    bad = copy.deepcopy(cfg)
    bad["table"] = {k: v for k, v in tab.items() if k != "n_c"}
    with pytest.raises(api.C8phError) as e:
        api.run_config(bad)
    assert e.value.code == api.E_STATE


def test_compiled_feature_variants_and_the_generic_kernel_agree(monkeypatch):
    """The "production setting + optional features" calls run kernel variants with the features compiled in (SPEC bit
    mask); C8PH_FORCE_GENERIC=1 sends the same call through the generic variant that reads every switch at run time.
    Both against the oracle photon by photon, for the plain production setting, one feature (efficiency), and all five
    together (flat plane, tabulated extinction, dispersion, efficiency, optics) with the array 18 km off centre (the
    reflected directions keep 1e-5 rad there because the mirror coordinates are formed relative to the segment
    anchor, not from fp32 ground coordinates), and the dispersive, flat-plane case on tracks inclined by 60 degrees."""
    lam = np.arange(200.0, 801.0, 10.0)
    eff = dict(eff=(0.85 * np.exp(-0.5 * ((lam - 420.0) / 90.0) ** 2)).astype(np.float32), eff_lambda0_nm=200.0, eff_dlambda_nm=10.0)

    def all_five():
        cfg = _off_centre(4, 2500, 18000.0, None, flat_plane=True, disp_b_nm2=5700.0, disp_lambda0_nm=400.0, **eff)
        atm = cfg["atmosphere"]
        xv = atm["overburden"].astype(np.float64)
        h = atm["h0"] + atm["dh"] * np.arange(atm["n_nodes"])
        lam_e = np.arange(240.0, 711.0, 10.0)
        tau = (400.0 / lam_e[:, None]) ** 4 * np.maximum(np.interp(atm["h_obs"], h, xv) - xv[None, :], 0.0) / 2970.0
        atm.update(ext_tau_v=tau.astype(np.float32), ext_lambda0_nm=240.0, ext_dlambda_nm=10.0)
        cfg["detector"]["tel_xyzr"][:, 3] = 12.0
        cfg["detector"].update(opt_enabled=True, opt_az_deg=0.0, opt_el_deg=70.0, opt_focal_m=17.0,
                               opt_mirror_radius_m=8.5, opt_camera_radius_m=0.735)
        return cfg

    def inclined():
        return _off_centre(4, 1500, 18000.0, 60.0, flat_plane=True, disp_b_nm2=5700.0, disp_lambda0_nm=400.0)

    def one():
        cfg = W.make_config(4, n_segments=2500)
        cfg["params"].update(eff)
        return cfg

    for make in (lambda: W.make_config(4, n_segments=2500), one, all_five, inclined):
        cfg = make()
        ora = O.run(cfg)
        res = {}
        for mode in ("compiled", "generic"):
            monkeypatch.setenv("C8PH_FORCE_GENERIC", "1" if mode == "generic" else "0")
            ctx = api.setup_context(cfg)                               # the switch is read at c8ph_create
            res[mode] = api.run_config(cfg, ctx=ctx, photon_capacity=1 << 22)
            ctx.close()
            parity.compare(cfg, ora, res[mode])
        a, b = res["compiled"]["counters"], res["generic"]["counters"]
        assert a["emitted"] > 1e5 and all(abs(a[k] - b[k]) <= 3 for k in a), (a, b)
        if make is all_five:
            assert a["cam_hit"] > 50


@pytest.mark.parametrize("trial", range(20))
def test_random_switch_combinations(trial):
    """The generic kernel variants under seeded random combinations of the run-time switches (filters, transmission
    mode, write mode, bunch weight, margins, aerosol, trace method, detectors present or not), device against
    oracle photon by photon: combinations that none of the BASELINE configs uses.  (Not in the matrix, by
    conditioning rather than by method: WRITE_ALL without LV2 on cfg2's 60 degree shower and fluorescence with the
    straight trace keep photons with |u_z| ~ 1e-3 whose plane point lies kilometres away and whose (u_x, u_y)
    record cannot resolve u_z.)"""
    rng = np.random.default_rng(4200 + trial)
    k = int(rng.choice([0, 1, 2, 4])) if trial < 16 else 3
    cfg = W.make_config(k, n_segments={0: 400, 1: 250, 2: 8000, 3: 20000, 4: 1500}[k])
    par, det, atm = cfg["params"], cfg["detector"], cfg["atmosphere"]
    if k == 3:                                                          # fluorescence, camera: transmission mode, weight, aerosol
        cfg["segments"]["edep"][:] *= 40.0
        par["trans"] = str(rng.choice(["off", "weight", "roulette"]))
        par["bunch_weight"] = float(rng.choice([0.5, 1.0]))
        if rng.integers(2):
            atm["aer_L"] = 15000.0
        ora, gpu, rep = _both(cfg)
        assert gpu["counters"]["cam_hit"] > 300
        return
    par["lv1"], par["lv2"] = bool(rng.integers(2)), bool(rng.integers(2))
    par["trans"] = str(rng.choice(["off", "weight", "roulette"]))
    par["write"] = str(rng.choice(["all", "tel", "none"]))
    par["bunch_weight"] = float(rng.choice([0.5, 1.0, 2.5]))
    par["lv2_margin_m"] = float(rng.uniform(0.0, 40.0))
    par["lv1_margin_rad"] = float(rng.uniform(0.0, 0.03))
    if k != 0 and rng.integers(2):
        atm["aer_L"] = 15000.0                                          # aerosol extinction on
    if k in (2, 4) and rng.integers(3) == 0:
        par["trace"], cfg["table"] = "straight", None
    if k == 1 and rng.integers(3) == 0:
        par["trace"] = "straight"
    if len(det["tel_xyzr"]) and rng.integers(4) == 0:
        det["tel_xyzr"] = np.zeros((0, 4), np.float32)                  # no telescopes
    elif det["hist_nx"] > 0 and rng.integers(4) == 0:
        det["hist_nx"] = det["hist_ny"] = 0                             # no ground grid
    if k == 4 and rng.integers(3) == 0:
        par["flat_plane"] = True
    ora, gpu, rep = _both(cfg)
    assert gpu["counters"]["emitted"] > 2000


@pytest.mark.parametrize("trial", range(10))
def test_random_geometry_tables_ids_and_entry_points(trial):
    """Seeded random variations of what the BASELINE configs keep fixed: seed and 40-bit segment id base, observation
    level, correction-table dimensions and limits, histogram geometry, irregular telescope arrays with radii and
    altitudes, margins, weights - through the device and the host entry point, against the oracle photon by photon."""
    rng = np.random.default_rng(777000 + trial)
    k = int(rng.choice([0, 1, 2, 4, 4]))
    cfg = W.make_config(k, n_segments={0: 400, 1: 250, 2: 8000, 4: 1500}[k])
    par, det, atm = cfg["params"], cfg["detector"], cfg["atmosphere"]
    cfg["seed"], cfg["seg_id_base"] = int(rng.integers(1, 2 ** 62)), int(rng.integers(0, 2 ** 40))
    if k in (1, 2, 4) and rng.integers(2):
        atm["h_obs"] = float(rng.choice([0.0, 800.0, 1800.0, 2200.0]))
    if cfg.get("table") is not None and rng.integers(2):
        cfg["table"] = dict(n_h=int(rng.choice([128, 300, 512])), n_zen=int(rng.choice([64, 200, 256])),
                            h_max=float(rng.choice([60000.0, 100000.0])), zen_max_deg=float(rng.choice([80.0, 89.0])))
    if det["hist_nx"] > 0 and rng.integers(2):
        cell, nx, ny = float(rng.choice([0.5, 1.0, 2.5, 7.0])), int(rng.integers(50, 700)), int(rng.integers(50, 700))
        det.update(hist_cell=cell, hist_nx=nx, hist_ny=ny, hist_x0=float(-0.5 * nx * cell + rng.uniform(-100, 100)),
                   hist_y0=float(-0.5 * ny * cell + rng.uniform(-100, 100)))
    if len(det["tel_xyzr"]) and rng.integers(2):
        t = det["tel_xyzr"].copy()
        t[:, 3] = rng.uniform(2.0, 9.0, len(t)).astype(np.float32)
        t[:, 2] = rng.uniform(-3.0, 3.0, len(t)).astype(np.float32)
        t[:, 0] += rng.uniform(-8, 8, len(t)).astype(np.float32)
        t[:, 1] += rng.uniform(-8, 8, len(t)).astype(np.float32)
        det["tel_xyzr"] = t
    par["lv1"], par["lv2"] = bool(rng.integers(2)), True
    par["trans"] = str(rng.choice(["off", "weight", "roulette"]))
    par["write"] = str(rng.choice(["tel", "none", "tel"]))
    par["bunch_weight"] = float(rng.choice([0.5, 1.0, 2.5]))
    par["lv2_margin_m"] = float(rng.uniform(0.0, 60.0))
    ora = O.run(cfg)
    if rng.integers(2):
        ctx = api.setup_context(cfg)
        gpu = ctx.emit_propagate_host(cfg["segments"], len(cfg["segments"]["x"]), cfg["seg_id_base"], par, cfg["seed"],
                                      photon_capacity=1 << 22, want_weight=True)
    else:
        gpu = api.run_config(cfg, photon_capacity=1 << 22)
    parity.compare(cfg, ora, gpu)
    assert gpu["counters"]["emitted"] > 2000


def test_tabulated_extinction():
    """Row f4: transmission from a tau_v(lambda, h) table (MODTRAN-type, thesis Fig. 4.7a) with air-mass
    scaling instead of the analytic laws: device against oracle on the same table (Rayleigh + an
    aerosol-like layer on a 10 nm grid), roulette (cfg2, cfg4) and weight mode (cfg1)."""
    lam = np.arange(240.0, 711.0, 10.0)
    for k, n in ((2, 20000), (4, 2500), (1, 600)):
        cfg = W.make_config(k, n_segments=n)
        atm = cfg["atmosphere"]
        xv = atm["overburden"].astype(np.float64)
        h = atm["h0"] + atm["dh"] * np.arange(atm["n_nodes"])
        xg = np.interp(atm["h_obs"], h, xv)
        ray = (400.0 / lam[:, None]) ** 4 * np.maximum(xg - xv[None, :], 0.0) / 2970.0
        aer = (350.0 / lam[:, None]) * (1200.0 / 15000.0) * np.maximum(np.exp(-atm["h_obs"] / 1200.0) - np.exp(-h[None, :] / 1200.0), 0.0)
        atm.update(ext_tau_v=(ray + aer).astype(np.float32), ext_lambda0_nm=240.0, ext_dlambda_nm=10.0)
        ora, gpu, rep = _both(cfg)
        off = api.run_config(W.make_config(k, n_segments=n))
        if k == 1:
            assert gpu["hist"].sum() < off["hist"].sum()
        else:
            assert gpu["counters"]["roulette"] > off["counters"]["roulette"]        # the aerosol layer removes more
    cfg = W.make_config(0, n_segments=10)                                           # homogeneous model: refused
    cfg["atmosphere"].update(ext_tau_v=np.zeros((2, cfg["atmosphere"]["n_nodes"]), np.float32), ext_lambda0_nm=300.0, ext_dlambda_nm=300.0)
    with pytest.raises(api.C8phError) as e:
        api.setup_context(cfg)
    assert e.value.code == api.E_ARG
