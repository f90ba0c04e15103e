"""Boundary behaviour of the C-ABI on the GPU (-m gpu): segment ids and order independence, the NONFINITE counter,
launches on several streams, graph capture of calls that use the context's wavelength tables, sharded runs reduced
over a process group (SURVEY 8(b), 8(e), section 5 "Race detection / sanitizers").
"""
import copy
import os
import socket

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
if not torch.cuda.is_available():                                     # pragma: no cover
    pytest.skip("no CUDA device", allow_module_level=True)

from oracle import c8ph_oracle as O                                    # noqa: E402
from paper_2405_04229_b200 import api, build, shard, workloads as W   # noqa: E402
import c8ph_parity as parity                                           # noqa: E402

build.build()


def _sorted_records(res, seg_map=None):
    p = res["photons"].copy()
    if seg_map is not None:
        p["seg"] = seg_map[p["seg"]]
    return p[np.argsort(p["seg"].astype(np.int64) << 32 | p["j_tel"])]


@pytest.mark.parametrize("k,n", [(4, 2500), (0, 500)])
def test_shuffled_segments_with_ids_give_identical_sorted_output(k, n):
    """results depend on (seed, segment id, photon index) only.  The segments are handed over in a
    random order together with their ids: histogram, counters and the photon list (mapped back to the original
    index and sorted) are those of the ordered run, bit for bit, on the device and in the oracle."""
    cfg = W.make_config(k, n_segments=n)
    ref = api.run_config(cfg)
    perm = np.random.default_rng(5).permutation(n)
    sh = copy.deepcopy(cfg)
    sh["segments"] = {f: np.ascontiguousarray(v[perm]) for f, v in cfg["segments"].items()}
    sh["segments"]["id"] = perm.astype(np.uint64) + np.uint64(cfg["seg_id_base"])
    got = api.run_config(sh)
    assert got["counters"] == ref["counters"]
    assert np.array_equal(got["hist"], ref["hist"]) and np.array_equal(got["tel_counts"], ref["tel_counts"])
    assert np.array_equal(_sorted_records(got, perm.astype(np.uint32)), _sorted_records(ref))
    # same through the host-buffer entry point (ids cross the PCIe pipeline too)
    ctx = api.setup_context(sh)
    host = ctx.emit_propagate_host(sh["segments"], n, 0, sh["params"], sh["seed"], photon_capacity=1 << 22)
    assert host["counters"] == ref["counters"] and np.array_equal(host["hist"], ref["hist"])
    assert np.array_equal(_sorted_records(host, perm.astype(np.uint32)), _sorted_records(ref))
    # and the oracle agrees with itself and with the device
    ora_ref, ora_sh = O.run(cfg), O.run(sh)
    assert ora_ref["counters"] == ora_sh["counters"] and np.array_equal(ora_ref["hist"], ora_sh["hist"])
    print("parity (shuffled):", parity.summary(parity.compare(cfg, ora_ref, ref)))


def test_non_finite_segments_are_dropped_and_counted():
    """NaN / Inf in any segment field, or a direction of zero length, drops the segment and counts it in
    NONFINITE on both sides; every other segment is untouched."""
    n = 1200
    cfg = W.make_config(4, n_segments=n)
    clean = api.run_config(cfg)
    bad = copy.deepcopy(cfg)
    seg = bad["segments"]
    fields = ("x", "y", "z", "dx", "dy", "dz", "len", "beta", "t0", "charge")
    hit = []
    for t, f in enumerate(fields):
        for m, v in enumerate((np.nan, np.inf, -np.inf)):
            i = 17 + 31 * t + 7 * m
            seg[f][i] = v
            hit.append(i)
    for i in (900, 901):
        seg["dx"][i] = seg["dy"][i] = seg["dz"][i] = 0.0
        hit.append(i)
    hit = sorted(set(hit))
    gpu = api.run_config(bad)
    ora = O.run(bad)
    assert gpu["counters"]["nonfinite"] == ora["counters"]["nonfinite"] == len(hit)
    assert gpu["counters"]["segments"] == n and clean["counters"]["nonfinite"] == 0
    assert not np.isin(gpu["photons"]["seg"], hit).any()
    assert np.isfinite(gpu["hist"]).all() and np.isfinite(gpu["tel_counts"]).all()
    parity.compare(bad, ora, gpu)
    # the surviving segments give exactly the photons of the clean run
    keep = ~np.isin(clean["photons"]["seg"], hit)
    assert np.array_equal(_sorted_records(gpu), _sorted_records({"photons": clean["photons"][keep]}))


def test_launches_on_two_streams_are_ordered_by_the_library():
    """One context, two streams, no synchronisation by the caller: the launches share the context's work cursor and
    segment slots, so the library orders them (c8ph.h); both results equal those of separate, sequential runs."""
    cfg_a = W.make_config(4, n_segments=40000)
    cfg_b = copy.deepcopy(cfg_a)
    cfg_b["segments"] = W.slice_segments(cfg_a["segments"], 20000, 40000)
    ctx = api.setup_context(cfg_a)
    want_a = api.run_config(cfg_a, ctx=ctx, photon_capacity=1 << 21)
    want_b = api.run_config(dict(cfg_b, seg_id_base=7_000_000), ctx=ctx, photon_capacity=1 << 21)
    seg_a, seg_b = api.segments_to_device(cfg_a["segments"]), api.segments_to_device(cfg_b["segments"])
    out_a, out_b = api.alloc_device_outputs(ctx, 1 << 21, True), api.alloc_device_outputs(ctx, 1 << 21, True)
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    torch.cuda.synchronize()
    for rep in range(3):
        for o in (out_a, out_b):
            for kk in ("hist", "tel_counts", "counters"):
                o[kk].zero_()
        torch.cuda.synchronize()
        ctx.emit_propagate(seg_a, 40000, 0, cfg_a["params"], cfg_a["seed"], out_a, stream=s1)
        ctx.emit_propagate(seg_b, 20000, 7_000_000, cfg_b["params"], cfg_b["seed"], out_b, stream=s2)
        ctx.emit_propagate(seg_b, 20000, 7_000_000, cfg_b["params"], cfg_b["seed"], out_b, stream=s1)
        torch.cuda.synchronize()
        got_a, got_b = api.outputs_to_host(ctx, out_a), api.outputs_to_host(ctx, out_b)
        assert got_a["counters"] == want_a["counters"] and np.array_equal(got_a["hist"], want_a["hist"])
        assert np.array_equal(_sorted_records(got_a), _sorted_records(want_a))
        assert np.array_equal(got_b["hist"], 2 * want_b["hist"])                      # accumulated by two launches
        assert got_b["counters"]["emitted"] == 2 * want_b["counters"]["emitted"]
        assert got_b["counters"]["written"] == 2 * want_b["counters"]["written"]


def test_graph_capture_of_calls_that_use_the_context_tables():
    """The line spectrum and the efficiency table live in the context (c8ph_set_line_spectrum / c8ph_set_efficiency):
    the hot call allocates and copies nothing, so fluorescence (cfg3) and a call with a detector efficiency can be
    captured into CUDA graphs; replays give the bits of the eager call."""
    cases = []
    c3 = W.make_config(3, n_segments=20000)
    c3["segments"]["edep"][:] *= 40.0
    cases.append(c3)
    c4 = W.make_config(4, n_segments=1500)
    lam = np.arange(200.0, 801.0, 10.0)
    c4["params"].update(eff=(0.85 * np.exp(-0.5 * ((lam - 420.0) / 90.0) ** 2)).astype(np.float32),
                        eff_lambda0_nm=200.0, eff_dlambda_nm=10.0)
    cases.append(c4)
    for cfg in cases:
        n = len(cfg["segments"]["x"])
        ctx = api.setup_context(cfg)
        eager = api.run_config(cfg, ctx=ctx)                           # also hands the tables to the context
        assert eager["counters"]["emitted"] > 1000
        seg = api.segments_to_device(cfg["segments"])
        out = api.alloc_device_outputs(ctx, 1 << 20, True)
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=side):
            for kk in ("hist", "tel_counts", "counters"):
                out[kk].zero_()
            ctx.emit_propagate(seg, n, 0, cfg["params"], cfg["seed"], out, stream=torch.cuda.current_stream())
        for _ in range(2):
            g.replay()
        torch.cuda.synchronize()
        rep = api.outputs_to_host(ctx, out)
        assert rep["counters"] == eager["counters"] and np.array_equal(rep["hist"], eager["hist"])
        assert np.array_equal(_sorted_records(rep), _sorted_records(eager))
        ctx.close()


def test_state_and_argument_errors_of_the_table_setters():
    cfg = W.make_config(3, n_segments=64)
    ctx = api.Context(0)
    ctx.init_atmosphere(cfg["atmosphere"])
    ctx.build_trace_table(cfg["table"])
    ctx.set_detector(cfg["detector"])
    seg = api.segments_to_device(cfg["segments"])
    out = api.alloc_device_outputs(ctx, 1024)
    # fluorescence without a line spectrum in the context: state error from the library itself
    par = dict(cfg["params"], line_nm=np.zeros(0, np.float32), line_cdf=np.zeros(0, np.float32))
    with pytest.raises(api.C8phError) as e:
        ctx.emit_propagate(seg, 64, 0, par, 1, out)
    assert e.value.code == api.E_STATE
    with pytest.raises(api.C8phError) as e:
        ctx.set_line_spectrum([400.0, 350.0], [0.7, 0.5])             # cdf must not fall
    assert e.value.code == api.E_ARG
    with pytest.raises(api.C8phError) as e:
        ctx.set_efficiency([0.5, 1.5], 300.0, 10.0)
    assert e.value.code == api.E_ARG
    # a camera needs exactly one telescope (hits on other spheres would enter its image)
    det = dict(cfg["detector"])
    det["tel_xyzr"] = np.concatenate([det["tel_xyzr"], det["tel_xyzr"] + np.float32([50, 0, 0, 0])]).astype(np.float32)
    with pytest.raises(api.C8phError) as e:
        ctx.set_detector(det)
    assert e.value.code == api.E_ARG
    ctx.close()


# ------------------------------------------------------------------------------------------ sharded runs
def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _shard_rank(rank, world, port, k, n, out_dir):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        cfg = W.make_config(k, n_segments=n)
        lo, hi = shard.shard_of(n, rank, world)
        sub = dict(cfg)
        sub["segments"] = W.slice_segments(cfg["segments"], lo, hi)
        ctx = api.setup_context(sub)
        seg = api.segments_to_device(sub["segments"])
        out = api.alloc_device_outputs(ctx, 1 << 21, False)
        ctx.emit_propagate(seg, hi - lo, lo, sub["params"], sub["seed"], out)         # seg_id_base = lo
        torch.cuda.synchronize()
        host = {kk: out[kk].cpu() for kk in ("hist", "tel_counts", "counters")}
        shard.reduce_results(host)                                                     # the one exchange step (8(e))
        if rank == 0:
            np.savez(os.path.join(out_dir, "reduced.npz"), hist=host["hist"].numpy(), tel=host["tel_counts"].numpy(),
                     cnt=host["counters"].numpy(), written_local=host["written_local"])
    finally:
        dist.destroy_process_group()


def test_two_library_shards_reduce_to_the_single_run(tmp_path):
    """two ranks (two processes, two contexts; here on one GPU, gloo for the exchange) each run their
    contiguous id range through the LIBRARY with seg_id_base = lo; the SUM all-reduce of histogram, telescope counters
    and event counters equals the single run bit for bit."""
    import torch.multiprocessing as mp
    k, n = 4, 6001
    cfg = W.make_config(k, n_segments=n)
    single = api.run_config(cfg)
    mp.spawn(_shard_rank, args=(2, _free_port(), k, n, str(tmp_path)), nprocs=2, join=True)
    red = np.load(os.path.join(str(tmp_path), "reduced.npz"))
    assert np.array_equal(red["hist"], single["hist"]) and np.array_equal(red["tel"], single["tel_counts"])
    for i, name in enumerate(api.COUNTER_NAMES):
        assert int(red["cnt"][i]) == single["counters"][name], name
    assert 0 < int(red["written_local"]) < single["counters"]["written"]


def test_substepping_counts_clipped_tracks_and_keeps_zero_length_tracks_finite():
    """c8ph_substep_plan never clips silently: tracks whose sagitta / step bounds ask for more than max_sub pieces are
    counted; a track of length 0 gives one finite piece of length 0 along its direction; max_sub is bounded."""
    n = 64
    cfg = W.make_config(4, n_segments=n)
    trk = {f: v.copy() for f, v in cfg["segments"].items() if f != "edep"}
    trk["len"][:] = 400.0
    trk["len"][:4] = 0.0
    trk["p_GeV"] = np.full(n, 0.01, np.float32)                       # 10 MeV/c in 45 uT: ~740 m radius
    ctx = api.setup_context(cfg)
    dev = {f: torch.from_numpy(v).cuda() for f, v in trk.items()}
    B = (2.0e-5, -0.5e-5, -4.3e-5)
    seg, off = ctx.substep_tracks(dev, n, B, 1e-4, max_sub=8)
    counts = np.diff(off.cpu().numpy())
    assert int(ctx.clipped_tracks.item()) == int((counts == 8).sum()) == n - 4
    assert np.all(counts[:4] == 1)
    for f in ("x", "y", "z", "dx", "dy", "dz", "len", "beta", "t0", "charge"):
        assert torch.isfinite(seg[f]).all(), f
    first = off[:4].cpu().numpy()
    assert np.all(seg["len"].cpu().numpy()[first] == 0.0)
    d = np.stack([seg[f].cpu().numpy()[first] for f in ("dx", "dy", "dz")], axis=1)
    want = np.stack([trk[f][:4] for f in ("dx", "dy", "dz")], axis=1).astype(np.float64)
    want /= np.linalg.norm(want, axis=1, keepdims=True)
    assert np.allclose(d, want, atol=1e-6)
    seg, off = ctx.substep_tracks(dev, n, B, 1e-4, max_sub=4096)
    assert int(ctx.clipped_tracks.item()) == 0
    with pytest.raises(api.C8phError) as e:
        ctx.substep_tracks(dev, n, B, 1e-4, max_sub=(1 << 20) + 1)
    assert e.value.code == api.E_ARG
