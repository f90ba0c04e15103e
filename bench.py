#!/usr/bin/env python
"""bench.py — propagated photons/s of the fused emit->trace->absorb->intersect->cut->bin path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 4]

Workload (N=1): BASELINE.json configs[4] — 1e7 synthetic 1 PeV-shower track segments, spherical
atmosphere, interpolation tracing, Rayleigh roulette, LV1+LV2 cuts, 10,000 telescope spheres +
1000x1000 ground histogram, fp32.  One "step" = one pass of the whole hot path over that batch:
zero the outputs, c8ph_emit_propagate, outputs left in HBM.  `value` = photons emitted and
propagated (post-LV1 bunches x bunch weight) per second of device time, inputs resident in HBM.
`e2e` = the same metric through c8ph_emit_propagate_host with pinned HOST buffers: H2D of the
segment arrays, the kernel, D2H of histogram, telescope counters, event counters and the
telescope-photon list, all inside the timed region.

N>1 (torchrun): weak scaling — every rank processes its own 1e7-segment batch with
seg_id_base = rank * 1e7 (independent segment ids => independent photons); no data-path collective;
time = max over ranks, value = photons of all ranks / that time.

--impl reference times the CPU oracle (oracle/, test infrastructure, as it stands) on the host
cores on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "propagated photons/sec"
UNIT = "photons/s"

# Roofline numerator 1 (`roofline.frac`): SURVEY.md section 8(d) "Algorithmic work per photon", an estimate made from the
# method's arithmetic BEFORE any kernel existed: Philox4x32-10 40, uniforms 8, wavelength 3, emission point / height 14,
# n(h_e) 6, cone angle 8, sincos 4, direction 12, straight line 14, LV2 + lattice index 20, zenith + acos 18, bilinear
# float4 lookup 25, apply + arrival angle + time 22, transmission + roulette 10, ray-sphere 14, bin + RED 8, compaction 6,
# loop / predicates 15 = 250 thread-instructions per emitted photon (+- 40).  Independent of this implementation.
I_ALG_SURVEY_PER_PHOTON = 250.0

# Roofline numerator 2 (`roofline.frac_own_audit`): instructions one unit of each stage executes on its way through THIS
# kernel, k_emit_propagate<CHERENKOV,TABLE,SPH,SPEC=1>, derived by tests/roofline_audit.py from the committed ncu source
# page profiles/r2_cfg4_source.csv.gz (tests/test_roofline_audit.py checks these numbers against it).  Not counted: the
# loop slot, the queue push, LV2 list walks, candidates that miss, partly filled drains, idle lanes.
I_ALG_OWN = {
    "segment": 1127.2,    # a1-a4: SoA ingest, fp64 yield / LV1 / Rodrigues / anchor, slot store (per segment)
    "emitted": 215.0,     # a5-a12: Philox4x32-10, uniforms, emission point, n(h), cone, sincos, straight line, LV2 box, zenith,
                          #         acos, bilinear float4 lookup, transmission, roulette
    "landed": 50.0,       # a15 + a14 pre-test: corrected position, telescope-grid cell + smallest key, bin index
    "in_grid": 6.0,       # a15: bin address + RED.ADD.F32
    "tel_hit": 160.0,     # a13/a14/a16: finish() (time, arrival direction, sphere search, record), once per hit
}


# dram__bytes_read.sum + dram__bytes_write.sum of one k_emit_propagate launch on the N=1 workload, from the
# ncu --set full capture summarised in profiles/r2_cfg4_final.md.  Reported as `roofline.traffic` only when the run is
# that workload (cfg4, 1e7 segments); otherwise null.
NCU_TRAFFIC_BYTES_CFG4 = 0.721679872e9 + 5.245904e9
NCU_ISSUE_SLOTS_BUSY_CFG4 = 0.7553                 # smsp issue slots busy of the same capture


def _stage_population(cnt: dict) -> dict:
    return {"segment": cnt["segments"], "emitted": cnt["emitted"], "landed": cnt["landed"],
            "in_grid": cnt["in_grid"], "tel_hit": cnt["tel_hit"]}


def algorithmic_instructions(cnt: dict) -> float:
    pop = _stage_population(cnt)
    return float(sum(I_ALG_OWN[k] * pop[k] for k in I_ALG_OWN))


def algorithmic_bytes(cnt: dict, n_hist: int, n_tel: int) -> float:
    """HBM bytes the path must move: 40 B/segment in, 32 B/written photon out, outputs once."""
    return 40.0 * cnt["segments"] + 32.0 * cnt["written"] + 4.0 * (n_hist + n_tel) * 2


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "50"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self) -> dict:
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.12)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        self.t.join(timeout=2)
        sm, mx, pw, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for r in self.rows:
            if len(r) < 9:
                continue
            try:
                sm.append(float(r[1])); mx.append(float(r[2])); pw.append(float(r[3]))
            except ValueError:
                continue
            for n, v in zip(names, r[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "power_w": float(np.median(pw)),
                "samples": len(sm), "reasons": sorted(reasons)}


def _dist_env():
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, world, local


def _workload_name(k: int, n: int) -> str:
    return f"cfg{k}: BASELINE configs[{k}], {n} segments/GPU"


# ------------------------------------------------------------------------------------------ CPU legs
def _oracle_rate(cfg, n_seg: int, threads=None):
    """Oracle (as it stands) on the first n_seg segments: (photons, seconds, cores)."""
    from oracle import c8ph_oracle as O
    from paper_2405_04229_b200 import workloads as W
    sub = dict(cfg)
    sub["segments"] = W.slice_segments(cfg["segments"], 0, n_seg)
    t0 = time.perf_counter()
    res = O.run(sub, record=False, threads=threads)
    dt = time.perf_counter() - t0
    return res["counters"]["emitted"] * float(cfg["params"]["bunch_weight"]), dt


def _oracle_setup(cfg):
    from oracle import c8ph_oracle as O
    O.build()
    if cfg.get("table") is not None:
        O.table_for(cfg)                       # built once per atmosphere, not timed
    cores = len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)
    return cores


def _cpu_model() -> str:
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def cpu_baseline(cfg, target_s: float = 12.0) -> dict:
    """The oracle as it stands (unoptimised fp64 test oracle: e.g. brute force over all telescopes per landed photon)
    on a prefix of the workload: all host cores (`value`) and one thread (`single_thread`).  A stated baseline, not a
    tuned CPU implementation."""
    cores = _oracle_setup(cfg)
    n_total = len(cfg["segments"]["x"])
    n0 = min(n_total, 400)
    ph0, dt0 = _oracle_rate(cfg, n0)
    rate0 = ph0 / max(dt0, 1e-9)
    per_seg = ph0 / n0
    n1 = int(min(n_total, max(n0, target_s * rate0 / max(per_seg, 1e-9))))
    ph, dt = _oracle_rate(cfg, n1)
    n2 = int(min(n_total, max(100, n1 // max(cores, 1) // 2)))          # ~ half that time on one thread
    ph1, dt1 = _oracle_rate(cfg, n2, threads=1)
    return {"value": ph / dt, "unit": UNIT, "cores": cores, "kind": "oracle", "cpu_model": _cpu_model(),
            "sample": f"first {n1} segments of the workload ({int(ph)} photons, {dt:.1f} s, fp64, OpenMP over segments)",
            "single_thread": {"value": ph1 / dt1, "unit": UNIT, "cores": 1,
                              "sample": f"first {n2} segments ({int(ph1)} photons, {dt1:.1f} s)"},
            "note": "unoptimised fp64 test oracle; the ratio to it says nothing about kernel quality"}


def run_reference(args):
    rank, world, _ = _dist_env()
    if rank != 0:
        return 0
    from paper_2405_04229_b200 import workloads as W
    k = args.config
    n_full = W.FULL_SEGMENTS[k] if args.segments is None else args.segments
    # the sample is a prefix of the workload's segment list; generating 2e5 segments is enough
    cfg = W.make_config(k, n_segments=min(n_full, 200000))
    cores = _oracle_setup(cfg)
    ph0, dt0 = _oracle_rate(cfg, min(400, len(cfg["segments"]["x"])))
    per_seg = ph0 / min(400, len(cfg["segments"]["x"]))
    n_step = int(min(len(cfg["segments"]["x"]), max(400, 5.0 * (ph0 / dt0) / max(per_seg, 1e-9))))
    for _ in range(args.warmup):
        _oracle_rate(cfg, min(n_step, 400))
    tot_ph, tot_t = 0.0, 0.0
    for _ in range(args.steps):
        ph, dt = _oracle_rate(cfg, n_step)
        tot_ph += ph
        tot_t += dt
    val = tot_ph / tot_t
    sample = f"first {n_step} segments of the workload per step ({int(tot_ph / args.steps)} photons), fp64, OpenMP"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": _workload_name(k, n_full), "sample_segments_per_step": n_step},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


def _apply_variant(cfg: dict, variant: str) -> None:
    """Optional features (R13-R15, R17, R19) on top of a BASELINE config."""
    if variant == "flat":
        cfg["params"].update(flat_plane=1)
    elif variant == "flattab":
        cfg["params"].update(flat_plane=2)
        cfg["table"] = dict(cfg["table"], n_rho=16, rho_max_m=30000.0)
    elif variant == "extinction":
        # a tau_v(lambda, h) table filled from the Rayleigh law of the config on a 10 nm grid
        atm = cfg["atmosphere"]
        lam = np.arange(240.0, 711.0, 10.0)
        xv = atm["overburden"].astype(np.float64)
        h = atm["h0"] + atm["dh"] * np.arange(atm["n_nodes"])
        xg = np.interp(atm["h_obs"], h, xv)
        tau = np.outer((atm["rayleigh_lambda"] / lam) ** 4 / atm["rayleigh_X"], np.maximum(xg - xv, 0.0))
        atm.update(ext_lambda0_nm=float(lam[0]), ext_dlambda_nm=10.0, ext_tau_v=tau.astype(np.float32))
    elif variant == "dispersion":
        cfg["params"].update(disp_b_nm2=5700.0, disp_lambda0_nm=400.0)
    elif variant == "efficiency":
        lam = np.arange(200.0, 801.0, 10.0)
        cfg["params"].update(eff=(0.85 * np.exp(-0.5 * ((lam - 420.0) / 90.0) ** 2)).astype(np.float32),
                             eff_lambda0_nm=200.0, eff_dlambda_nm=10.0)
    elif variant == "optics":
        tel = cfg["detector"]["tel_xyzr"].copy()
        tel[:, 3] = 12.0
        cfg["detector"]["tel_xyzr"] = tel
        cfg["detector"].update(opt_enabled=True, opt_az_deg=0.0, opt_el_deg=70.0, opt_focal_m=17.0,
                               opt_mirror_radius_m=8.5, opt_camera_radius_m=0.735)


def run_substep(args):
    """Throughput of the sub-stepping entry points (row f2) on synthetic tracks: cfg4's segment recipe
    with track lengths 5-400 m and momenta 10 MeV - 10 GeV in a 45 uT field, 1 cm sagitta."""
    import torch
    from paper_2405_04229_b200 import api, build, workloads as W
    build.build()
    n = args.substep
    cfg = W.make_config(4, n_segments=n)
    rng = np.random.default_rng(7)
    trk = {kk: v for kk, v in cfg["segments"].items() if kk != "edep"}
    trk["len"] = rng.uniform(5.0, 400.0, n).astype(np.float32)
    trk["p_GeV"] = (10 ** rng.uniform(-2.0, 1.0, n)).astype(np.float32)
    ctx = api.setup_context(W.make_config(4 if args.substep_ms is not None else 0, n_segments=1))
    dev = {kk: torch.from_numpy(v).cuda() for kk, v in trk.items()}
    B, tol = (2.0e-5, -0.5e-5, -4.3e-5), 0.01
    ms = []
    for i in range(args.warmup + args.steps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        seg, off = ctx.substep_tracks(dev, n, B, tol, ms_max_step_m=args.substep_ms)
        e1.record()
        torch.cuda.synchronize()
        if i >= args.warmup:
            ms.append(e0.elapsed_time(e1))
    pieces = int(off[-1].item())
    t = float(np.median(ms)) * 1e-3
    print(json.dumps({"metric": "sub-stepped tracks/sec", "value": n / t, "unit": "tracks/s", "pieces_per_s": pieces / t,
                      "tracks": n, "pieces": pieces, "multiple_scattering_step_m": args.substep_ms, "ms": 1e3 * t, "steps": args.steps, "warmup": args.warmup,
                      "note": "plan (3 kernels) + 8-byte D2H of the total + allocation + fill (1 kernel), CUDA events",
                      "alg_bytes": 44 * n + 8 * (n + 1) + 40 * pieces, "gpu_launches": 4 * args.steps}), flush=True)
    return 0


# ------------------------------------------------------------------------------------------ GPU arm
def run_ours(args):
    import torch
    rank, world, local = _dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    # one rank per GPU; C8PH_BENCH_BACKEND=gloo lets the N>1 plumbing be exercised on a box with fewer GPUs
    # than ranks (ranks then share devices; a plumbing check, not a measurement)
    backend = os.environ.get("C8PH_BENCH_BACKEND", "nccl")
    local = local % torch.cuda.device_count()
    red_dev = f"cuda:{local}" if backend == "nccl" else "cpu"
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        if backend == "nccl":
            dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
        else:
            dist.init_process_group(backend)
    from paper_2405_04229_b200 import api, build, shard, workloads as W
    if rank == 0:
        build.build()
    if dist:
        dist.barrier()
    k = args.config
    n = W.FULL_SEGMENTS[k] if args.segments is None else args.segments
    cfg = W.make_config(k, n_segments=n)
    _apply_variant(cfg, args.variant)
    n_total = n
    if args.scaling == "strong" and world > 1:
        # ONE shower sharded over the ranks by contiguous id range: total work fixed
        lo, hi = shard.shard_of(n_total, rank, world)
        cfg["segments"] = W.slice_segments(cfg["segments"], lo, hi)
        n, seg_id_base = hi - lo, lo
    else:
        seg_id_base = rank * n                           # weak scaling: disjoint segment ids per rank
    ctx = api.setup_context(cfg, device=local)
    par, seed = cfg["params"], cfg["seed"]
    w = float(par["bunch_weight"])
    seg_host = {f: v for f, v in cfg["segments"].items() if not (f == "edep" and par["emit"] == "cherenkov")}
    seg_dev = api.segments_to_device(seg_host, local)

    # size the photon list from a first (warm-up) pass with a generous bound
    cap = int(args.photon_capacity)
    out = api.alloc_device_outputs(ctx, cap, False, local)

    def zero(o):
        o["hist"].zero_(); o["tel_counts"].zero_(); o["counters"].zero_()

    def exchange(o):
        """The one exchange step of the sharded path: SUM all-reduce of histogram, telescope
        counters and event counters; NCCL on the launch stream (gloo: through host copies, plumbing check only)."""
        if not dist:
            return o
        if backend == "nccl":
            return shard.reduce_results(o)
        host = {kk: o[kk].cpu() for kk in ("hist", "tel_counts", "counters")}
        shard.reduce_results(host)
        for kk, v in host.items():
            if kk != "written_local" and hasattr(v, "shape"):
                o[kk].copy_(v)
        return o

    def step():
        zero(out)
        ctx.emit_propagate(seg_dev, n, seg_id_base, par, seed, out)

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    cnt = {kk: int(v) for kk, v in zip(api.COUNTER_NAMES, out["counters"].cpu().numpy())}
    if cnt["overflow"]:
        raise SystemExit(f"bench.py: photon list overflow ({cnt['overflow']}); raise --photon-capacity")
    if dist:
        exchange(out)                                    # warm-up of the collective (communicator set-up)

    # ---- timed region: K steps, device-resident inputs (400 MB of segments > 126 MB L2)
    sampler = ClockSampler(local)
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(args.steps)]
    launches0 = ctx.launch_count()
    if dist:
        dist.barrier()
    torch.cuda.synchronize()
    sampler.start()
    t_wall = time.perf_counter()
    for s in range(args.steps):
        ev[s][0].record()
        zero(out)
        ev[s][1].record()
        ctx.emit_propagate(seg_dev, n, seg_id_base, par, seed, out)
        ev[s][2].record()
        exchange(out)
        ev[s][3].record()
    torch.cuda.synchronize()
    t_wall = time.perf_counter() - t_wall
    clocks = sampler.stop()
    if dist:
        dist.barrier()
    # our kernels inside the timed region (the library's own count) + torch's three fill kernels per step
    gpu_launches = int(ctx.launch_count() - launches0) + 3 * args.steps
    total_ms = ev[0][0].elapsed_time(ev[-1][3])
    kern_ms = [e[1].elapsed_time(e[2]) for e in ev]
    exch_ms = float(np.mean([e[2].elapsed_time(e[3]) for e in ev])) if dist else 0.0
    total_ms = shard.max_over_ranks(total_ms, red_dev)
    photons_rank = cnt["emitted"] * w
    photons_job = shard.sum_over_ranks(photons_rank, red_dev)
    value = photons_job * args.steps / (total_ms * 1e-3)
    # checksum of the (reduced) result: N = 1 and a strong-scaling run at any N give the same bits (integral weights)
    import zlib
    hist_host = out["hist"].cpu().numpy()
    checksum = {"hist_sum": float(hist_host.astype(np.float64).sum()), "hist_crc32": int(zlib.crc32(hist_host.tobytes())),
                "tel_sum": float(out["tel_counts"].double().sum().item())}

    # ---- roofline of the one kernel of the step (ALU issue bound)
    props = torch.cuda.get_device_properties(local)
    n_sm = props.multi_processor_count
    k_ms = float(np.mean(kern_ms))
    i_own = algorithmic_instructions(cnt)
    i_survey = I_ALG_SURVEY_PER_PHOTON * cnt["emitted"]
    sm_max = clocks.get("sm_max_mhz") or 1965.0
    peak = n_sm * 128 * sm_max * 1e6 / 1e9                # G thread-inst/s at clocks.max.sm
    achieved = i_survey / (k_ms * 1e-3) / 1e9
    achieved_own = i_own / (k_ms * 1e-3) / 1e9
    peaks_file = os.path.join(ROOT, "MEASURED_PEAKS.json")
    hbm_peak, peak_src = 6650.0, "fallback"
    if os.path.exists(peaks_file):
        try:
            hbm_peak, peak_src = float(json.load(open(peaks_file))["hbm_gbs"]), "measured"
        except Exception:
            pass
    alg_bytes = algorithmic_bytes(cnt, ctx.n_hist(), ctx._n_tel)
    headline = (k == 4 and n == W.FULL_SEGMENTS[4] and args.variant == "base")
    roofline = {"bound": "alu", "kernel": "k_emit_propagate", "achieved": achieved, "peak": peak,
                "unit": "Ginst/s", "frac": achieved / peak,
                "numerator": "SURVEY 8(d): 250 thread-instructions per emitted photon (implementation-independent estimate)",
                "frac_own_audit": achieved_own / peak, "achieved_own_audit": achieved_own,
                "own_audit_inst_per_photon": i_own / max(cnt["emitted"], 1),
                "own_audit": "tests/roofline_audit.py on profiles/r2_cfg4_source.csv.gz (stage counts of this kernel's SASS)",
                "issue_slots_busy_ncu": NCU_ISSUE_SLOTS_BUSY_CFG4 if headline else None,
                "traffic": NCU_TRAFFIC_BYTES_CFG4 if headline else None,
                "traffic_unit": "bytes per launch (ncu dram read+write); algorithmic bytes = %.4g" % alg_bytes,
                "peak_def": f"{n_sm} SMs x 4 schedulers x 32 lanes x clocks.max.sm {sm_max:.0f} MHz (issue slots)",
                "frac_at_measured_clock": (achieved / (n_sm * 128 * clocks["sm_mhz"] * 1e-3)) if clocks.get("sm_mhz") else None,
                "kernel_ms": k_ms,
                "hbm": {"achieved": alg_bytes / (k_ms * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s",
                        "frac": alg_bytes / (k_ms * 1e-3) / 1e9 / hbm_peak, "peak_source": peak_src,
                        "alg_bytes_per_photon": alg_bytes / max(cnt["emitted"], 1)}}

    # ---- e2e: HOST buffers through c8ph_emit_propagate_host (pinned memory), copies inside the timed region
    e2e = None
    if not args.no_e2e:
        pin = {f: torch.from_numpy(np.ascontiguousarray(v)).pin_memory() for f, v in seg_host.items()}
        cap_h = int(cnt["written"] * 1.02) + 1024
        hout = dict(hist=torch.zeros(max(ctx.n_hist(), 1), dtype=torch.float32).pin_memory().numpy()[:ctx.n_hist()],
                    tel_counts=torch.zeros(max(ctx._n_tel, 1), dtype=torch.float32).pin_memory().numpy()[:ctx._n_tel],
                    photons=torch.zeros((cap_h, 32), dtype=torch.uint8).pin_memory().numpy().view(api.PHOTON_DTYPE).reshape(-1),
                    photon_weight=None, counters_raw=np.zeros(api.N_COUNTERS, dtype=np.uint64))
        del out
        torch.cuda.empty_cache()
        e_steps = max(1, min(args.steps, args.e2e_steps))
        ctx.emit_propagate_host(pin, n, seg_id_base, par, seed, out=hout)          # warm-up (allocates the arena)
        if dist:
            dist.barrier()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(e_steps):
            res = ctx.emit_propagate_host(pin, n, seg_id_base, par, seed, out=hout)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        dt = shard.max_over_ranks(dt, red_dev)
        h2d = sum(int(v.numel()) * 4 for v in pin.values())
        d2h = 4 * (ctx.n_hist() + ctx._n_tel) + 8 * api.N_COUNTERS + 32 * res["counters"]["written"]
        assert res["counters"]["emitted"] == cnt["emitted"] and res["counters"]["overflow"] == 0
        e2e = {"value": photons_job * e_steps / dt, "unit": UNIT, "h2d_bytes_per_step": h2d,
               "d2h_bytes_per_step": d2h, "steps": e_steps, "ms_per_step": 1e3 * dt / e_steps,
               "hist_checksum": float(res["hist"].sum())}

    if rank != 0:
        if dist:
            dist.destroy_process_group()
        return 0
    base = None if args.no_cpu_baseline or world > 1 else cpu_baseline(
        W.make_config(k, n_segments=min(n, 200000)))
    bad = [r for r in clocks.get("reasons", []) if r in ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown")]
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": total_ms / args.steps, "higher_is_better": True,
            "scaling": args.scaling if world > 1 else "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": _workload_name(k, n_total) + ("" if args.variant == "base" else f" + {args.variant}"), "segments_per_gpu": n, "photons_per_step_per_gpu": photons_rank,
                       "landed": cnt["landed"], "in_grid": cnt["in_grid"], "tel_hit": cnt["tel_hit"], "written": cnt["written"],
                       "l2": f"inputs ({40 * n / 1e6:.0f} MB of segments) and photon list ({32 * cnt['written'] / 1e9:.2f} GB) vs 126 MB L2; outputs re-zeroed each step",
                       "parallelism": (f"segments sharded over {world} ranks by id range ({args.scaling}), results SUM all-reduced "
                                       f"each step ({backend})") if world > 1 else "1 GPU"},
            "counters": cnt, "clocks": clocks, "clock_rejected": bool(bad),
            "e2e": e2e, "gpu_launches": gpu_launches, "roofline": roofline, "cpu_baseline": base,
            "exchange_ms_per_step": exch_ms, "result_checksum": checksum,
            "wall_ms_per_step": 1e3 * t_wall / args.steps}
    print(json.dumps(line), flush=True)
    if dist:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=("ours", "reference"), default="ours")
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--scaling", choices=("weak", "strong"), default="weak",
                    help="N > 1: weak = every rank its own full batch (default, the driver's contract); strong = ONE batch sharded "
                         "by contiguous segment-id range (SURVEY 8(e)); both end each step with the SUM all-reduce of the results")
    ap.add_argument("--segments", type=int, default=None, help="override the segment count (debugging only)")
    ap.add_argument("--photon-capacity", type=int, default=220_000_000)
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--variant", choices=("base", "generic", "flat", "flattab", "extinction", "dispersion", "efficiency", "optics"), default="base",
                    help="optional features of SURVEY 8(f) switched on (generic kernel variant); the headline is 'base'")
    ap.add_argument("--substep", type=int, default=0, help="time c8ph_substep_plan + c8ph_substep_fill on this many tracks and exit")
    ap.add_argument("--substep-ms", type=float, default=None, metavar="STEP_M",
                    help="with --substep: multiple-scattering pieces of at most STEP_M metres (DESIGN.md R18)")
    args = ap.parse_args()
    if args.variant == "generic":                                     # same switches as 'base' through the generic kernel variant
        os.environ["C8PH_FORCE_GENERIC"] = "1"
    if args.substep:
        return run_substep(args)
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
