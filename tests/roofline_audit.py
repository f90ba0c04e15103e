#!/usr/bin/env python
"""Audit of the per-stage instruction counts behind bench.py's `roofline.frac_own_audit`.

    python tests/roofline_audit.py [profiles/r2_cfg4_source.csv.gz] [profiles/r2_cfg4_bench.json]

Input 1 is `ncu -i <report> --page source --csv` of ONE launch of k_emit_propagate<CHERENKOV,TABLE,SPH,SPEC=1> on
BASELINE configs[4] (per SASS instruction: warp-level and thread-level execution counts and stall samples; the command
that made it is in profiles/r2_cfg4_final.md).  Input 2 is the bench.py line of the same build, whose event counters give
the stage populations (emitted, landed, in-grid, telescope hits, segments).

An instruction belongs to a stage when the number of THREADS that executed it equals the stage's population: every
emitted photon executes the instructions of a5-a12 exactly once, every landed photon those of the landed stage, and so
on; nothing else in the kernel has those counts.  finish() runs once per batch of up to 32 queued telescope candidates
with all 32 lanes on: its instructions are the ones with 32 active lanes whose warp-level count is the number of batches.
What is NOT a stage of the method (and is not counted as algorithmic work): the loop slot (iteration counter, photon
index, queue-full vote: executed once per warp iteration with all 32 lanes), the queue push, drains of partly filled
batches, LV2 list walks, candidates that miss, idle lanes.

Output: the class table of profiles/r2_cfg4_final.md and the dictionary bench.py carries as I_ALG_OWN
(tests/test_roofline_audit.py checks that the two agree).
"""
from __future__ import annotations

import csv
import gzip
import io
import json
import os
import sys
from collections import Counter

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
DEFAULT_CSV = os.path.join(ROOT, "profiles", "r2_cfg4_source.csv.gz")
DEFAULT_BENCH = os.path.join(ROOT, "profiles", "r2_cfg4_bench.json")


def read_source_csv(path: str):
    """Rows of the ncu source page: (sass, warp_count, thread_count, samples)."""
    opener = gzip.open if path.endswith(".gz") else open
    with opener(path, "rt") as f:
        text = f.read()
    text = text.split("\n", 1)[1]                       # first line: kernel name
    rows = []
    for r in csv.DictReader(io.StringIO(text)):
        rows.append((r["Source"].strip(), int(r["Instructions Executed"]), int(r["Thread Instructions Executed"]),
                     int(r["# Samples"])))
    return rows


def audit(rows, pop: dict) -> dict:
    """pop: segments, emitted, landed, in_grid, tel_hit (event counters of the launch)."""
    warp_total = sum(r[1] for r in rows)
    thread_total = sum(r[2] for r in rows)
    # warp iterations of the photon loop: the warp-level count that carries the most thread instructions
    by_count = Counter()
    for _, w, t, _ in rows:
        by_count[w] += t
    iters = by_count.most_common(1)[0][0]

    def n_with_threads(lo, hi):
        return sum(1 for r in rows if r[1] > 0 and lo - 2 <= r[2] <= hi + 2)

    # a5-a12: executed by every emitted photon, or by every emitted photon that is still alive after the up-going cut,
    # the LV2 test and the table-range check (all of them reach the roulette): thread count between landed + roulette
    # and emitted
    emitted = n_with_threads(pop["landed"] + pop["roulette"], pop["emitted"])
    landed = n_with_threads(pop["landed"], pop["landed"])
    in_grid = n_with_threads(pop["in_grid"], pop["in_grid"])
    loop_slot = sum(1 for r in rows if r[1] == iters and r[2] == 32 * iters)
    # finish(): full-warp instructions executed once per batch of queued candidates
    full = Counter(r[1] for r in rows if r[1] > 0 and r[2] == 32 * r[1] and iters // 100 < r[1] < iters // 2)
    batches, finish = full.most_common(1)[0] if full else (0, 0)
    # segment preparation: everything executed less than once per 100 warp iterations, per segment
    seg_threads = sum(r[2] for r in rows if 0 < r[1] < iters // 100)
    segment = seg_threads / max(pop["segments"], 1)
    own = {"segment": round(segment, 1), "emitted": emitted, "landed": landed, "in_grid": in_grid, "tel_hit": finish}
    alg = (own["segment"] * pop["segments"] + emitted * pop["emitted"] + landed * pop["landed"] + in_grid * pop["in_grid"] +
           finish * pop["tel_hit"])
    # class table: (executions per warp iteration, active lanes) -> instructions, thread instructions per emitted photon
    classes = Counter()
    thr = Counter()
    for _, w, t, _ in rows:
        if w == 0:
            continue
        key = (round(w / iters, 2), round(t / w, 1))
        classes[key] += 1
        thr[key] += t
    table = sorted(((thr[k] / pop["emitted"], k, classes[k]) for k in classes), reverse=True)
    return {"iterations": iters, "finish_batches": batches, "loop_slot": loop_slot, "own": own,
            "alg_thread_inst": alg, "alg_per_emitted": alg / pop["emitted"],
            "executed_thread_inst_per_emitted": thread_total / pop["emitted"],
            "issued_lane_slots_per_emitted": 32.0 * warp_total / pop["emitted"],
            "warp_inst_per_iteration": warp_total / iters, "sass_instructions": len(rows), "table": table}


def populations(bench_line: dict) -> dict:
    c = bench_line["counters"]
    return {k: int(c[k]) for k in ("segments", "emitted", "upgoing", "lv2", "table_range", "roulette", "landed", "in_grid", "tel_hit")}


def main(argv):
    src = argv[1] if len(argv) > 1 else DEFAULT_CSV
    bench = argv[2] if len(argv) > 2 else DEFAULT_BENCH
    pop = populations(json.load(open(bench)))
    a = audit(read_source_csv(src), pop)
    print(f"SASS instructions {a['sass_instructions']}, warp iterations {a['iterations']}, finish() batches {a['finish_batches']}")
    print(f"warp instructions per iteration {a['warp_inst_per_iteration']:.1f}; per emitted photon: issued lane slots "
          f"{a['issued_lane_slots_per_emitted']:.1f}, executed thread instructions {a['executed_thread_inst_per_emitted']:.1f}, "
          f"algorithmic (own audit) {a['alg_per_emitted']:.1f}")
    print("I_ALG_OWN =", a["own"], " loop slot (not counted):", a["loop_slot"])
    print("| executions per warp iteration | active lanes | SASS instructions | thread instructions per emitted photon |")
    print("|---|---|---|---|")
    rest = 0.0
    for i, (t, (x, lanes), n) in enumerate(a["table"]):
        if i < 16:
            print(f"| {x:.2f} | {lanes:.1f} | {n} | {t:.2f} |")
        else:
            rest += t
    print(f"| (all other classes) | | | {rest:.2f} |")
    return 0


if __name__ == "__main__":
    sys.exit(main(sys.argv))
