"""bench.py's own-audit stage counts are what tests/roofline_audit.py derives from the committed ncu source page
(profiles/r2_cfg4_source.csv.gz) and the bench line of the same build (profiles/r2_cfg4_bench.json)."""
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import bench                                                          # noqa: E402
import roofline_audit as RA                                           # noqa: E402


def test_own_audit_counts_follow_from_the_committed_profile():
    line = json.load(open(RA.DEFAULT_BENCH))
    pop = RA.populations(line)
    a = RA.audit(RA.read_source_csv(RA.DEFAULT_CSV), pop)
    assert a["own"] == {k: (round(v, 1) if k == "segment" else int(v)) for k, v in bench.I_ALG_OWN.items()}
    # the bench line's fractions follow from its own inputs
    r = line["roofline"]
    peak = 148 * 128 * 1965.0e6 / 1e9
    assert abs(r["peak"] - peak) < 1e-6 * peak
    own = sum(v * pop["segments" if k == "segment" else k] for k, v in bench.I_ALG_OWN.items())
    assert abs(r["frac_own_audit"] - own / (r["kernel_ms"] * 1e-3) / 1e9 / peak) < 2e-3
    assert abs(r["frac"] - bench.I_ALG_SURVEY_PER_PHOTON * pop["emitted"] / (r["kernel_ms"] * 1e-3) / 1e9 / peak) < 1e-9
    # sanity of the classes: algorithmic <= executed <= issued lane slots, loop slot and queue push excluded
    assert a["alg_per_emitted"] < a["executed_thread_inst_per_emitted"] < a["issued_lane_slots_per_emitted"]
    assert r["frac"] <= r["frac_own_audit"] <= r["issue_slots_busy_ncu"] <= 1.0
