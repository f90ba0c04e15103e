"""Multi-GPU plumbing on CPU (-m "not gpu"): segments sharded by contiguous id range over
world_size-2 ``gloo`` ranks, per-rank results summed with ``shard.reduce_results``.

The per-rank compute here is the CPU oracle (tests may use it; the product path never does): what
is under test is the sharding contract of SURVEY 8(e) / DESIGN.md section 7 — a rank that is handed
segments [lo, hi) with seg_id_base = lo produces exactly the photons of the single run, so the
all-reduced histogram, telescope counters and event counters equal the single-run ones bit for bit
(integral bunch weights).
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2405_04229_b200 import shard, workloads as W
from paper_2405_04229_b200.api import COUNTER_NAMES


def test_plan_shards_covers_and_balances():
    for n, w in ((10, 3), (0, 2), (5, 8), (10_000_000, 8), (7, 1)):
        plan = shard.plan_shards(n, w)
        assert len(plan) == w and plan[0][0] == 0 and plan[-1][1] == n
        assert all(a[1] == b[0] for a, b in zip(plan, plan[1:]))
        sizes = [hi - lo for lo, hi in plan]
        assert max(sizes) - min(sizes) <= 1
        assert shard.shard_of(n, w - 1, w) == plan[-1]
    with pytest.raises(ValueError):
        shard.plan_shards(-1, 2)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _oracle_counters_tensor(cnt: dict) -> torch.Tensor:
    return torch.tensor([int(cnt.get(k, 0)) for k in COUNTER_NAMES], dtype=torch.int64)


def _rank_main(rank, world, port, k, n, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), OMP_NUM_THREADS="2")
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from oracle import c8ph_oracle as O
        cfg = W.make_config(k, n_segments=n)
        lo, hi = shard.shard_of(n, rank, world)
        sub = dict(cfg)
        sub["segments"] = W.slice_segments(cfg["segments"], lo, hi)
        sub["seg_id_base"] = lo
        res = O.run(sub, record=False)
        result = dict(hist=torch.from_numpy(np.asarray(res["hist"], dtype=np.float64).copy()),
                      tel_counts=torch.from_numpy(np.asarray(res["tel_counts"], dtype=np.float64).copy()),
                      counters=_oracle_counters_tensor(res["counters"]))
        # each rank's photon list stays local; only its length is kept aside by reduce_results
        result["counters"][COUNTER_NAMES.index("written")] = res["counters"]["tel_hit"]
        shard.reduce_results(result)
        t = shard.max_over_ranks(float(rank + 1))
        ssum = shard.sum_over_ranks(float(rank + 1))
        if rank == 0:
            np.savez(os.path.join(out_dir, "reduced.npz"), hist=result["hist"].numpy(),
                     tel=result["tel_counts"].numpy(), cnt=result["counters"].numpy(),
                     written_local=result["written_local"], tmax=t, tsum=ssum)
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("k,n", [(4, 240), (2, 3001)])
def test_two_gloo_ranks_reproduce_the_single_run(tmp_path, k, n):
    from oracle import c8ph_oracle as O
    O.build()
    cfg = W.make_config(k, n_segments=n)
    O.table_for(cfg)                                   # build once, the ranks read the cached table
    single = O.run(cfg, record=False)
    world = 2
    mp.spawn(_rank_main, args=(world, _free_port(), k, n, str(tmp_path)), nprocs=world, join=True)
    red = np.load(os.path.join(str(tmp_path), "reduced.npz"))
    assert np.array_equal(red["hist"], np.asarray(single["hist"], dtype=np.float64))
    assert np.array_equal(red["tel"], np.asarray(single["tel_counts"], dtype=np.float64))
    want = _oracle_counters_tensor(single["counters"]).numpy()
    got = red["cnt"]
    for name in ("segments", "seg_below_threshold", "seg_lv1", "seg_emitting", "emitted", "upgoing", "lv2",
                 "table_range", "roulette", "landed", "in_grid", "tel_hit"):
        i = COUNTER_NAMES.index(name)
        assert got[i] == want[i], name
    assert got[COUNTER_NAMES.index("written")] == single["counters"]["tel_hit"]
    assert 0 <= int(red["written_local"]) <= single["counters"]["tel_hit"]
    assert float(red["tmax"]) == 2.0 and float(red["tsum"]) == 3.0
