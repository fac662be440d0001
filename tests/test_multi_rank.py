"""world_size-2 gloo tests (CPU) of the multi-GPU host logic in paper_2408_13170_b200/dist.py."""
import os
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    from paper_2408_13170_b200 import dist as scd
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        out = {}
        # timing: max over ranks; work: sum over ranks (bench.py's reduction)
        out["tmax"] = scd.max_over_ranks(10.0 + rank)
        out["units"] = scd.sum_over_ranks(1000.0 * (rank + 1))
        # whole swarms per rank: no exchange
        out["shard4"] = scd.shard_swarms(40000, 4, rank, world)
        # one swarm split over both ranks: exchange of the best
        a, b, need = scd.shard_swarms(10000, 1, rank, world)
        out["shard1"] = (a, b, need)
        rng = np.random.default_rng(7)
        vals = np.round(rng.normal(0, 1, 10000), 1)                     # many ties
        pos = rng.random((10000, 8))
        li = a + int(np.argmax(vals[a:b]))                               # local arg max, lowest index
        v, i, p = scd.swarm_best_exchange(torch.tensor(vals[li]), li, torch.from_numpy(pos[li]))
        out["best"] = (v, i, p.numpy().tolist())
        out["want"] = (float(vals.max()), int(np.argmax(vals)), pos[int(np.argmax(vals))].tolist())
        out["tiles"] = scd.tiles_for_rank(7, rank, world)
        q.put((rank, out))
    finally:
        dist.destroy_process_group()


def test_two_rank_host_logic():
    world, port = 2, 29500 + os.getpid() % 2000
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = dict(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for r in range(world):
        o = res[r]
        assert o["tmax"] == 11.0 and o["units"] == 3000.0
        assert o["shard4"] == (r * 20000, (r + 1) * 20000, False)
        assert o["shard1"] == (r * 5000, (r + 1) * 5000, True)
        assert o["best"][0] == o["want"][0] and o["best"][1] == o["want"][1] and o["best"][2] == o["want"][2]
    assert sorted(res[0]["tiles"] + res[1]["tiles"]) == list(range(7))


def test_shard_validation():
    sys.path.insert(0, ROOT)
    from paper_2408_13170_b200 import dist as scd
    with pytest.raises(ValueError):
        scd.shard_swarms(10, 3, 0, 2)
    with pytest.raises(ValueError):
        scd.shard_swarms(30000, 3, 0, 2)
    assert scd.shard_swarms(40000, 4, 3, 4) == (30000, 40000, False)
    assert scd.shard_swarms(40000, 4, 5, 8) == (25000, 30000, True)
