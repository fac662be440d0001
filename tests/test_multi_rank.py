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


# ---------------------------------------------------------------------------------------------- sharded PSO step (host logic)
class _FakeHandle:
    """CPU stand-in for the three C-ABI calls dist.pso_step_sharded makes (sc_pso_best / sc_pso_pick / sc_pso_move), written
    with the oracle's uniforms: lets the gloo test check the ORCHESTRATION (offsets, gather order, groups) against the
    oracle's whole-population O7 step.  The CUDA kernels themselves are checked on the GPU (test_pso_step_sharded_...)."""

    def __init__(self, oracle):
        self.o = oracle

    def pso_best(self, state, stat, cand, n_swarms, index_offset=0, stream=None):
        P = state["pos"].shape[0]
        per = P // n_swarms
        upd = stat > state["pbest_val"]
        state["pbest_val"][upd] = stat[upd]
        state["pbest_pos"][upd] = state["pos"][upd]
        for s in range(n_swarms):
            v = state["pbest_val"][s * per:(s + 1) * per].numpy()
            i = int(np.argmax(v))                                     # first maximum = lowest index
            cand[s, 0] = float(v[i])
            cand[s, 1] = float(index_offset + s * per + i)
            cand[s, 2:] = state["pbest_pos"][s * per + i]

    def pso_pick(self, cand, state, stream=None):
        c = cand.numpy()
        for s in range(c.shape[1]):
            order = sorted(range(c.shape[0]), key=lambda r: (-c[r, s, 0], c[r, s, 1]))
            state["gbest_val"][s] = c[order[0], s, 0]
            state["gbest_pos"][s] = torch.from_numpy(c[order[0], s, 2:].copy())

    def pso_move(self, state, lo, hi, eps_min, omega, phi_p, phi_g, seed, it, n_swarms, index_offset=0, stream=None):
        pos, vel, pbp, gp = (state[k].numpy() for k in ("pos", "vel", "pbest_pos", "gbest_pos"))
        P = pos.shape[0]
        per = P // n_swarms
        for p in range(P):
            rP, rG = self.o.pso_uniforms(seed, index_offset + p, it)
            for m in range(8):
                th = pos[p, m]
                u = (omega * vel[p, m] + (phi_p * rP[m]) * (pbp[p, m] - th)) + (phi_g * rG[m]) * (gp[p // per, m] - th)
                au = abs(u)
                v = (max(eps_min[m], au) * (u / au)) if au > 0 else (eps_min[m] if eps_min[m] > 0 else 0.0)
                x = th + v
                if x < lo[m]:
                    x, v = lo[m], -v
                elif x > hi[m]:
                    x, v = hi[m], -v
                pos[p, m], vel[p, m] = x, v


def _sharded_worker(rank, world, port, q, n_swarms):
    sys.path.insert(0, ROOT)
    from oracle import sc_oracle as orc
    from paper_2408_13170_b200 import dist as scd
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        P = 240
        rng = np.random.default_rng(11)
        lo, hi = np.zeros(8), np.ones(8)
        pos, vel = rng.random((P, 8)), rng.uniform(-0.4, 0.4, (P, 8))
        eps = np.full(8, 0.01)
        a, b, need = scd.shard_swarms(P, n_swarms, rank, world)
        group = scd.make_swarm_group(n_swarms, rank, world)
        n_local = max(1, n_swarms // world)
        t = lambda x: torch.from_numpy(np.ascontiguousarray(x).copy())
        st = dict(pos=t(pos[a:b]), vel=t(vel[a:b]), pbest_pos=t(pos[a:b]), pbest_val=torch.full((b - a,), -np.inf, dtype=torch.float64),
                  gbest_pos=torch.zeros((n_local, 8), dtype=torch.float64), gbest_val=torch.zeros(n_local, dtype=torch.float64))
        ref = dict(pos=pos.copy(), vel=vel.copy(), pbp=pos.copy(), pbv=np.full(P, -np.inf), gp=np.zeros((n_swarms, 8)), gv=np.zeros(n_swarms))
        H = _FakeHandle(orc)
        ok = True
        for it in range(3):
            stat = np.round(rng.normal(50, 2, P), 0)                  # ties across shards
            scd.pso_step_sharded(H, st, t(stat[a:b]), lo, hi, eps, 0.5, 0.2, 0.3, 2408, it, n_local, a, group=group, exchange=need)
            orc.pso_step(ref["pos"], ref["vel"], ref["pbp"], ref["pbv"], stat, ref["gp"], ref["gv"], lo, hi, eps, 0.5, 0.2, 0.3, 2408, it, n_swarms)
            s0 = a // (P // n_swarms)
            ok = ok and np.array_equal(st["pos"].numpy(), ref["pos"][a:b]) and np.array_equal(st["vel"].numpy(), ref["vel"][a:b])
            ok = ok and np.array_equal(st["pbest_val"].numpy(), ref["pbv"][a:b])
            ok = ok and np.array_equal(st["gbest_val"].numpy(), ref["gv"][s0:s0 + n_local])
            ok = ok and np.array_equal(st["gbest_pos"].numpy(), ref["gp"][s0:s0 + n_local])
        q.put((rank, dict(ok=bool(ok), shard=(a, b, need))))
    except Exception as ex:                                           # report instead of leaving the parent to time out
        q.put((rank, dict(ok=False, shard=(0, 0, None), error=repr(ex))))
        raise
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("n_swarms", [1, 2, 4])
def test_pso_step_sharded_two_ranks(n_swarms):
    """One swarm cut over two ranks (exchange), two and four swarms on two ranks (whole swarms per rank, no exchange):
    every rank's shard after three iterations equals the oracle's whole-population O7 step bit for bit."""
    world, port = 2, 31500 + (os.getpid() + 7 * n_swarms) % 2000
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_sharded_worker, args=(r, world, port, q, n_swarms)) for r in range(world)]
    for p in procs:
        p.start()
    res = dict(q.get(timeout=180) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for r in range(world):
        assert res[r]["ok"], (r, res[r])
        assert res[r]["shard"][2] == (n_swarms < world)


def test_bench_spawns_its_own_ranks():
    """`python bench.py --gpus 2` with no launcher must start 2 ranks itself (torch.distributed.run on 127.0.0.1) and print
    n_gpus = 2 from rank 0 with max-over-ranks time and summed work; checked here on the CPU with the gloo self-test leg."""
    import json
    import subprocess
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--dist-selftest"], env=env,
                         capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [json.loads(ln) for ln in out.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1                                        # rank 0 alone prints
    assert lines[0]["n_gpus"] == 2 and lines[0]["ms_max"] == 11.0 and lines[0]["units"] == 40000.0
    assert lines[0]["shard0"] == [0, 20000, False]
