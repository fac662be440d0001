"""Multi-GPU plumbing: one process per GPU, torch.distributed for the few scalars that cross ranks.

The statistic shards over independent problems ("This can be done in parallel",
PAPER.md:365-367 one GPU per tile): every rank owns whole tiles or whole swarms, the whitened data is replicated,
and the data path has NO collective.  The only exchange that can ever be needed is the swarm best when ONE swarm is
split over ranks: a (value, global index) arg-max plus the 64-byte winning position -- latency-bound, done here with
an all-gather of 10 doubles per rank and swarm (pso_step_sharded: sc_pso_best -> all-gather -> sc_pso_pick -> sc_pso_move,
everything on the device and on the stream, no host synchronisation).  Works on NCCL (GPU tensors) and gloo (CPU tensors).
"""
import torch
import torch.distributed as dist


def tiles_for_rank(n_tiles, rank, world):
    """Round-robin assignment of independent search tiles to ranks."""
    return list(range(rank, n_tiles, world))


def shard_swarms(n_particles, n_swarms, rank, world):
    """Contiguous particle range [start, stop) of this rank.  Whole swarms per rank when n_swarms >= world (no exchange
    needed); otherwise each swarm is cut into world/n_swarms equal pieces (needs swarm_best_exchange)."""
    if n_particles % n_swarms:
        raise ValueError("n_particles must be a multiple of n_swarms")
    per = n_particles // n_swarms
    if n_swarms >= world:
        if n_swarms % world:
            raise ValueError("n_swarms must be a multiple of the world size")
        k = n_swarms // world
        return rank * k * per, (rank + 1) * k * per, False
    if world % n_swarms or per % (world // n_swarms):
        raise ValueError("world size must split every swarm evenly")
    pieces = world // n_swarms
    piece = per // pieces
    return rank * piece, (rank + 1) * piece, True


def max_over_ranks(value, device=None):
    """Device-timed durations are reported as the max over ranks."""
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    if dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return t.item()


def sum_over_ranks(value, device=None):
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    if dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return t.item()


def swarm_best_exchange(local_val, local_idx, local_pos, group=None):
    """Swarm best over the ranks of `group` that share one swarm: arg max of value, lowest GLOBAL particle index on ties
    (the rule of sc_pso_step).  local_val: 0-d tensor, local_idx: global index (int), local_pos: [8] tensor.
    Returns (val, idx, pos)."""
    world = dist.get_world_size(group)
    pack = torch.empty(10, dtype=torch.float64, device=local_pos.device)
    pack[0] = local_val
    pack[1] = float(local_idx)
    pack[2:] = local_pos
    allp = [torch.empty_like(pack) for _ in range(world)]
    dist.all_gather(allp, pack, group=group)
    best = None
    for p in allp:
        v, i = p[0].item(), int(p[1].item())
        if best is None or v > best[0] or (v == best[0] and i < best[1]):
            best = (v, i, p[2:].clone())
    return best


def swarm_groups(n_swarms, world):
    """Ranks that share a swarm when swarms are cut over ranks (n_swarms < world): [[ranks of swarm 0], ...].  Every rank
    must create every group (torch.distributed.new_group is collective): see make_swarm_group."""
    pieces = world // n_swarms
    return [list(range(s * pieces, (s + 1) * pieces)) for s in range(n_swarms)]


def make_swarm_group(n_swarms, rank, world):
    """The process group of the ranks sharing this rank's swarm (None when every rank owns whole swarms)."""
    if n_swarms >= world:
        return None
    mine = None
    for ranks in swarm_groups(n_swarms, world):
        g = dist.new_group(ranks)
        if rank in ranks:
            mine = g
    return mine


def pso_step_sharded(H, state, stat, lo, hi, eps_min, omega, phi_p, phi_g, seed, it, n_swarms_local, index_offset,
                     group=None, exchange=True, stream=None):
    """One PSO iteration (Eq. 13-15) on this rank's shard of the population, bit-identical to H.pso_step on the whole
    population: personal bests and the shard's candidate per swarm (sc_pso_best), all-gather of the candidates over the
    ranks that share the swarms (10 doubles per swarm and rank), pick (sc_pso_pick: value, then lowest GLOBAL index), move
    (sc_pso_move; the Philox counter is the global particle index).  state: the rank's pos, vel, pbest_pos, pbest_val and
    gbest_pos [n_swarms_local, 8], gbest_val [n_swarms_local]; index_offset = global index of the rank's first particle.
    exchange=False (whole swarms per rank): no collective."""
    pos = state["pos"]
    cand = torch.empty((n_swarms_local, 10), dtype=torch.float64, device=pos.device)
    H.pso_best(state, stat, cand, n_swarms_local, index_offset, stream)
    if exchange and dist.is_initialized() and dist.get_world_size(group) > 1:
        w = dist.get_world_size(group)
        flat = torch.empty((w * n_swarms_local, 10), dtype=torch.float64, device=pos.device)      # rank-major concatenation
        dist.all_gather_into_tensor(flat, cand, group=group)
        allc = flat.view(w, n_swarms_local, 10)
    else:
        allc = cand[None]
    H.pso_pick(allc, state, stream)
    H.pso_move(state, lo, hi, eps_min, omega, phi_p, phi_g, seed, it, n_swarms_local, index_offset, stream)
