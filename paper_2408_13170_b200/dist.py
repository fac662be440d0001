"""Multi-GPU plumbing: one process per GPU, torch.distributed for the few scalars that cross ranks.

The statistic shards over independent problems ("This can be done in parallel",
PAPER.md:365-367 one GPU per tile): every rank owns whole tiles or whole swarms, the whitened data is replicated,
and the data path has NO collective.  The only exchange that can ever be needed is the swarm best when ONE swarm is
split over ranks: a (value, global index) arg-max plus the 64-byte winning position -- latency-bound, done here with
an all-gather of 10 doubles per rank.  Works on NCCL (GPU tensors) and gloo (CPU tensors).
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
