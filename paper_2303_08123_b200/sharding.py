"""Batch sharding over ranks: simulations never interact, so rank r owns a contiguous
range of GLOBAL simulation ids; the only communication is the gather of fitness values (and the broadcast of
the next protocol table).  No device code here -- plain torch.distributed plumbing, tested on CPU with gloo."""
import numpy as np


def shard_range(total, world, rank):
    """Contiguous, balanced split of `total` simulations: returns (first_global_id, count) of `rank`."""
    base, rem = divmod(int(total), int(world))
    first = rank * base + min(rank, rem)
    return first, base + (1 if rank < rem else 0)


def shard_protocols(dose, delay, nfrac, world, rank):
    """Rows of the protocol table owned by `rank` plus its sim_id_base."""
    first, count = shard_range(len(nfrac), world, rank)
    sl = slice(first, first + count)
    return np.asarray(dose)[sl], np.asarray(delay)[sl], np.asarray(nfrac)[sl], first


def gather_fitness(local, total, dist=None):
    """All ranks receive the fitness of all `total` simulations, ordered by global id (one all_gather of B floats)."""
    local = np.ascontiguousarray(local, dtype=np.float32)
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return local.copy()
    import torch
    world = dist.get_world_size()
    sizes = [shard_range(total, world, r)[1] for r in range(world)]
    pad = max(sizes)
    buf = torch.zeros(pad, dtype=torch.float32)
    buf[:len(local)] = torch.from_numpy(local)
    out = [torch.zeros(pad, dtype=torch.float32) for _ in range(world)]
    dist.all_gather(out, buf)
    return np.concatenate([o.numpy()[:s] for o, s in zip(out, sizes)])


def broadcast_protocols(dose, delay, nfrac, dist=None, src=0):
    """Rank `src` owns the next generation's table (host GA); everybody gets a copy."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return dose, delay, nfrac
    obj = [(dose, delay, nfrac) if dist.get_rank() == src else None]
    dist.broadcast_object_list(obj, src=src)
    return obj[0]
