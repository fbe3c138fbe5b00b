"""Sharding of a parameter batch across ranks (one process per GPU).

The hot path shards by parameter vector ("sharding chains or live points across GPUs and
batching likelihood calls within each device"): the units are independent, the tables are replicated and
there is no data-path collective.  The only exchanges are the final gather of the B log-likelihoods and
the max-over-ranks of a timing; both go through torch.distributed (NCCL on GPUs, gloo in the CPU tests).
"""


def shard_slice(n_total, rank, world):
    """Contiguous balanced split of range(n_total): -> (lo, hi) of this rank; sizes differ by at most 1."""
    if world < 1 or not (0 <= rank < world) or n_total < 0:
        raise ValueError("bad shard arguments")
    base, rem = divmod(n_total, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def gather_vectors(local, n_total, group=None):
    """All ranks receive the concatenation (in rank order) of every rank's 1-D `local` tensor, where rank r
    holds the shard_slice(n_total, r, world) part.  Ragged shards are padded for the all_gather."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return local.clone()
    world = dist.get_world_size(group)
    sizes = [hi - lo for lo, hi in (shard_slice(n_total, r, world) for r in range(world))]
    width = max(sizes) if sizes else 0
    pad = torch.zeros(width, dtype=local.dtype, device=local.device)
    pad[:local.numel()] = local
    parts = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(parts, pad, group=group)
    return torch.cat([p[:s] for p, s in zip(parts, sizes)])


def max_over_ranks(values, device=None, group=None):
    """Element-wise max over ranks of a list of floats (timings): -> list of floats."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized():
        dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return [float(x) for x in t]
