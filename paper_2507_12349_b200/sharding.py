"""Batch sharding across ranks: configurations are independent units, so a global batch is cut into
contiguous per-rank slices and every rank evaluates its own slice with its own handle.  No data-path collective:
torch.distributed is used only for the barrier and the max-over-ranks timing of bench.py."""


def shard_bounds(batch, rank, world):
    """[begin, end) of rank's contiguous slice of `batch` configurations; slices differ by at most one
    configuration, cover the batch exactly once, and are empty for ranks >= batch."""
    batch, rank, world = int(batch), int(rank), int(world)
    if world < 1 or not (0 <= rank < world) or batch < 0:
        raise ValueError("shard_bounds: need 0 <= rank < world and batch >= 0")
    q, r = divmod(batch, world)
    begin = rank * q + min(rank, r)
    return begin, begin + q + (1 if rank < r else 0)


def shard_vertices(vertices, batch, rank, world):
    """This rank's slice of a global batch of vertex configurations: `vertices` is the dict of batch-innermost arrays
    (sites [n][2][B], tau [n][B], ...) every rank draws from the same seed; returns (begin, end, dict of contiguous
    slices [..., begin:end]).  Used by `bench.py --scaling strong` and by the 2-rank gloo test: the same code."""
    import numpy as np
    b0, b1 = shard_bounds(batch, rank, world)
    return b0, b1, {k: np.ascontiguousarray(a[..., b0:b1]) for k, a in vertices.items()}


def max_over_ranks(values, device=None):
    """Element-wise MAX over ranks of a list of floats (identity when torch.distributed is not initialised)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return [float(v) for v in values]
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t.tolist()]
