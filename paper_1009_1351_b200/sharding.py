"""Slice sharding for more than one GPU: host-side bookkeeping only.

Slices are independent units of the path (no term of Eq. 1 couples them), so a job of S
slices is split contiguously across ranks and every rank runs the single-GPU library on its own
range.  Nothing is exchanged on the data path; timings are combined as the max over ranks.
"""


def slice_range(n_slices: int, world_size: int, rank: int) -> range:
    """Contiguous, balanced partition of range(n_slices): the first n_slices % world_size ranks
    get one slice more.  A rank may get an empty range when world_size > n_slices."""
    if n_slices < 0 or world_size < 1 or not (0 <= rank < world_size):
        raise ValueError("need n_slices >= 0, world_size >= 1 and 0 <= rank < world_size")
    base, extra = divmod(n_slices, world_size)
    lo = rank * base + min(rank, extra)
    return range(lo, lo + base + (1 if rank < extra else 0))


def max_over_ranks(value: float, dist=None, device="cpu") -> float:
    """Max of a per-rank scalar (a timing) over the default process group; identity without one."""
    if dist is None or not dist.is_initialized():
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def gather_slices(local, n_slices: int, dist=None):
    """Concatenate per-rank result tensors [S_rank, ...] (CPU or CUDA, same trailing shape) into
    [n_slices, ...] on every rank, in slice order.  Used once at the end of a sharded job."""
    if dist is None or not dist.is_initialized():
        return local
    import torch
    world = dist.get_world_size()
    sizes = [len(slice_range(n_slices, world, r)) for r in range(world)]
    pad = max(sizes)
    buf = local.new_zeros((pad,) + tuple(local.shape[1:]))
    buf[: local.shape[0]] = local
    parts = [torch.empty_like(buf) for _ in range(world)]
    dist.all_gather(parts, buf)
    return torch.cat([p[:s] for p, s in zip(parts, sizes)], dim=0)
