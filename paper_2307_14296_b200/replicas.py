"""Multi-GPU host logic: replicas only.  The (operator, frequency) response systems are independent
(PAPER.md:199-201), so N ranks each own a full context and a slice of the systems; the only inter-rank traffic is the
max-over-ranks of the device time (and, for a sweep, gathering scalars).  No arithmetic of the method lives here."""
import torch
import torch.distributed as dist


def shard(nitems, rank, world):
    """Contiguous balanced slice [lo, hi) of ``nitems`` independent systems owned by ``rank`` (sizes differ by at most 1)."""
    if not (0 <= rank < world):
        raise ValueError("rank %d outside world %d" % (rank, world))
    base, extra = divmod(nitems, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def max_over_ranks(values, device="cpu"):
    """Element-wise MAX over ranks of a list of floats (identity when torch.distributed is not initialised)."""
    t = torch.tensor([float(x) for x in values], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


def gather_scalars(values, device="cpu"):
    """All ranks' lists of complex scalars (equal length per rank), concatenated in rank order, on every rank."""
    t = torch.tensor([complex(x) for x in values], dtype=torch.complex128, device=device)
    if not (dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1):
        return [complex(x) for x in t]
    real = torch.view_as_real(t).contiguous()
    rparts = [torch.empty_like(real) for _ in range(dist.get_world_size())]
    dist.all_gather(rparts, real)
    return [complex(float(a), float(b)) for p in rparts for a, b in p.tolist()]
