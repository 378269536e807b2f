"""Multi-GPU layout of the particle-by-particle sweep: walkers are independent Markov chains
 and every GPU keeps its own replica of the read-only table (L311), so the
path shards by WALKERS with no data-path collective.  This module holds the
host-side logic only: which walkers a rank owns, and the max-over-ranks reduction of a timing
taken OUTSIDE the timed region.  It works with any torch.distributed backend (nccl on GPUs,
gloo in the CPU tests)."""
import numpy as np
import torch


def walker_range(rank, world, nw_total):
    """Contiguous block of walkers owned by `rank` when nw_total walkers are dealt over `world`
    ranks as evenly as possible (the first nw_total % world ranks get one more)."""
    if not (0 <= rank < world) or nw_total < 0:
        raise ValueError(f"bad shard request rank={rank} world={world} nw_total={nw_total}")
    base, extra = divmod(nw_total, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def shard_inputs(pos, delta, unif, rank, world):
    """This rank's slice of the walker-indexed inputs: pos [W][N][3], delta [S][N][W][3],
    unif [S][N][W].  Returns contiguous copies."""
    lo, hi = walker_range(rank, world, pos.shape[0])
    return (np.ascontiguousarray(pos[lo:hi]), np.ascontiguousarray(delta[:, :, lo:hi]),
            np.ascontiguousarray(unif[:, :, lo:hi]))


def max_over_ranks(value, device="cpu"):
    """Max of a per-rank scalar (a CUDA-event time in ms) over all ranks; identity without a
    process group.  One all_reduce of one double, outside any timed region."""
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(values, device="cpu"):
    """Element-wise sum of a short per-rank vector of statistics (moves, accepted moves)."""
    import torch.distributed as dist
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return [float(v) for v in t.tolist()]
