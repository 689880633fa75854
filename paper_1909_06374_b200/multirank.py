"""Host-side logic of the multi-GPU path: curves are independent, so a job is a partition
of curve numbers over ranks and a max-over-ranks of the device time.  No data-path collective exists.

Plumbing only (torch.distributed); none of the method's arithmetic is here.
"""
import torch


def partition_curves(B_total, rank, world):
    """Contiguous split of curve numbers 0..B_total-1 over `world` ranks: returns (curve0, B_local).
    The first B_total % world ranks get one extra curve.  Philox counters carry the absolute curve number
    (curve0 + row), so the union over ranks equals the single-rank result bit for bit."""
    if not (0 <= rank < world) or B_total < 0:
        raise ValueError("bad partition arguments")
    base, extra = divmod(int(B_total), int(world))
    b_local = base + (1 if rank < extra else 0)
    curve0 = rank * base + min(rank, extra)
    return curve0, b_local


def weak_curve0(B_per_rank, rank):
    """Weak scaling (bench.py): every rank runs its own B_per_rank curves, numbered after the lower ranks'."""
    return int(rank) * int(B_per_rank)


def max_over_ranks(value, device=None, dist=None):
    """MAX all-reduce of one scalar (device time in ms): multi-GPU numbers are the slowest rank's."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
