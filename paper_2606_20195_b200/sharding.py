"""Row sharding of one sketch over the ranks of a process group.

S is d x m, so a sketch of a tall matrix splits by rows: rank g applies the SAME map to rows
[row_begin, row_begin + rows) -- the global row index enters the hash -- into a private d x n sketch,
and the partial sketches are summed with one all-reduce.  No method arithmetic here: only the row
bookkeeping and the collective call, so the N > 1 path can be covered on CPU with the gloo backend.
"""
from __future__ import annotations


def shard_rows(m_total: int, world_size: int, rank: int, align: int = 4):
    """Contiguous row range of `rank`: (row_begin, rows).  Boundaries are multiples of `align` (the
    privatised kernel scatters aligned groups of <= 4 rows), the last rank takes the remainder."""
    if world_size < 1 or not (0 <= rank < world_size) or m_total < 0 or align < 1:
        raise ValueError("bad shard request")
    per = -(-m_total // world_size)          # ceil
    per = -(-per // align) * align           # round up to the alignment
    begin = min(rank * per, m_total)
    end = min(begin + per, m_total)
    return begin, end - begin


def all_reduce_sketch(partial, dist=None):
    """Sum the ranks' partial sketches in place (NCCL on GPUs, gloo on CPU) -- the one collective of the sharded path,
    called by bench.py after every apply.  `partial` is a torch tensor of the sketch dtype; for FP16 sketches this is one
    more level of the accumulation hierarchy.  Runs whenever a process group exists, also with a single rank (the
    communicator is then exercised on whatever box this is); without a process group it is the identity."""
    if dist is None:
        import torch.distributed as dist  # noqa: PLC0415
    if dist.is_available() and dist.is_initialized():
        dist.all_reduce(partial)
    return partial


def max_over_ranks(value: float, dist=None, device=None) -> float:
    """The slowest rank's value (bench.py's timing rule: a multi-GPU number is the max over ranks of the device time).
    One FP64 all-reduce with MAX on `device` (the rank's GPU under NCCL, CPU under gloo); identity without a process group."""
    import torch  # noqa: PLC0415

    if dist is None:
        import torch.distributed as dist  # noqa: PLC0415
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized():
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
