"""Parameter-range sharding across ranks.

The step is element-wise independent in the parameter index, so rank r runs the unchanged
single-GPU step on its own contiguous element range and NO data-path collective exists.  The
only cross-rank quantities are the a5 diagnostics (sums over elements), which are added with
one small all-reduce.  Works with any torch.distributed backend (nccl on GPUs; gloo in the CPU
tests)."""
import numpy as np

from .binding import hadpsgd_shard_range


def rank_shard(P_padded, dist=None):
    """[lo, hi) of this rank (whole range when torch.distributed is not initialised)."""
    if dist is None or not dist.is_initialized():
        return 0, P_padded
    return hadpsgd_shard_range(P_padded, dist.get_world_size(), dist.get_rank())


def allreduce_diagnostics(diag, dist, device="cpu"):
    """Sum the per-shard diagnostics dict {gsq, wsq, gap} over all ranks (in place, returns it)."""
    import torch
    S = len(diag["gsq"])
    t = torch.tensor(np.concatenate([diag["gsq"], diag["wsq"], diag["gap"]]), dtype=torch.float64, device=device)
    dist.all_reduce(t)
    t = t.cpu().numpy()
    diag["gsq"], diag["wsq"], diag["gap"] = t[:S].copy(), t[S:2 * S].copy(), t[2 * S:].copy()
    return diag


def max_over_ranks(value, dist, device="cpu"):
    """Max of a python float over ranks (the timing rule: device time, max over ranks)."""
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t[0])
