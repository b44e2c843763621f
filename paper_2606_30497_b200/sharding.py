"""Host-side logic of the multi-GPU paths; no method arithmetic here.

* Training does not shard (step t+1 needs the weights of step t): N ranks run N independent
  replicas; the job time is the maximum over ranks (`max_over_ranks`).
* The eval pass shards by rows: rank r evaluates rows `row_shard(n, r, world)` with
  `mlp_eval_loss` on its own GPU and the per-rank mean losses are combined with one scalar
  all-reduce (`combine_eval`): L = sum_r n_r L_r / n   (eq. 4, is a sum over rows).
"""
from __future__ import annotations


def row_shard(n: int, rank: int, world: int, align: int = 128):
    """Contiguous row range [lo, hi) of rank `rank`; boundaries are multiples of `align` rows
    (one TMA tile) except the end of the data, and the union over ranks is exactly [0, n)."""
    if n < 0 or world < 1 or not 0 <= rank < world:
        raise ValueError("bad shard arguments")
    tiles = (n + align - 1) // align
    lo_t = tiles * rank // world
    hi_t = tiles * (rank + 1) // world
    return min(n, lo_t * align), min(n, hi_t * align)


def combine_eval(local_mean_loss: float, local_rows: int, group=None) -> float:
    """Mean loss over all ranks' rows from each rank's mean loss over its own rows."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([local_mean_loss * local_rows, float(local_rows)], dtype=torch.float64)
    if dist.is_available() and dist.is_initialized():
        if dist.get_backend(group) == "nccl":
            t = t.cuda()
        dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    return float(t[0].item() / t[1].item()) if t[1].item() > 0 else float("nan")


def max_over_ranks(ms: float, group=None) -> float:
    """Job time of a replicas-only run: the slowest rank's device time."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64)
    if dist.is_available() and dist.is_initialized():
        if dist.get_backend(group) == "nccl":
            t = t.cuda()
        dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return float(t.item())
