"""Frame-range sharding over ranks and the one exchange step.

Frames are independent units (Algorithm 1's `parallel for f`): rank r scans the
contiguous shard `shard_range(total, r, world)` of a class's frame range with
kripke_eval_batch_range, then `combine` adds the counts (all-reduce SUM) and keeps the
lexicographically first witness (all-reduce MIN on the 64-bit keys of kripke_witness_to_keys).
The tensors may live on any device torch.distributed's backend supports (NCCL on GPUs; the CPU
tests use gloo).
"""
from __future__ import annotations


def shard_range(total: int, rank: int, world: int):
    """Contiguous shard [begin, begin + count) of `total` frames for `rank`; shards tile the range."""
    begin = total * rank // world
    return begin, total * (rank + 1) // world - begin


def combine(counts, keys, group=None):
    """In-place all-reduce of per-rank partial results: counts (int64, any shape) by SUM, witness
    keys (int64) by MIN.  Returns (counts, keys)."""
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(counts, op=dist.ReduceOp.SUM, group=group)
        dist.all_reduce(keys, op=dist.ReduceOp.MIN, group=group)
    return counts, keys
