"""Multi-GPU sharding of the disorder pool.

Disorder samples are independent (the paper's overline is a plain average over realisations,
PAPER.md:49), while the replicas and temperature slots of one sample interact (PT, overlaps) and stay
together.  The pool is split into contiguous ranges of whole packed words (32 samples); every Philox
stream is keyed by the GLOBAL sample / word index (sg_set_first_sample), so results do not depend on
the number of GPUs.  No communication during the run; one reduction of the moment sums at the end.
"""
from typing import Tuple


def shard_range(n_samples: int, world: int, rank: int) -> Tuple[int, int]:
    """(first_sample, count) of rank's shard: whole 32-sample words, as even as possible, in rank order."""
    if world < 1 or not (0 <= rank < world) or n_samples < 1:
        raise ValueError("bad shard arguments")
    words = (n_samples + 31) // 32
    base, extra = divmod(words, world)
    w0 = rank * base + min(rank, extra)
    nw = base + (1 if rank < extra else 0)
    first = w0 * 32
    count = max(0, min(n_samples, (w0 + nw) * 32) - first)
    return first, count


def reduce_moment_sums(local_sums, group=None):
    """All-reduce (sum, fp64) of per-slot moment sums [n_temps][NMOM] over the ranks: the only
    exchange step of the sharded job.  `local_sums` is a torch tensor on the backend's device
    (CUDA for nccl, CPU for gloo); returned tensor is the same on every rank."""
    import torch.distributed as dist
    out = local_sums.clone()
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(out, op=dist.ReduceOp.SUM, group=group)
    return out
