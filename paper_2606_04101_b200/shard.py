"""Multi-GPU host logic: the path shards by independent (layer, microbatch) instances.

Every rank plans its own instances with the identical kernels; there is NO data-path
collective (the paper's all-gather of the R x E count matrix belongs to the
real multi-rank histogram, which this single-GPU emulation folds into one kernel).  The only
cross-rank traffic in bench.py is the barrier and a MAX all-reduce of the device-measured time.
"""
from __future__ import annotations


def global_instance(rank: int, local: int, n_inst: int) -> int:
    """Global id of a rank's local instance: ranks own disjoint contiguous blocks."""
    return rank * n_inst + local


def step_schedule(steps: int, n_inst: int, rank: int, world: int) -> list[int]:
    """Local instance index used by each of this rank's `steps` timed steps (weak scaling:
    every rank runs `steps` steps; consecutive steps use different instances => L2-cold)."""
    assert steps >= 0 and n_inst >= 1 and 0 <= rank < world
    return [j % n_inst for j in range(steps)]


def total_units(steps: int, world: int) -> int:
    """Layers planned by the whole job in the timed region."""
    return steps * world


def reduce_max_time(value_ms: float, group=None) -> float:
    """max over ranks of a device-measured duration (works with gloo on CPU and nccl on GPU)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return float(value_ms)
    dev = "cuda" if dist.get_backend(group) == "nccl" else "cpu"
    t = torch.tensor([value_ms], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return float(t.item())
