"""Multi-GPU host logic.

Two ways to use N GPUs, both one process per GPU:
  * independent (layer, microbatch) instances sharded over ranks — what `bench.py --gpus N`
    times: every rank plans its own instances with the identical kernels, weak scaling, NO
    data-path collective (a barrier and a MAX all-reduce of the device-measured time only);
  * one layer's tokens sharded over ranks, the paper's deployment:
    count locally, ONE all-gather of the count rows, identical plan everywhere, local lookup —
    `exchange_counts` / `TokenShardedLayer` below around uep_shard_count / uep_shard_finish.
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


# ---- token-sharded path (uep.h: uep_shard_count / uep_shard_rows / uep_shard_finish) ----------
# The paper's own deployment: every GPU ranks and counts its local
# tokens, ONE all-gather of the count rows, then every GPU solves the identical plan and looks up
# its own slots.  Only the exchange lives here; every other step is a kernel behind the C ABI.

def exchange_counts(ws, offset0: int, n_bytes: int, rank: int, world: int, group=None) -> None:
    """In-place all-gather of the shards' count rows inside the workspace tensor `ws` (uint8):
    shard g's rows are ws[offset0 + g*n_bytes : offset0 + (g+1)*n_bytes] (uep_shard_rows), and
    after the call every rank holds all of them.  Enqueued on the current stream under NCCL."""
    import torch.distributed as dist
    assert 0 <= rank < world and n_bytes >= 0
    if n_bytes == 0 or not (dist.is_available() and dist.is_initialized()):
        assert world == 1 or n_bytes == 0, "world > 1 needs an initialised process group"
        return
    region = ws[offset0:offset0 + world * n_bytes]
    mine = region[rank * n_bytes:(rank + 1) * n_bytes]
    if dist.get_backend(group) != "nccl":
        mine = mine.clone()                      # only NCCL documents the aliased (in-place) form
    dist.all_gather_into_tensor(region, mine, group=group)


class TokenShardedLayer:
    """One GPU's side of the token-sharded path for one layer shape: owns the context's
    workspace, plan and outputs for the local S/G slots.  step() = count -> all-gather -> finish."""

    def __init__(self, ctx, rank: int, world: int, group=None, gates: bool = True):
        import torch
        self.ctx, self.rank, self.world, self.group = ctx, rank, world, group
        self.ws = ctx.new_workspace()
        self.plan = ctx.new_plan()
        self.off0, self.n_bytes = ctx.uep_shard_rows(0, world)
        S = ctx.T * ctx.k
        assert S % world == 0
        self.S_local = S // world
        dev = ctx.device
        i32 = lambda n: torch.empty(max(n, 1), dtype=torch.int32, device=dev)
        self.expert_count = i32(ctx.E)
        self.out_replica, self.out_rank, self.out_offset = i32(self.S_local), i32(self.S_local), i32(self.S_local)
        self.n_inflight = torch.zeros(max(ctx.R, 4), dtype=torch.int32, device=dev)
        self.out_gate = None
        self.gates = gates

    def step(self, ids_local, gate_local=None):
        import torch
        c = self.ctx
        if gate_local is not None and self.out_gate is None:
            self.out_gate = torch.zeros(max(c.T * c.k, 1), dtype=gate_local.dtype, device=c.device)
        c.uep_shard_count(self.rank, self.world, ids_local, self.ws)
        exchange_counts(self.ws, self.off0, self.n_bytes, self.rank, self.world, self.group)
        c.uep_shard_finish(self.rank, self.world, gate_local, self.expert_count, self.plan,
                           self.out_replica, self.out_rank, self.out_offset,
                           self.out_gate if gate_local is not None else None, self.n_inflight, self.ws)
