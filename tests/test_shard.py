"""N>1 host logic on CPU: world_size-2 gloo. The path shards by independent instances (weak
scaling, no data-path collective); the only cross-rank traffic is a barrier and a MAX reduce."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_04101_b200 import shard


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    n_inst, steps = 4, 6
    sched = shard.step_schedule(steps, n_inst, rank, world)
    owned = [shard.global_instance(rank, i, n_inst) for i in range(n_inst)]
    t = shard.reduce_max_time(10.0 + 5.0 * rank)
    # ranks plan identical inputs identically: an all_gather of a per-rank digest would be
    # the check on a real box; here we gather the owned instance ids
    got = [None] * world
    dist.all_gather_object(got, owned)
    dist.barrier()
    q.put((rank, sched, owned, t, got))
    dist.destroy_process_group()


def test_world_size_2_gloo():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, s0, o0, t0, g0), (r1, s1, o1, t1, g1) = res
    assert s0 == s1 == [0, 1, 2, 3, 0, 1]                  # every rank runs `steps` steps
    assert set(o0).isdisjoint(o1) and sorted(o0 + o1) == list(range(8))   # disjoint instances
    assert t0 == t1 == 15.0                                  # max over ranks
    assert g0 == g1 == [o0, o1]
    assert shard.total_units(6, world) == 12


def test_single_process_paths():
    assert shard.reduce_max_time(3.5) == 3.5
    assert shard.step_schedule(0, 3, 0, 1) == []
    assert shard.step_schedule(5, 2, 0, 1) == [0, 1, 0, 1, 0]
