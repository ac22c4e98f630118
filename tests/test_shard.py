"""N>1 host logic on CPU: world_size-2 gloo.  bench.py shards independent instances (weak
scaling, no data-path collective: a barrier and a MAX reduce only); the token-sharded path of
SURVEY §8(e) has one exchange, the in-place all-gather of the shards' count rows."""
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


def E_pad_row_bytes(E_pad):
    return 4 * E_pad                       # row 0 of the prefix table stays zero in the real layout


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
    # token-sharded path: the exchange of count rows inside a workspace-shaped byte tensor.
    # Shard g's rows (E_pad int32 per chunk) sit at off0 + g*nb; the kernels that fill and consume
    # them need a GPU, the exchange itself does not.
    E_pad, chunks, off0 = 16, 3, 256 + 2048 + 64 + E_pad_row_bytes(16)
    nb = chunks * E_pad * 4
    ws = torch.full((off0 + world * nb + 128,), 0xAB, dtype=torch.uint8)
    mine = (torch.arange(chunks * E_pad, dtype=torch.int32) + 1000 * (rank + 1))
    ws[off0 + rank * nb: off0 + (rank + 1) * nb] = mine.view(torch.uint8)
    shard.exchange_counts(ws, off0, nb, rank, world)
    dist.barrier()
    q.put((rank, sched, owned, t, got, ws.numpy().copy(), off0, nb))
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
    (r0, s0, o0, t0, g0, w0, off0, nb), (r1, s1, o1, t1, g1, w1, _, _) = res
    import numpy as np
    assert np.array_equal(w0, w1)                                          # every rank holds every row
    rows = w0[off0: off0 + 2 * nb].view(np.int32).reshape(2, -1)
    assert np.array_equal(rows[0], np.arange(rows.shape[1]) + 1000)
    assert np.array_equal(rows[1], np.arange(rows.shape[1]) + 2000)
    assert (w0[:off0] == 0xAB).all() and (w0[off0 + 2 * nb:] == 0xAB).all()  # nothing else touched
    assert s0 == s1 == [0, 1, 2, 3, 0, 1]                  # every rank runs `steps` steps
    assert set(o0).isdisjoint(o1) and sorted(o0 + o1) == list(range(8))   # disjoint instances
    assert t0 == t1 == 15.0                                  # max over ranks
    assert g0 == g1 == [o0, o1]
    assert shard.total_units(6, world) == 12


def _lambda_worker(rank, world, port, q):
    """Two ranks run the HOST side of the token-sharded path: each counts its own
    source ranks' token blocks (here with the oracle, standing in for uep_shard_count), the rows of
    Lambda[R][E_pad] are all-gathered in place, and every rank derives lambda_e and the global rank
    base of every source rank from the gathered matrix."""
    import numpy as np
    import oracle
    from paper_2606_04101_b200 import synth
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    T, k, E, R = 4096, 2, 13, 8                       # E_pad = 16
    E_pad = (E + 3) // 4 * 4
    ids = synth.zipf_topk_ids(T, k, E, 1.2, 7).numpy()
    ids[5, 0] = -1                                     # an invalid id is in no row
    rps, block = R // world, T // R
    off0 = 4096                                        # byte offset of Lambda inside a workspace-shaped buffer
    nb = rps * E_pad * 4
    ws = torch.full((off0 + world * nb + 64,), 0xCD, dtype=torch.uint8)
    mine = np.zeros((rps, E_pad), np.int32)
    for j in range(rps):
        r = rank * rps + j
        mine[j, :E], _ = oracle.histogram(ids[r * block:(r + 1) * block], E)
    ws[off0 + rank * nb: off0 + (rank + 1) * nb] = torch.from_numpy(mine.reshape(-1).view(np.uint8).copy())
    shard.exchange_counts(ws, off0, nb, rank, world)
    dist.barrier()
    Lam = ws[off0: off0 + world * nb].numpy().view(np.int32).reshape(R, E_pad)
    lam, bad = oracle.histogram(ids, E)
    ok_tot = bool((Lam[:, :E].sum(axis=0) == lam).all()) and bad == 1
    base = np.cumsum(Lam[:, :E], axis=0) - Lam[:, :E]                      # global rank base of (source rank, expert)
    flat = ids.reshape(-1)
    ok_base = all(int(base[r, e]) == int((flat[:r * block * k] == e).sum()) for r in range(R) for e in range(E))
    q.put((rank, ok_tot, ok_base, nb, Lam.copy()))
    dist.destroy_process_group()


def test_lambda_rows_exchange_world_2():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_lambda_worker, args=(r, world, port, q)) for r in range(world)]
    for p in ps:
        p.start()
    res = sorted((q.get(timeout=120) for _ in range(world)), key=lambda x: x[0])
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    import numpy as np
    assert all(r[1] and r[2] for r in res)
    assert res[0][3] == 4 * 16 * 8 // 2                                    # 4 * E_pad * R / G bytes per GPU
    assert np.array_equal(res[0][4], res[1][4])                            # every rank holds the same matrix


def test_single_process_paths():
    ws = torch.arange(64, dtype=torch.uint8)
    shard.exchange_counts(ws, 16, 32, 0, 1)                               # world 1: a no-op
    assert torch.equal(ws, torch.arange(64, dtype=torch.uint8))
    assert shard.reduce_max_time(3.5) == 3.5
    assert shard.step_schedule(0, 3, 0, 1) == []
    assert shard.step_schedule(5, 2, 0, 1) == [0, 1, 0, 1, 0]
