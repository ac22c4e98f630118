"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element,
on the same seeded inputs.  Bar: bit-exact on every integer / index array and scalar,
byte-exact pack and gates (all of the path is integer or byte work; there is no floating-point
tolerance anywhere).  All tests need a B200 and are marked gpu."""
import os

import numpy as np
import pytest
import torch

import oracle
import uep_checks as ck
from paper_2606_04101_b200 import binding, synth

pytestmark = pytest.mark.gpu
DEV = "cuda"

PLAN_ARRAYS = ("slot_expert", "inst_off", "inst_rank", "inst_phys", "inst_cum", "phys_count",
               "phys_base", "rank_load", "rank_base", "scalars", "U")


def gpu_chain(ids, gate, E, R, n_slot, u_min, mode=binding.FLOOR_TOLERANT, home=None,
              states=(), use_balance=False, beta=(101, 100)):
    """Run hist -> plan -> remap -> pack on the GPU; return host copies of everything."""
    T, k = ids.shape
    gd = binding.GATE_NONE if gate is None else \
        (binding.GATE_BF16 if gate.element_size() == 2 else binding.GATE_F32)
    ctx = binding.Context(T, k, E, R, n_slot, u_min, beta[0], beta[1], mode, gd, home)
    ws = ctx.new_workspace()
    plan = ctx.new_plan(dense_U=True)
    d_ids = ids.to(DEV)
    d_gate = None if gate is None else gate.to(DEV)
    count = torch.full((E,), -7, dtype=torch.int32, device=DEV)
    rep, rnk, off, og = ctx.new_outputs(d_gate)
    for t in (rep, rnk, off):
        t.fill_(-9)
    srcs = [s.to(DEV) for s in states]
    sentinels = []
    for sr in srcs:                       # random bytes: empty slots must survive untouched
        sn = torch.empty((R, max(n_slot, 1)) + tuple(sr.shape[1:]), dtype=sr.dtype, device=DEV)
        sn.view(torch.uint8).copy_(torch.randint(0, 256, sn.view(torch.uint8).shape,
                                                 dtype=torch.uint8, device=DEV))
        sentinels.append(sn)
    dsts = [sn.clone() for sn in sentinels]
    if use_balance:
        ctx.uep_balance(d_ids, d_gate, count, plan, rep, rnk, off, og, srcs, dsts, ws)
    else:
        ctx.uep_histogram(d_ids, count, ws)
        ctx.uep_plan(count, plan, ws)
        ctx.uep_remap(d_ids, d_gate, plan, rep, rnk, off, og, ws)
        if srcs:
            ctx.uep_pack(plan, srcs, dsts)
    torch.cuda.synchronize()
    res = dict(count=count.cpu().numpy(), plan=plan.host(), rep=rep.cpu().numpy(),
               rnk=rnk.cpu().numpy(), off=off.cpu().numpy(),
               og=None if og is None else og.cpu(), dsts=[d.cpu() for d in dsts],
               sentinels=[s.cpu() for s in sentinels], ctx=ctx)
    return res


def oracle_chain(ids, gate, E, R, n_slot, u_min, mode=oracle.FLOOR_TOLERANT, home=None,
                 beta=(101, 100)):
    ids_np = ids.numpy()
    lam, bad = oracle.histogram(ids_np, E)
    p = oracle.plan(lam, R, n_slot, u_min, beta[0], beta[1], mode, home, S_total=ids_np.size)
    g_np = None
    if gate is not None:
        g_np = gate.view(torch.int16).numpy().view(np.uint16) if gate.element_size() == 2 \
            else gate.view(torch.int32).numpy().view(np.uint32)
    rep, rnk, off, og = oracle.remap(ids_np, g_np, p)
    return lam, p, rep, rnk, off, og


def assert_parity(g, o, ids, gate, states=(), n_valid=None):
    lam, p, rep, rnk, off, og = o
    assert np.array_equal(g["count"], lam)
    hp = g["plan"]
    for n in PLAN_ARRAYS:
        a, b = getattr(hp, n), getattr(p, n)
        assert np.array_equal(np.asarray(a).reshape(-1), np.asarray(b).reshape(-1)), n
    # inst_base is a derived view of the oracle's receive layout: phys_base[inst_rank][inst_phys]
    n_inst = int(p.inst_off[-1])
    exp_base = np.asarray(p.phys_base).reshape(p.R, -1)[np.asarray(p.inst_rank)[:n_inst],
                                                        np.asarray(p.inst_phys)[:n_inst]]
    assert np.array_equal(np.asarray(hp.inst_base)[:n_inst], exp_base), "inst_base"
    assert not np.asarray(hp.inst_base)[n_inst:].any()
    assert np.array_equal(g["rep"], rep) and np.array_equal(g["rnk"], rnk) \
        and np.array_equal(g["off"], off)
    if gate is not None:
        nv = int(p.rank_base[-1])
        gg = g["og"]
        gbits = gg.view(torch.int16).numpy().view(np.uint16) if gg.element_size() == 2 \
            else gg.view(torch.int32).numpy().view(np.uint32)
        assert np.array_equal(gbits[:nv], og[:nv])
    for st, d, sn in zip(states, g["dsts"], g["sentinels"]):
        src_b = st.contiguous().view(torch.uint8).numpy().reshape(st.shape[0], -1)
        ref = sn.contiguous().view(torch.uint8).numpy().reshape(p.R, max(p.n_slot, 1), -1).copy()
        if p.n_slot:
            oracle.pack(p.slot_expert, np.ascontiguousarray(src_b), ref)
        got = d.contiguous().view(torch.uint8).numpy().reshape(ref.shape)
        assert np.array_equal(got, ref)


def with_layout(hp, home=None):
    """Attach the static layout (h(e), main slot index) so uep_checks can run on a GPU plan."""
    hp.home, hp.main_phys, M = oracle.layout(hp.E, hp.R, home)
    assert M == hp.M
    return hp


def test_tiny_config_full_chain_both_modes():
    c = synth.CONFIGS["tiny"]
    ids = synth.zipf_topk_ids(c["T"], c["k"], c["E"], c["zipf_s"], 2024)
    gate = synth.gates_uniform_renorm(c["T"], c["k"], 11)
    state = synth.expert_state(c["E"], 256 * 512, 5)
    for mode in (binding.FLOOR_STRICT, binding.FLOOR_TOLERANT):
        for use_balance in (False, True):
            g = gpu_chain(ids, gate, c["E"], c["R"], c["n_slot"], c["u_min"], mode,
                          states=[state], use_balance=use_balance)
            o = oracle_chain(ids, gate, c["E"], c["R"], c["n_slot"], c["u_min"], mode)
            assert_parity(g, o, ids, gate, [state])
            assert o[1].n_replicas > 0


GRID = [  # (T, k, E, R, n_slot, s)  — sizes spanning several chunks/rounds and ragged tails
    (4099, 2, 16, 4, 1, 1.2), (8191, 8, 128, 32, 2, 0.6), (65536, 8, 128, 32, 2, 1.4),
    (50001, 8, 256, 64, 2, 1.0), (16384, 4, 512, 256, 4, 2.0), (4097, 1, 64, 8, 1, 0.0),
    (8192, 8, 160, 40, 4, 1.0), (2048, 4, 64, 256, 1, 1.0), (30011, 8, 512, 8, 3, 1.6),
    (1, 1, 1, 1, 0, 0.0), (3, 2, 5, 3, 2, 0.5), (131, 1, 7, 2, 1, 1.0), (700000, 4, 500, 250, 3, 1.1),
]


@pytest.mark.parametrize("T,k,E,R,n_slot,s", GRID)
@pytest.mark.parametrize("mode", [binding.FLOOR_STRICT, binding.FLOOR_TOLERANT])
def test_grid_parity(T, k, E, R, n_slot, s, mode):
    ids = synth.zipf_topk_ids(T, k, E, s, seed=T + E + R)
    gate = synth.gates_uniform_renorm(T, k, 3)
    u_min = synth.stress_u_min(T * k, R)
    state = synth.expert_state(E, 1000 * 8 + 8, 1)     # ragged: 16016 B per expert, < one tile
    g = gpu_chain(ids, gate, E, R, n_slot, u_min, mode, states=[state])
    o = oracle_chain(ids, gate, E, R, n_slot, u_min, mode)
    assert_parity(g, o, ids, gate, [state])


STRESS = [  # (S, k, E, R, n_slot, dist)
    (1024, 1, 64, 8, 1, "uniform"), (1024, 4, 256, 64, 2, "zipf2"), (4096, 8, 512, 256, 4, "one"),
    (262144, 8, 64, 256, 3, "zipf2"), (262144, 4, 256, 8, 1, "one"), (1 << 20, 8, 512, 64, 2, "uniform"),
    (1 << 22, 8, 256, 64, 4, "zipf2"), (1 << 22, 8, 512, 256, 4, "one"), (1 << 22, 1, 64, 8, 1, "uniform"),
    (1 << 22, 4, 512, 256, 1, "zipf2"),
]


@pytest.mark.parametrize("S,k,E,R,n_slot,dist", STRESS)
def test_stress_sweep_parity(S, k, E, R, n_slot, dist):
    T = S // k
    if dist == "one":
        ids = synth.one_expert_ids(T, k, E // 3)
    else:
        ids = synth.zipf_topk_ids(T, k, E, 2.0 if dist == "zipf2" else 0.0, seed=S + E)
    gate = synth.gates_uniform_renorm(T, k, 9)
    u_min = synth.stress_u_min(S, R)
    state = synth.expert_state(E, 2048 * 16, 2)         # 64 KiB per expert: 4 tiles
    g = gpu_chain(ids, gate, E, R, n_slot, u_min, states=[state])
    o = oracle_chain(ids, gate, E, R, n_slot, u_min)
    assert_parity(g, o, ids, gate, [state])
    ck.check_plan(o[0], with_layout(g["plan"]), u_min)


def test_invalid_ids_gate_bits_and_bf16():
    rng = np.random.default_rng(3)
    T, k, E, R = 20000, 4, 16, 4
    ids = torch.from_numpy(rng.integers(-3, 20, size=(T, k)).astype(np.int32))
    bits = (np.arange(T * k, dtype=np.uint32) * np.uint32(2654435761)).astype(np.uint32)
    bits[:8] = [0x7FC00001, 0xFFC12345, 0x80000000, 0x00000001, 0x807FFFFF, 0x7F800000,
                0xFF800000, 0x7FA00000]
    gate = torch.from_numpy(bits.view(np.float32).reshape(T, k).copy())
    g = gpu_chain(ids, gate, E, R, 1, 32)
    o = oracle_chain(ids, gate, E, R, 1, 32)
    assert_parity(g, o, ids, gate)
    assert int(g["plan"].scalars[binding.SC_N_INVALID]) == int(((ids < 0) | (ids >= E)).sum())
    gate16 = synth.gates_softmax_bf16(T, k, 4)
    g = gpu_chain(ids, gate16, E, R, 1, 32)
    o = oracle_chain(ids, gate16, E, R, 1, 32)
    assert_parity(g, o, ids, gate16)
    g = gpu_chain(ids, None, E, R, 1, 32)                # no gates at all
    o = oracle_chain(ids, None, E, R, 1, 32)
    assert_parity(g, o, ids, None)


def test_explicit_home_map_and_identity_cases():
    rng = np.random.default_rng(8)
    T, k, E, R = 30000, 4, 64, 8
    ids = synth.zipf_topk_ids(T, k, E, 1.0, 77)
    home = rng.integers(0, R, E).astype(np.int32)
    g = gpu_chain(ids, None, E, R, 3, 256, home=home)
    o = oracle_chain(ids, None, E, R, 3, 256, home=home)
    assert_parity(g, o, ids, None)
    # balanced input -> identity (S4); n_slot = 0; R = 1
    ids_b = (torch.arange(T * k, dtype=torch.int32) % E).view(T, k)
    for (RR, ns) in ((8, 2), (8, 0), (1, 2)):
        for ii in (ids_b, ids):
            g = gpu_chain(ii, None, E, RR, ns, 16)
            o = oracle_chain(ii, None, E, RR, ns, 16)
            assert_parity(g, o, ii, None)


def test_multi_tensor_pack_training_state():
    """config-3 style moved state: bf16 W + fp32 grad/m/v, several tiles and a ragged last tile."""
    T, k, E, R, ns = 32768, 8, 64, 16, 2
    ids = synth.zipf_topk_ids(T, k, E, 1.3, 5)
    n = 40000 + 8                                        # 80016 B bf16 / 160032 B fp32 per expert
    states = [synth.expert_state(E, n, 1), synth.expert_state(E, n, 2, torch.float32),
              synth.expert_state(E, n, 3, torch.float32), synth.expert_state(E, n, 4, torch.float32)]
    g = gpu_chain(ids, None, E, R, ns, 512, states=states, use_balance=True)
    o = oracle_chain(ids, None, E, R, ns, 512)
    assert o[1].n_replicas > 4
    assert_parity(g, o, ids, None, states)


@pytest.mark.parametrize("name,s", [("glm_air", 0.6), ("glm_air", 1.0), ("glm_air", 1.4), ("dsv3_prefill", 1.0)])
def test_full_size_configs_bit_exact(name, s):
    """BASELINE configs 1 and 2 at full size, in the launch configuration bench.py times
    (uep_balance): every integer output against the oracle, element by element."""
    c = synth.CONFIGS[name]
    ids = synth.zipf_topk_ids(c["T"], c["k"], c["E"], s, 4242, device=DEV).cpu()
    gate = synth.gates_softmax_bf16(c["T"], c["k"], 6) if c["gate"] == "bf16" \
        else synth.gates_uniform_renorm(c["T"], c["k"], 6)
    state = synth.expert_state(c["E"], 1 << 20, 3)       # 2 MiB per expert stands in for 88 MB
    g = gpu_chain(ids, gate, c["E"], c["R"], c["n_slot"], c["u_min"], states=[state],
                  use_balance=True)
    o = oracle_chain(ids, gate, c["E"], c["R"], c["n_slot"], c["u_min"])
    assert_parity(g, o, ids, gate, [state])
    ck.check_plan(o[0], with_layout(g["plan"]), c["u_min"])
    ck.check_remap(ids.numpy(), g["plan"], g["rep"], g["rnk"], g["off"])


def test_graph_capture_replay_and_determinism():
    c = synth.CONFIGS["glm_air"]
    T, k, E, R, ns = 16384, c["k"], c["E"], c["R"], c["n_slot"]
    ctx = binding.Context(T, k, E, R, ns, 256)
    ws = ctx.new_workspace()
    plan = ctx.new_plan(dense_U=True)
    d_ids = torch.zeros((T, k), dtype=torch.int32, device=DEV)
    d_gate = torch.zeros((T, k), dtype=torch.float32, device=DEV)
    count = torch.zeros(E, dtype=torch.int32, device=DEV)
    rep, rnk, off, og = ctx.new_outputs(d_gate)
    state = synth.expert_state(E, 20000, 1, device=DEV)
    dst = torch.zeros((R, ns, 20000), dtype=state.dtype, device=DEV)
    stream = torch.cuda.Stream()
    stream.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(stream):
        ctx.uep_balance(d_ids, d_gate, count, plan, rep, rnk, off, og, [state], [dst], ws)  # warm
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=stream):
            ctx.uep_balance(d_ids, d_gate, count, plan, rep, rnk, off, og, [state], [dst], ws)
    torch.cuda.synchronize()
    prev = None
    for it, seed in enumerate((1, 2, 2)):
        ids = synth.zipf_topk_ids(T, k, E, 0.8 + 0.4 * seed, seed)
        gate = synth.gates_uniform_renorm(T, k, seed)
        d_ids.copy_(ids)
        d_gate.copy_(gate)
        dst.zero_()
        torch.cuda.synchronize()
        graph.replay()
        torch.cuda.synchronize()
        g = dict(count=count.cpu().numpy(), plan=plan.host(), rep=rep.cpu().numpy(),
                 rnk=rnk.cpu().numpy(), off=off.cpu().numpy(), og=og.cpu(), dsts=[dst.cpu()],
                 sentinels=[torch.zeros_like(dst).cpu()])
        o = oracle_chain(ids, gate, E, R, ns, 256)
        assert_parity(g, o, ids, gate, [state.cpu()])
        if it == 2:                                       # same input twice: bit-identical
            for a, b in zip(prev, (g["rep"], g["rnk"], g["off"], g["og"].numpy())):
                assert np.array_equal(a, b)
        prev = (g["rep"], g["rnk"], g["off"], g["og"].numpy())


def test_error_codes_and_empty_input():
    with pytest.raises(binding.UepError):
        binding.Context(16, 2, 513, 4, 1, 8)             # E > UEP_MAX_E
    with pytest.raises(binding.UepError):
        binding.Context(16, 2, 16, 4, 5, 8)              # n_slot > 4
    with pytest.raises(binding.UepError):
        binding.Context(16, 2, 16, 4, 1, 0)              # u_min < 1
    with pytest.raises(binding.UepError):
        binding.Context(1 << 22, 8, 16, 4, 1, 8)         # S >= 2^24
    ctx = binding.Context(1024, 2, 16, 4, 1, 8)
    ws = ctx.new_workspace()
    plan = ctx.new_plan()
    count = torch.zeros(16, dtype=torch.int32, device=DEV)
    ids = torch.zeros((1024, 2), dtype=torch.int32, device=DEV)
    with pytest.raises(binding.UepError):                # misaligned ids pointer
        ctx.uep_histogram(ids.view(-1)[1:], count, ws)
    src = torch.zeros((16, 24), dtype=torch.uint8, device=DEV)     # 24 B per expert: not % 16
    dst = torch.zeros((4, 1, 24), dtype=torch.uint8, device=DEV)
    with pytest.raises(binding.UepError):
        ctx.uep_pack(plan, [src], [dst])
    # T = 0: everything runs, identity plan
    ctx0 = binding.Context(0, 2, 16, 4, 1, 8)
    ws0 = ctx0.new_workspace()
    p0 = ctx0.new_plan()
    e_ids = torch.zeros((0, 2), dtype=torch.int32, device=DEV)
    r0, k0, o0, _ = ctx0.new_outputs(None)
    ctx0.uep_balance(e_ids, None, count, p0, r0, k0, o0, None, [], [], ws0)
    torch.cuda.synchronize()
    assert int(count.sum()) == 0 and int(p0.scalars[binding.SC_N_REPLICAS]) == 0
    op = oracle.plan(np.zeros(16, np.int32), 4, 1, 8)
    hp = p0.host()
    for n in PLAN_ARRAYS[:-1]:
        assert np.array_equal(np.asarray(getattr(hp, n)).reshape(-1),
                              np.asarray(getattr(op, n)).reshape(-1)), n


def test_remap_halves_on_two_streams_and_workspace_reuse():
    """uep_remap_rank is plan-independent: run it on a second stream beside histogram + plan, join,
    then uep_remap_lookup; and reuse the same context/workspace for a second, different input."""
    T, k, E, R, ns, um = 40000, 4, 96, 24, 2, 128          # ragged: S = 160000 is not a chunk multiple
    ctx = binding.Context(T, k, E, R, ns, um)
    ws = ctx.new_workspace()
    plan = ctx.new_plan(dense_U=True)
    main, side = torch.cuda.Stream(), torch.cuda.Stream()
    for seed in (3, 4):
        ids = synth.zipf_topk_ids(T, k, E, 1.3, seed)
        gate = synth.gates_uniform_renorm(T, k, seed)
        d_ids, d_gate = ids.to(DEV), gate.to(DEV)
        count = torch.zeros(E, dtype=torch.int32, device=DEV)
        rep, rnk, off, og = ctx.new_outputs(d_gate)
        torch.cuda.synchronize()
        ctx.uep_remap_rank(d_ids, ws, side)
        ev = torch.cuda.Event()
        ev.record(side)
        ctx.uep_histogram(d_ids, count, ws, main)
        ctx.uep_plan(count, plan, ws, main)
        main.wait_event(ev)
        ctx.uep_remap_lookup(d_gate, plan, rep, rnk, off, og, ws, main)
        torch.cuda.synchronize()
        g = dict(count=count.cpu().numpy(), plan=plan.host(), rep=rep.cpu().numpy(),
                 rnk=rnk.cpu().numpy(), off=off.cpu().numpy(), og=og.cpu(), dsts=[], sentinels=[])
        assert_parity(g, oracle_chain(ids, gate, E, R, ns, um), ids, gate)


@pytest.mark.parametrize("T,k,E,R,n_slot", [
    (1, 1, 1, 1, 0),            # one slot, one expert, one rank
    (3, 1, 5, 7, 1),            # E < R: ranks without main experts
    (777, 3, 33, 5, 3),         # nothing is a multiple of anything
    (8192, 8, 512, 256, 4),     # the limits of E, R and N_slot together
    (524288, 8, 64, 8, 1),      # 4 Mi slots: many remap chunks per SM, two waves
])
def test_odd_shapes_parity(T, k, E, R, n_slot):
    S = T * k
    um = synth.stress_u_min(S, R)
    ids = synth.zipf_topk_ids(T, min(k, E), E, 1.1, 17) if k <= E else None
    if ids is None or ids.shape[1] != k:
        ids = torch.randint(0, E, (T, k), dtype=torch.int32,
                            generator=torch.Generator().manual_seed(5))
    gate = synth.gates_uniform_renorm(T, k, 9)
    g = gpu_chain(ids, gate, E, R, n_slot, um, use_balance=True)
    o = oracle_chain(ids, gate, E, R, n_slot, um)
    assert_parity(g, o, ids, gate)
    ck.check_remap(ids.numpy(), g["plan"], g["rep"], g["rnk"], g["off"])


def test_batched_planning_matches_single_and_oracle():
    """uep_plan_batched: one launch, one cluster per instance; each instance bit-identical to the
    oracle (and hence to uep_plan) — including a balanced instance (identity plan) and the
    all-to-one-expert instance."""
    E, R, ns, um, T, k = 128, 32, 2, 512, 32768, 8
    ctx = binding.Context(T, k, E, R, ns, um)
    lams = []
    for b, s in enumerate((0.0, 0.6, 1.0, 1.4, 2.0)):
        ids = synth.zipf_topk_ids(T, k, E, s, 40 + b)
        lams.append(np.bincount(ids.numpy().ravel(), minlength=E).astype(np.int32))
    one = np.zeros(E, np.int32); one[77] = T * k
    lams.append(one)
    lams.append(np.full(E, T * k // E, np.int32))          # perfectly balanced
    n = len(lams)
    counts = torch.from_numpy(np.stack(lams)).to(DEV)
    plan = ctx.new_plan(dense_U=True, batch=n)
    ctx.uep_plan_batched(n, counts, plan)
    torch.cuda.synchronize()
    for b in range(n):
        hp = plan.host(b)
        op = oracle.plan(lams[b], R, ns, um, S_total=T * k)
        for name in PLAN_ARRAYS:
            assert np.array_equal(np.asarray(getattr(hp, name)).ravel(),
                                  np.asarray(getattr(op, name)).ravel()), (b, name)


@pytest.mark.parametrize("layer,mb", [(0, 0), (17, 3), (57, 1)])
def test_training_sweep_instances_full_size(layer, mb):
    """BASELINE config 3: (layer, microbatch) instances of the DeepSeek-V3 training sweep at full
    size (Zipf s ~ U[0.6,1.6] per instance, fresh permutation), four state tensors (bf16 W + fp32
    grad, m, v; 64 K elements each stand in for 7168 x 2048), through uep_balance."""
    c = synth.CONFIGS["dsv3_train"]
    base = 20260604
    s = synth.train_sweep_s(base, layer, mb)
    assert 0.6 <= s <= 1.6
    seed = synth.instance_seed(base, layer, mb)
    ids = synth.zipf_topk_ids(c["T"], c["k"], c["E"], s, seed, device=DEV).cpu()
    gate = synth.gates_uniform_renorm(c["T"], c["k"], seed)
    states = [synth.expert_state(c["E"], 1 << 16, 11, dtype=torch.bfloat16)] + \
             [synth.expert_state(c["E"], 1 << 16, 12 + j, dtype=torch.float32) for j in range(3)]
    g = gpu_chain(ids, gate, c["E"], c["R"], c["n_slot"], c["u_min"], states=states, use_balance=True)
    o = oracle_chain(ids, gate, c["E"], c["R"], c["n_slot"], c["u_min"])
    assert_parity(g, o, ids, gate, states)
    ck.check_plan(o[0], with_layout(g["plan"]), c["u_min"])


@pytest.mark.parametrize("T,k,E,R,n_slot,s,elems", [
    (4096, 2, 16, 4, 1, 1.2, 1000 * 4 + 4),        # tiny config, ragged tile (16016 B per expert)
    (65536, 8, 128, 32, 2, 1.4, 3 * 8192 + 12),    # several tiles and a ragged tail
    (32768, 8, 64, 8, 4, 2.0, 8192),               # four slots per rank, high fan-out
])
def test_grad_reduce_and_inverse_remap(T, k, E, R, n_slot, s, elems):
    """NEXT-2: backward gradient reduction (fp32) and the inverse remap against the oracle."""
    um = synth.stress_u_min(T * k, R)
    ids = synth.zipf_topk_ids(T, k, E, s, 77)
    ctx = binding.Context(T, k, E, R, n_slot, um, gate_dtype=binding.GATE_NONE)
    ws, plan = ctx.new_workspace(), ctx.new_plan()
    d_ids = ids.to(DEV)
    count = torch.zeros(E, dtype=torch.int32, device=DEV)
    rep, rnk, off, _ = ctx.new_outputs(None)
    ctx.uep_balance(d_ids, None, count, plan, rep, rnk, off, None, [], [], ws)
    g = torch.Generator().manual_seed(5)
    mains = [torch.randn((E, elems), generator=g), torch.randn((E, 64), generator=g)]
    slots = [torch.randn((R, n_slot, elems), generator=g), torch.randn((R, n_slot, 64), generator=g)]
    d_main = [m.to(DEV) for m in mains]
    d_slot = [x.to(DEV) for x in slots]
    ctx.uep_grad_reduce(plan, d_main, d_slot)
    src = torch.full((T * k,), -7, dtype=torch.int32, device=DEV)
    ctx.uep_remap_inverse(rnk, off, plan, src)
    torch.cuda.synchronize()
    lam, _ = oracle.histogram(ids.numpy(), E)
    p = oracle.plan(lam, R, n_slot, um, S_total=T * k)
    assert p.n_replicas > 0
    for m, x, dm, dx in zip(mains, slots, d_main, d_slot):
        m64, s_ref = oracle.grad_reduce(p, m.numpy(), x.numpy())
        got = dm.cpu().numpy()
        # fp32 sum of at most 1 + n_replicas(e) terms vs the exact sum: |err| <= n * 2^-24 * sum|terms|
        mag = np.abs(m.numpy()).astype(np.float64)
        nterm = np.ones(E)
        for t in range(R):
            for q in range(n_slot):
                e = int(p.slot_expert[t, q])
                if e >= 0:
                    mag[e] += np.abs(x.numpy()[t, q]); nterm[e] += 1
        assert (np.abs(got - m64) <= (nterm[:, None] * 2.0 ** -24) * mag + 1e-30).all()
        # and bit-equal to the sequential fp32 sum in instance order (main, replicas as accepted)
        seq = m.numpy().copy()
        for e in range(E):
            for i in range(p.inst_off[e] + 1, p.inst_off[e + 1]):
                seq[e] = seq[e] + x.numpy()[p.inst_rank[i], p.inst_phys[i] - p.M]
        assert np.array_equal(got, seq)
        assert np.array_equal(dx.cpu().numpy(), s_ref)              # used slots cleared, empty untouched
    o_rep, o_rnk, o_off, _ = oracle.remap(ids.numpy(), None, p)
    assert np.array_equal(src.cpu().numpy(), oracle.inverse_remap(p, o_rnk, o_off))


@pytest.mark.parametrize("T,k,E,R,n_slot,dist", [
    (262144, 8, 256, 64, 2, "one"),        # f = 63: the closed form of the oracle pin
    (65536, 8, 128, 32, 2, "zipf1.4"),
    (65536, 8, 512, 256, 4, "zipf2"),      # fan-outs well above the relay threshold, R = 256
    (4096, 2, 16, 4, 1, "zipf1.2"),        # nothing eligible: direct sends only
])
def test_relay_plan_parity(T, k, E, R, n_slot, dist):
    """NEXT-3: relay trees and send volumes, bit-exact against the oracle."""
    um = synth.stress_u_min(T * k, R)
    ids = synth.one_expert_ids(T, k, 0) if dist == "one" else \
        synth.zipf_topk_ids(T, k, E, float(dist[4:]), 31)
    ctx = binding.Context(T, k, E, R, n_slot, um, gate_dtype=binding.GATE_NONE)
    ws, plan = ctx.new_workspace(), ctx.new_plan()
    count = torch.zeros(E, dtype=torch.int32, device=DEV)
    ctx.uep_histogram(ids.to(DEV), count, ws)
    ctx.uep_plan(count, plan, ws)
    parent = torch.full((E + R * n_slot,), -5, dtype=torch.int32, device=DEV)
    vol = torch.full((R,), -5, dtype=torch.int32, device=DEV)
    ctx.uep_relay_plan(plan, parent, vol)
    torch.cuda.synchronize()
    lam, _ = oracle.histogram(ids.numpy(), E)
    p = oracle.plan(lam, R, n_slot, um, S_total=T * k)
    o_parent, o_vol = oracle.relay_plan(p)
    assert np.array_equal(parent.cpu().numpy(), o_parent)
    assert np.array_equal(vol.cpu().numpy(), o_vol)


@pytest.mark.parametrize("T,k,E,R,n_slot,s,gate_bf16", [
    (4096, 2, 16, 4, 1, 1.2, False),         # tiny config
    (8192, 4, 64, 16, 2, 2.0, True),         # the oracle-pin shape, bf16 gates
    (65536, 8, 128, 32, 2, 1.0, False),      # GLM-Air-like: two chunks per source rank
    (4096, 8, 512, 256, 4, 2.0, False),      # R = 256: 16 tokens per source rank
    (262144, 8, 256, 64, 2, 1.0, False),     # DeepSeek-V3 prefill at full size
])
def test_remap_local_parity(T, k, E, R, n_slot, s, gate_bf16):
    """NEXT-1: source-aware reroute + token assignment, bit-exact against the oracle (O-8)."""
    um = synth.stress_u_min(T * k, R) if T * k < 2000000 else 1024
    ids = synth.zipf_topk_ids(T, k, E, s, 123)
    gate = synth.gates_softmax_bf16(T, k, 4) if gate_bf16 else synth.gates_uniform_renorm(T, k, 4)
    gd = binding.GATE_BF16 if gate_bf16 else binding.GATE_F32
    ctx = binding.Context(T, k, E, R, n_slot, um, gate_dtype=gd)
    ws, plan = ctx.new_workspace(), ctx.new_plan()
    d_ids, d_gate = ids.to(DEV), gate.to(DEV)
    count = torch.zeros(E, dtype=torch.int32, device=DEV)
    ctx.uep_histogram(d_ids, count, ws)
    ctx.uep_plan(count, plan, ws)
    rep, rnk, off, og = ctx.new_outputs(d_gate)
    infl = torch.full((R,), -3, dtype=torch.int32, device=DEV)
    ctx.uep_remap_local(d_ids, d_gate, plan, rep, rnk, off, og, infl, ws)
    torch.cuda.synchronize()
    lam, _ = oracle.histogram(ids.numpy(), E)
    p = oracle.plan(lam, R, n_slot, um, S_total=T * k)
    gbits = gate.view(torch.int16).numpy().view(np.uint16) if gate_bf16 \
        else gate.view(torch.int32).numpy().view(np.uint32)
    o_rep, o_rnk, o_off, o_og, _, o_infl = oracle.remap_local(ids.numpy(), gbits, p)
    assert np.array_equal(rep.cpu().numpy(), o_rep)
    assert np.array_equal(rnk.cpu().numpy(), o_rnk)
    assert np.array_equal(off.cpu().numpy(), o_off)
    got = og.cpu()
    got = got.view(torch.int16).numpy().view(np.uint16) if gate_bf16 else got.view(torch.int32).numpy().view(np.uint32)
    assert np.array_equal(got, o_og)
    assert np.array_equal(infl.cpu().numpy(), o_infl)


def test_balance_host_end_to_end():
    """uep_balance_host (the bench's e2e leg): pinned HOST ids and gates in, HOST remap outputs and
    scalars back, expert state packed meanwhile; the device->host copies overlap the pack."""
    T, k, E, R, ns, um = 32768, 8, 128, 32, 2, 256
    ids = synth.zipf_topk_ids(T, k, E, 1.2, 8)
    gate = synth.gates_uniform_renorm(T, k, 8)
    state = synth.expert_state(E, 1 << 18, 2)
    ctx = binding.Context(T, k, E, R, ns, um)
    ws, plan = ctx.new_workspace(), ctx.new_plan()
    h_ids, h_gate = ids.pin_memory(), gate.pin_memory()
    d_ids, d_gate = torch.empty_like(ids, device=DEV), torch.empty_like(gate, device=DEV)
    count = torch.zeros(E, dtype=torch.int32, device=DEV)
    rep, rnk, off, og = ctx.new_outputs(d_gate)
    pin = lambda t: torch.empty(t.shape, dtype=t.dtype).pin_memory()
    h_rep, h_rnk, h_off, h_og = pin(rep), pin(rnk), pin(off), pin(og)
    h_sc = torch.zeros(16, dtype=torch.int32).pin_memory()
    d_state = state.to(DEV)
    dst = torch.zeros((R, ns, state.shape[1]), dtype=state.dtype, device=DEV)
    torch.cuda.synchronize()
    stream = torch.cuda.Stream()
    for _ in range(2):                                        # twice: the side stream is re-joined
        ctx.uep_balance_host(h_ids, h_gate, d_ids, d_gate, count, plan, rep, rnk, off, og, h_rep, h_rnk,
                             h_off, h_og, h_sc, [d_state], [dst], ws, stream)
    lam, _ = oracle.histogram(ids.numpy(), E)
    p = oracle.plan(lam, R, ns, um, S_total=T * k)
    o_rep, o_rnk, o_off, o_og = oracle.remap(ids.numpy(), gate.numpy().view(np.uint32), p)
    assert np.array_equal(h_rep.numpy(), o_rep) and np.array_equal(h_rnk.numpy(), o_rnk)
    assert np.array_equal(h_off.numpy(), o_off)
    assert np.array_equal(h_og.numpy().view(np.uint32), o_og)
    assert np.array_equal(h_sc.numpy(), p.scalars)
    ref = np.zeros((R, ns, state.shape[1]), dtype=np.int16)
    oracle.pack(p.slot_expert, state.view(torch.int16).numpy(), ref)
    assert np.array_equal(dst.cpu().view(torch.int16).numpy(), ref)   # uep_balance_host returned after the pack


def test_more_error_codes():
    ctx = binding.Context(1000, 2, 16, 3, 1, 8)          # T % R != 0: no source-aware remap
    ws, plan = ctx.new_workspace(), ctx.new_plan()
    ids = torch.zeros((1000, 2), dtype=torch.int32, device=DEV)
    rep, rnk, off, _ = ctx.new_outputs(None)
    with pytest.raises(binding.UepError, match="unsupported"):
        ctx.uep_remap_local(ids, None, plan, rep, rnk, off, None, None, ws)
    ctx2 = binding.Context(1024, 2, 16, 4, 1, 8, gate_dtype=binding.GATE_NONE)
    plan2 = ctx2.new_plan()
    count = torch.zeros(16, dtype=torch.int32, device=DEV)
    ctx2.uep_plan_batched(0, count, plan2)                 # nothing to do is not an error
    with pytest.raises(binding.UepError):
        ctx2.uep_grad_reduce(plan2, [torch.zeros((16, 6), device=DEV)], [torch.zeros((4, 1, 6), device=DEV)])  # 24 B
    torch.cuda.synchronize()


@pytest.mark.parametrize("T,k,E,R,n_slot,s,G,gate_bf16", [
    (4096, 2, 16, 4, 1, 1.2, 2, False),          # tiny config on two GPUs
    (8192, 4, 64, 16, 2, 2.0, 4, True),          # bf16 gates, four shards
    (65536, 8, 128, 32, 2, 1.0, 8, False),       # GLM-Air-like on 8 GPUs (two chunks per source rank)
    (4100 * 8, 4, 64, 8, 2, 1.4, 2, False),      # ragged last chunk of every source rank's block
    (262144, 8, 256, 64, 2, 1.0, 1, False),      # full DeepSeek-V3 shape, G = 1 (the whole problem)
    (262144, 8, 256, 64, 2, 1.0, 8, False),      # and on 8 GPUs
])
def test_token_sharded_path_matches_global_remap(T, k, E, R, n_slot, s, G, gate_bf16):
    """G token shards (one per real GPU), run here one after the other on one GPU
    with the all-gather done by copying count rows between the shards' workspaces.  Every shard
    must publish the oracle's lambda and plan; the concatenated outputs must equal the oracle's
    global stable-order remap bit for bit; out_gate entries of other shards' slots stay untouched."""
    from paper_2606_04101_b200 import shard as shard_mod
    um = synth.stress_u_min(T * k, R) if T * k < 2000000 else 1024
    ids = synth.zipf_topk_ids(T, k, E, s, 77)
    ids[5, 0] = -1                                             # an invalid id on shard 0
    gate = synth.gates_softmax_bf16(T, k, 5) if gate_bf16 else synth.gates_uniform_renorm(T, k, 5)
    gd = binding.GATE_BF16 if gate_bf16 else binding.GATE_F32
    ctx = binding.Context(T, k, E, R, n_slot, um, gate_dtype=gd)
    S, Sl = T * k, T * k // G
    layers = [shard_mod.TokenShardedLayer(ctx, g, G) for g in range(G)]
    d_ids = ids.to(DEV).reshape(-1)
    d_gate = gate.to(DEV).reshape(-1)
    off0, nb = ctx.uep_shard_rows(0, G)
    for g, L in enumerate(layers):
        assert ctx.uep_shard_rows(g, G) == (off0 + g * nb, nb)
        L.out_gate = torch.full((S,), 0x7fff if gate_bf16 else 0x7fc0dead, dtype=torch.int32, device=DEV) \
            .to(torch.int16 if gate_bf16 else torch.int32).view(gate.dtype)
        ctx.uep_shard_count(g, G, d_ids[g * Sl:(g + 1) * Sl], L.ws)
    torch.cuda.synchronize()
    # the exchange, emulated: every workspace receives every shard's rows
    rows = torch.cat([L.ws[off0 + g * nb: off0 + (g + 1) * nb] for g, L in enumerate(layers)])
    for L in layers:
        L.ws[off0: off0 + G * nb] = rows
    for g, L in enumerate(layers):
        L.n_inflight.fill_(-3)
        ctx.uep_shard_finish(g, G, d_gate[g * Sl:(g + 1) * Sl], L.expert_count, L.plan, L.out_replica,
                             L.out_rank, L.out_offset, L.out_gate, L.n_inflight, L.ws)
    torch.cuda.synchronize()

    lam, p, o_rep, o_rnk, o_off, o_og = oracle_chain(ids, gate, E, R, n_slot, um)
    # per-chunk count rows = plain bincount of each chunk (the subdivided rows of Lambda[R,E])
    E_pad = (E + 3) // 4 * 4
    block = (T // R) * k
    got_rows = rows.view(torch.int32).cpu().numpy().reshape(-1, E_pad)
    cpg = got_rows.shape[0] // R
    flat = ids.numpy().reshape(-1)
    Lam = np.zeros((R, E), dtype=np.int64)
    for r in range(R):
        Lam[r] = got_rows[r * cpg:(r + 1) * cpg, :E].sum(axis=0)
        blk = flat[r * block:(r + 1) * block]
        assert np.array_equal(Lam[r], np.bincount(blk[(blk >= 0) & (blk < E)], minlength=E))
    assert np.array_equal(Lam.sum(axis=0), lam)
    for g, L in enumerate(layers):
        assert np.array_equal(L.expert_count.cpu().numpy()[:E], lam)
        hp = L.plan.host()
        for n in PLAN_ARRAYS:
            if n == "U":                                       # the layers' plans carry no dense U
                continue
            assert np.array_equal(np.asarray(getattr(hp, n)).reshape(-1), np.asarray(getattr(p, n)).reshape(-1)), (g, n)
    cat = lambda name: torch.cat([getattr(L, name)[:Sl] for L in layers]).cpu().numpy().reshape(T, k)
    assert np.array_equal(cat("out_replica"), o_rep)
    assert np.array_equal(cat("out_rank"), o_rnk)
    assert np.array_equal(cat("out_offset"), o_off)
    # gates: shard g wrote exactly the dispatch positions of its own slots
    bits = lambda t: t.view(torch.int16).cpu().numpy().view(np.uint16) if gate_bf16 \
        else t.view(torch.int32).cpu().numpy().view(np.uint32)
    sentinel = np.uint16(0x7fff) if gate_bf16 else np.uint32(0x7fc0dead)
    rank_base = np.asarray(p.rank_base)
    dest = np.where(o_rnk.reshape(-1) >= 0, rank_base[np.maximum(o_rnk.reshape(-1), 0)] + o_off.reshape(-1), -1)
    for g, L in enumerate(layers):
        mine = dest[g * Sl:(g + 1) * Sl]
        mine = mine[mine >= 0]
        gb = bits(L.out_gate)
        assert np.array_equal(gb[mine], o_og[mine])
        other = np.ones(S, dtype=bool)
        other[mine] = False
        assert (gb[other] == sentinel).all()
    # in-flight slots per source rank (slots whose destination is not their source rank)
    src = np.arange(S) // block
    fly = np.bincount(src[(o_rnk.reshape(-1) >= 0) & (o_rnk.reshape(-1) != src)], minlength=R)
    rps = R // G
    for g, L in enumerate(layers):
        got = L.n_inflight.cpu().numpy()[:R]
        assert np.array_equal(got[g * rps:(g + 1) * rps], fly[g * rps:(g + 1) * rps])
        assert (np.delete(got, np.s_[g * rps:(g + 1) * rps]) == -3).all()


def test_token_sharded_step_captured_as_its_first_use_full_size():
    """uep_shard_count forks the rank kernel onto the context's side stream and uep_shard_finish joins
    it in front of the lookup.  Under stream capture that join is a PROGRAMMATIC edge (the lookup is
    launched with the programmatic attribute), so the rank kernel must not trigger early there: the
    lookup's prologue reads what it writes.  A fresh context, workspace never used, the step captured
    without an eager run in front of it (stale ranks of an earlier identical run would hide a race),
    four layers in one graph, replayed twice with new ids each time; every output against the oracle."""
    from paper_2606_04101_b200 import shard as shard_mod
    T, k, E, R, n_slot, um, n = 262144, 8, 256, 64, 2, 1024, 4
    ctx = binding.Context(T, k, E, R, n_slot, um, gate_dtype=binding.GATE_F32)
    layers = [shard_mod.TokenShardedLayer(ctx, 0, 1) for _ in range(n)]       # four layers, one context
    d_ids = [torch.empty(T * k, dtype=torch.int32, device=DEV) for _ in range(n)]
    d_gate = [torch.empty(T * k, dtype=torch.float32, device=DEV) for _ in range(n)]
    for L in layers:
        L.out_gate = torch.zeros(T * k, dtype=torch.float32, device=DEV)
    st = torch.cuda.Stream()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.stream(st):
        with torch.cuda.graph(g, stream=st):
            for i, L in enumerate(layers):
                L.step(d_ids[i], d_gate[i])
    for rep in range(2):
        ins = []
        for i in range(n):
            ids = synth.zipf_topk_ids(T, k, E, 1.0, 900 + 10 * rep + i)
            gate = synth.gates_uniform_renorm(T, k, 900 + 10 * rep + i)
            d_ids[i].copy_(ids.reshape(-1))
            d_gate[i].copy_(gate.reshape(-1))
            ins.append((ids, gate))
            for t in (layers[i].out_replica, layers[i].out_rank, layers[i].out_offset):
                t.fill_(-9)
        torch.cuda.synchronize()
        with torch.cuda.stream(st):
            g.replay()
        torch.cuda.synchronize()
        for (ids, gate), L in zip(ins, layers):
            lam, p, o_rep, o_rnk, o_off, o_og = oracle_chain(ids, gate, E, R, n_slot, um)
            assert np.array_equal(L.expert_count.cpu().numpy()[:E], lam)
            assert np.array_equal(L.out_replica.cpu().numpy().reshape(T, k), o_rep)
            assert np.array_equal(L.out_rank.cpu().numpy().reshape(T, k), o_rnk)
            assert np.array_equal(L.out_offset.cpu().numpy().reshape(T, k), o_off)
            nv = int(p.rank_base[-1])
            assert np.array_equal(L.out_gate.view(torch.int32).cpu().numpy().view(np.uint32)[:nv], o_og[:nv])


def test_token_shard_argument_errors():
    ctx = binding.Context(4096, 2, 16, 4, 1, 64)
    ws = ctx.new_workspace()
    ids = torch.zeros(4096, dtype=torch.int32, device=DEV)
    for shard, G in ((0, 3), (2, 2), (-1, 2), (0, 0)):          # G must divide R; 0 <= shard < G
        with pytest.raises(binding.UepError):
            ctx.uep_shard_count(shard, G, ids, ws)
        with pytest.raises(binding.UepError):
            ctx.uep_shard_rows(shard, G)
    with pytest.raises(binding.UepError):                        # T % R != 0: unsupported
        c2 = binding.Context(4098, 2, 16, 4, 1, 64)
        c2.uep_shard_count(0, 2, ids, c2.new_workspace())


@pytest.mark.parametrize("seed", [1, 2, 3])
def test_random_shapes_fuzz(seed):
    """Seeded random walk over the argument space (shapes incl. E, R not powers of two and E < R,
    k, n_slot 0..4, u_min, beta, both floor modes, home maps, skew, invalid ids, with/without
    gates, uep_balance or the four calls): everything bit-exact against the oracle."""
    import random
    rng = random.Random(seed)
    for _ in range(120):
        k = rng.choice([1, 2, 4, 8])
        E = rng.choice([1, 2, 3, 7, 16, 33, 64, 100, 128, 255, 256, 300, 512, rng.randint(1, 512)])
        R = rng.choice([1, 2, 4, 8, 16, 32, 64, 128, 256, rng.randint(1, 256)])
        n_slot = rng.randint(0, 4)
        T = rng.choice([1, 5, 64, 1000, 4096, 10000, rng.randint(1, 20000)])
        k = k if k <= E else 1
        S = T * k
        u_min = rng.choice([1, 2, 7, max(1, S // R // 32), max(1, S // R // 8), max(1, S // R // 2),
                            rng.randint(1, max(1, S // R))])
        beta = rng.choice([(101, 100), (1, 1), (11, 10), (3, 2), (1001, 1000)])
        strict = rng.random() < 0.5
        kind = rng.choice(["zipf", "zipf", "zipf", "uniform", "one", "few"])
        sd = rng.randint(0, 1 << 30)
        g = torch.Generator().manual_seed(sd)
        if kind == "zipf":
            ids = synth.zipf_topk_ids(T, k, E, rng.choice([0.0, 0.6, 1.0, 1.4, 2.0, 3.0]), sd)
        elif kind == "uniform":
            ids = torch.randint(0, E, (T, k), dtype=torch.int32, generator=g)
        elif kind == "one":
            ids = torch.full((T, k), rng.randrange(E), dtype=torch.int32)
        else:
            few = torch.tensor([rng.randrange(E) for _ in range(3)], dtype=torch.int32)
            ids = few[torch.randint(0, 3, (T, k), generator=g)]
        if rng.random() < 0.3:
            bad = torch.tensor(rng.choice([-1, E, 1 << 20]), dtype=torch.int32)
            ids = torch.where(torch.rand((T, k), generator=g) < 0.01, bad, ids)
        gate = None if rng.random() < 0.2 else synth.gates_uniform_renorm(T, k, sd)
        home = np.random.default_rng(sd).integers(0, R, size=E).astype(np.int32) if rng.random() < 0.25 else None
        case = dict(T=T, k=k, E=E, R=R, n_slot=n_slot, u_min=u_min, beta=beta, strict=strict, kind=kind, sd=sd)
        try:
            go = gpu_chain(ids, gate, E, R, n_slot, u_min,
                           binding.FLOOR_STRICT if strict else binding.FLOOR_TOLERANT, home, beta=beta,
                           use_balance=rng.random() < 0.5)
            oo = oracle_chain(ids, gate, E, R, n_slot, u_min,
                              oracle.FLOOR_STRICT if strict else oracle.FLOOR_TOLERANT, home, beta=beta)
            assert_parity(go, oo, ids, gate)
        except Exception as ex:                                  # name the case that failed
            raise AssertionError(f"fuzz case {case}") from ex


@pytest.mark.skipif(not os.environ.get("UEP_FUZZ_SECONDS"), reason="opt-in: UEP_FUZZ_SECONDS=<budget>")
def test_long_fuzz_opt_in():
    """The walk of test_random_shapes_fuzz for a time budget, with token counts up to 300 000 (many
    chunks, instance boundaries inside chunks) and, through the bodies of the NEXT-row tests, random
    arguments for uep_remap_local, the token-sharded path and relay plans.
    Last run, at the final sources of round 2 with UEP_FUZZ_SECONDS=900 on one B200: 42 320 chain
    cases and 2 091 sets of NEXT-row cases, no mismatch (earlier developer runs of similar walks
    rejected only shard slices that are not 16-byte aligned,
    UEP_ERR_INVALID_ARG as include/uep.h states — this walk keeps them aligned)."""
    import random
    import time
    budget = float(os.environ["UEP_FUZZ_SECONDS"])
    t0, seed, n_chain, n_next = time.time(), 1000, 0, 0
    while time.time() - t0 < budget:
        seed += 1
        rng = random.Random(seed)
        for _ in range(20):
            k = rng.choice([1, 2, 4, 8])
            E = rng.choice([16, 33, 64, 100, 128, 255, 256, 300, 481, 500, 512, rng.randint(1, 512)])
            R = rng.choice([2, 4, 8, 16, 32, 64, 128, 256, rng.randint(1, 256)])
            n_slot = rng.randint(0, 4)
            T = rng.choice([4096, 20000, 65536, 100000, 262144, rng.randint(1, 300000)])
            k = k if k <= E else 1
            S = T * k
            u_min = rng.choice([1, 7, max(1, S // R // 32), max(1, S // R // 8), max(1, S // R // 2),
                                rng.randint(1, max(1, S // R))])
            beta = rng.choice([(101, 100), (1, 1), (11, 10), (3, 2), (1001, 1000)])
            strict = rng.random() < 0.5
            sd = rng.randint(0, 1 << 30)
            g = torch.Generator().manual_seed(sd)
            kind = rng.choice(["zipf", "zipf", "uniform", "one"])
            if kind == "zipf":
                ids = synth.zipf_topk_ids(T, k, E, rng.choice([0.0, 0.6, 1.0, 1.4, 2.0, 3.0]), sd)
            elif kind == "uniform":
                ids = torch.randint(0, E, (T, k), dtype=torch.int32, generator=g)
            else:
                ids = torch.full((T, k), rng.randrange(E), dtype=torch.int32)
            if rng.random() < 0.3:
                bad = torch.tensor(rng.choice([-1, E, 1 << 20]), dtype=torch.int32)
                ids = torch.where(torch.rand((T, k), generator=g) < 0.01, bad, ids)
            gate = None if rng.random() < 0.2 else synth.gates_uniform_renorm(T, k, sd)
            case = dict(T=T, k=k, E=E, R=R, n_slot=n_slot, u_min=u_min, beta=beta, strict=strict, kind=kind, sd=sd)
            try:
                go = gpu_chain(ids, gate, E, R, n_slot, u_min,
                               binding.FLOOR_STRICT if strict else binding.FLOOR_TOLERANT, None, beta=beta,
                               use_balance=rng.random() < 0.5)
                oo = oracle_chain(ids, gate, E, R, n_slot, u_min,
                                  oracle.FLOOR_STRICT if strict else oracle.FLOOR_TOLERANT, None, beta=beta)
                assert_parity(go, oo, ids, gate)
                go["ctx"].close()
                n_chain += 1
            except Exception as ex:
                raise AssertionError(f"fuzz case {case}") from ex
        # NEXT rows: T a multiple of R, at least 8 tokens, shard slices 16-byte aligned
        R = rng.choice([1, 2, 4, 8, 16, 32, 64, 128, 256])
        E = min(max(rng.choice([R, 2 * R, 4 * R, 8 * R]), 8), 512)
        k = min(rng.choice([1, 2, 4, 8]), E)
        T = R * rng.choice([8, 16, 104, 512, 1000, 4096, 8 * rng.randint(1, 400)])
        if T * k > 3_000_000:
            continue
        n_slot, s, bf = rng.randint(0, 4), rng.choice([0.0, 0.6, 1.0, 1.4, 2.0, 3.0]), rng.random() < 0.4
        G = rng.choice([g_ for g_ in (1, 2, 4, 8, 16) if R % g_ == 0])
        test_remap_local_parity(T, k, E, R, n_slot, s, bf)
        test_token_sharded_path_matches_global_remap(T, k, E, R, n_slot, s, G, bf)
        if n_slot > 0:
            test_relay_plan_parity(T, k, E, R, n_slot, rng.choice(["one", "zipf1.4", "zipf2", "zipf1.2"]))
        n_next += 1
    print(f"long fuzz: {n_chain} chain cases, {n_next} sets of NEXT-row cases, no mismatch")


def _seq_grad(p, m, x):
    """sequential fp32 sum in instance order (what the kernel must reproduce bit for bit)"""
    seq = m.copy()
    for e in range(p.E):
        for i in range(p.inst_off[e] + 1, p.inst_off[e + 1]):
            seq[e] = seq[e] + x[p.inst_rank[i], p.inst_phys[i] - p.M]
    return seq


@pytest.mark.parametrize("seed", [0, 1])
def test_streaming_kernels_odd_sizes_streams_and_replay(seed):
    """pack / grad_reduce hand their tiles out from self-resetting counters: tensor sizes that are
    not a multiple of the tile (down to 16 B), up to 8 tensors, launches in flight on three streams
    of one context at once, and graph replays must all stay byte-exact / bit-exact."""
    import random
    rng = random.Random(seed)
    T, k, E, R, n_slot = 16384, 4, 64, 16, 2
    um = synth.stress_u_min(T * k, R)
    ctx = binding.Context(T, k, E, R, n_slot, um, gate_dtype=binding.GATE_NONE)
    plans, oplans = [], []
    for i in range(3):
        ids = synth.zipf_topk_ids(T, k, E, 1.2 + 0.4 * i, 10 * seed + i)
        ws, plan = ctx.new_workspace(), ctx.new_plan()
        count = torch.zeros(E, dtype=torch.int32, device=DEV)
        ctx.uep_histogram(ids.to(DEV), count, ws)
        ctx.uep_plan(count, plan, ws)
        lam, _ = oracle.histogram(ids.numpy(), E)
        plans.append(plan)
        oplans.append(oracle.plan(lam, R, n_slot, um, S_total=T * k))
        assert oplans[-1].n_replicas > 0
    sizes = [16, 48, 8192, 16384, 16400, 40000 // 16 * 16, 1 << 20, rng.randrange(1, 9000) * 16]
    nt = [8, 3, 1]
    g = torch.Generator().manual_seed(seed)
    srcs, dsts, sents, mains, slots, dmain, dslot = [], [], [], [], [], [], []
    for i in range(3):                                       # one tensor set per stream
        bs = rng.sample(sizes, nt[i])
        srcs.append([torch.randint(0, 256, (E, b), dtype=torch.uint8, generator=g).to(DEV) for b in bs])
        sents.append([torch.randint(0, 256, (R, n_slot, b), dtype=torch.uint8, generator=g) for b in bs])
        dsts.append([s.to(DEV) for s in sents[i]])
        mains.append([torch.randn((E, b // 4), generator=g) for b in bs])
        slots.append([torch.randn((R, n_slot, b // 4), generator=g) for b in bs])
        dmain.append([m.to(DEV) for m in mains[i]])
        dslot.append([x.to(DEV) for x in slots[i]])
    streams = [torch.cuda.Stream() for _ in range(3)]
    torch.cuda.synchronize()
    for rep in range(3):                                     # pack is idempotent: repeat it
        for i, st in enumerate(streams):
            with torch.cuda.stream(st):
                ctx.uep_pack(plans[i], srcs[i], dsts[i])
    for i, st in enumerate(streams):
        with torch.cuda.stream(st):
            ctx.uep_grad_reduce(plans[i], dmain[i], dslot[i])
            ctx.uep_grad_reduce(plans[i], dmain[i], dslot[i])   # slots are zero now: adds nothing
    torch.cuda.synchronize()
    for i in range(3):
        p = oplans[i]
        for s_, d_, sn in zip(srcs[i], dsts[i], sents[i]):
            ref = sn.numpy().reshape(R, n_slot, -1).copy()
            oracle.pack(p.slot_expert, np.ascontiguousarray(s_.cpu().numpy()), ref)
            assert np.array_equal(d_.cpu().numpy(), ref)
        for m, x, dm, dx in zip(mains[i], slots[i], dmain[i], dslot[i]):
            assert np.array_equal(dm.cpu().numpy(), _seq_grad(p, m.numpy(), x.numpy()))
            _, s_ref = oracle.grad_reduce(p, m.numpy(), x.numpy())
            assert np.array_equal(dx.cpu().numpy(), s_ref)
    # graph replay: the counters must be rearmed by every launch
    st = streams[0]
    for d_, sn in zip(dsts[0], sents[0]):
        d_.copy_(sn)
    gr = torch.cuda.CUDAGraph()
    with torch.cuda.stream(st):
        with torch.cuda.graph(gr, stream=st):
            ctx.uep_pack(plans[0], srcs[0], dsts[0])
            ctx.uep_pack(plans[1], srcs[0], dsts[0])
        for _ in range(4):
            gr.replay()
    torch.cuda.synchronize()
    for s_, d_, sn in zip(srcs[0], dsts[0], sents[0]):       # plan 0 then plan 1 over the same buffers
        ref = sn.numpy().reshape(R, n_slot, -1).copy()
        oracle.pack(oplans[0].slot_expert, np.ascontiguousarray(s_.cpu().numpy()), ref)
        oracle.pack(oplans[1].slot_expert, np.ascontiguousarray(s_.cpu().numpy()), ref)
        assert np.array_equal(d_.cpu().numpy(), ref)


@pytest.mark.parametrize("n_slot,u_min,s,strict", [
    (1, 1024, 1.0, False),     # tau* ~1000 above tau_lo: the path leaves the all-feasible spine mid-way
    (2, 8192, 1.0, False),     # coarse floor
    (2, 1024, 1.0, True),      # Alg. 1 verbatim: feasibility not monotone, tau* far from tau_lo
    (4, 1, 2.0, True),         # u_min = 1: strict == tolerant, long accept lists
    (2, 1024, 0.0, False),     # balanced input: few or no probes
])
def test_planner_paths_off_the_spine_full_size(n_slot, u_min, s, strict):
    """The planner's first round speculates along the all-feasible spine of the bisection tree;
    whatever the path really is, plan and scalars (tau, n_probes on the SEQUENTIAL path, ...) must
    equal the oracle's.  DeepSeek-V3 shape, several instances each."""
    T, k, E, R = 262144, 8, 256, 64
    mode_g = binding.FLOOR_STRICT if strict else binding.FLOOR_TOLERANT
    mode_o = oracle.FLOOR_STRICT if strict else oracle.FLOOR_TOLERANT
    ctx = binding.Context(T, k, E, R, n_slot, u_min, floor_mode=mode_g, gate_dtype=binding.GATE_NONE)
    ws = ctx.new_workspace()
    seen = set()
    for seed in range(4):
        ids = synth.zipf_topk_ids(T, k, E, s, 300 + seed)
        plan = ctx.new_plan(dense_U=True)
        count = torch.zeros(E, dtype=torch.int32, device=DEV)
        ctx.uep_histogram(ids.to(DEV), count, ws)
        ctx.uep_plan(count, plan, ws)
        torch.cuda.synchronize()
        lam, _ = oracle.histogram(ids.numpy(), E)
        p = oracle.plan(lam, R, n_slot, u_min, 101, 100, mode_o, None, S_total=T * k)
        hp = plan.host()
        for n in PLAN_ARRAYS:
            assert np.array_equal(np.asarray(getattr(hp, n)).reshape(-1), np.asarray(getattr(p, n)).reshape(-1)), n
        sc = np.asarray(hp.scalars)
        seen.add((int(sc[binding.SC_TAU] - sc[binding.SC_TAU_LO0]) > 0, int(sc[binding.SC_N_PROBES]) > 0))
    assert seen                                   # (documentation of what the cases exercised)


@pytest.mark.parametrize("entry", ["balance", "remap", "remap_local"])
def test_back_to_back_calls_in_one_graph_full_size(entry):
    """The launch configuration bench.py times: several instances of the DeepSeek-V3 shape run
    back to back in ONE CUDA graph on one workspace (each call's kernels are launched
    programmatically dependent on their predecessors, so a missing dependency between the
    prefix rows of one call and the lookup of the same or the next call shows up here and not in
    a single call).  Every instance's outputs are compared with the oracle, after three replays."""
    c = synth.CONFIGS["dsv3_prefill"]
    T, k, E, R, ns, um = c["T"], c["k"], c["E"], c["R"], c["n_slot"], c["u_min"]
    n_inst = 5
    ctx = binding.Context(T, k, E, R, ns, um)
    ws = ctx.new_workspace()
    ins, outs = [], []
    for b in range(n_inst):
        ids = synth.zipf_topk_ids(T, k, E, 0.7 + 0.2 * b, 900 + b, device=DEV).cpu()
        gate = synth.gates_uniform_renorm(T, k, 40 + b)
        d_ids, d_gate = ids.to(DEV), gate.to(DEV)
        rep, rnk, off, og = ctx.new_outputs(d_gate)
        ins.append((ids, gate, d_ids, d_gate))
        outs.append(dict(count=torch.zeros(E, dtype=torch.int32, device=DEV), plan=ctx.new_plan(),
                         rep=rep, rnk=rnk, off=off, og=og,
                         infl=torch.zeros(R, dtype=torch.int32, device=DEV)))
    stream = torch.cuda.Stream()
    stream.wait_stream(torch.cuda.current_stream())

    def call(b):
        _, _, d_ids, d_gate = ins[b]
        o = outs[b]
        if entry == "balance":
            ctx.uep_balance(d_ids, d_gate, o["count"], o["plan"], o["rep"], o["rnk"], o["off"],
                            o["og"], [], [], ws)
        elif entry == "remap":
            ctx.uep_remap(d_ids, d_gate, o["plan"], o["rep"], o["rnk"], o["off"], o["og"], ws)
        else:
            ctx.uep_remap_local(d_ids, d_gate, o["plan"], o["rep"], o["rnk"], o["off"], o["og"],
                                o["infl"], ws)

    with torch.cuda.stream(stream):
        for b in range(n_inst):                      # plans for the remap-only entries; warm-up
            ctx.uep_histogram(ins[b][2], outs[b]["count"], ws)
            ctx.uep_plan(outs[b]["count"], outs[b]["plan"], ws)
            call(b)
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=stream):
            for b in range(n_inst):
                call(b)
    torch.cuda.synchronize()
    for o in outs:
        for t in (o["rep"], o["rnk"], o["off"], o["og"]):
            t.fill_(0)
    torch.cuda.synchronize()
    for _ in range(3):
        graph.replay()
    torch.cuda.synchronize()
    for b in range(n_inst):
        ids, gate = ins[b][0], ins[b][1]
        lam, p, rep, rnk, off, og = oracle_chain(ids, gate, E, R, ns, um)
        o = outs[b]
        assert np.array_equal(o["count"].cpu().numpy(), lam)
        assert np.array_equal(np.asarray(o["plan"].host().inst_cum).ravel(), np.asarray(p.inst_cum).ravel())
        gbits = gate.view(torch.int32).numpy().view(np.uint32)
        if entry == "remap_local":
            rep, rnk, off, og, _, o_infl = oracle.remap_local(ids.numpy(), gbits, p)
            assert np.array_equal(o["infl"].cpu().numpy(), o_infl)
        assert np.array_equal(o["rep"].cpu().numpy(), rep), (entry, b)
        assert np.array_equal(o["rnk"].cpu().numpy(), rnk), (entry, b)
        assert np.array_equal(o["off"].cpu().numpy(), off), (entry, b)
        nv = int(p.rank_base[-1])
        assert np.array_equal(o["og"].cpu().view(torch.int32).numpy().view(np.uint32)[:nv], og[:nv])


def test_histogram_accumulator_stays_clean_between_calls():
    """uep_histogram and uep_balance share the workspace's accumulator: each must leave it zero
    (publish_kernel / the lookup clear it).  Many calls of both kinds on ONE workspace, back to back
    in one CUDA graph and replayed, with different inputs and an invalid id: every count exact."""
    T, k, E, R, ns, um = 30001, 8, 200, 25, 2, 64
    ctx = binding.Context(T, k, E, R, ns, um)
    ws, plan = ctx.new_workspace(), ctx.new_plan()
    n = 6
    ids = [synth.zipf_topk_ids(T, k, E, 0.5 + 0.3 * b, 70 + b) for b in range(n)]
    ids[2][5, 1] = E + 3                                   # skipped, not counted (S14)
    d_ids = [x.to(DEV) for x in ids]
    counts = [torch.full((E,), -1, dtype=torch.int32, device=DEV) for _ in range(n)]
    rep, rnk, off, _ = ctx.new_outputs(None)
    stream = torch.cuda.Stream()
    stream.wait_stream(torch.cuda.current_stream())

    def run_all():
        for b in range(n):
            if b % 3 == 2:
                ctx.uep_balance(d_ids[b], None, counts[b], plan, rep, rnk, off, None, [], [], ws)
            else:
                ctx.uep_histogram(d_ids[b], counts[b], ws)

    with torch.cuda.stream(stream):
        run_all()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=stream):
            run_all()
    torch.cuda.synchronize()
    for _ in range(3):
        for c in counts:
            c.fill_(-1)
        graph.replay()
        torch.cuda.synchronize()
        for b in range(n):
            lam, bad = oracle.histogram(ids[b].numpy(), E)
            assert np.array_equal(counts[b].cpu().numpy(), lam), b
            assert bad == (1 if b == 2 else 0)
    # the chunk table (by-product of uep_histogram): its rows sum to the counts
    ctx.uep_histogram(d_ids[0], counts[0], ws)
    torch.cuda.synchronize()
    assert int(counts[0].sum()) == T * k


def _fullsize_plan(ctx, c, seed, zipf_s=1.0):
    """ids of one full-size instance on the device, and the ORACLE's plan for them."""
    ids = synth.zipf_topk_ids(c["T"], c["k"], c["E"], zipf_s, seed, device=DEV)
    lam, _ = oracle.histogram(ids.cpu().numpy(), c["E"])
    p = oracle.plan(lam, c["R"], c["n_slot"], c["u_min"], S_total=c["T"] * c["k"])
    assert p.n_replicas > 8
    return ids, lam, p


def test_pack_at_the_benchmarked_byte_size():
    """uep_pack at the size bench.py times (dsv3_prefill: 88 080 384 B per expert, 22.5 GB of source,
    11.3 GB of slot buffers: byte offsets beyond 4 GiB, 5376 tiles per expert), once through
    uep_balance (the timed launch configuration) and once through uep_pack on another plan.  Compared
    on the device, slot by slot (BASELINE.md §5 allows the chunk-wise compare): every destination
    slot equals the source expert that the ORACLE's slot_expert names, byte for byte, and every empty
    slot still holds the sentinel ("remains empty"; weight distribution PAPER.md:162)."""
    c = synth.CONFIGS["dsv3_prefill"]
    T, k, E, R, ns, um = c["T"], c["k"], c["E"], c["R"], c["n_slot"], c["u_min"]
    elems = c["state"][0][1]
    assert elems * 2 == 88080384
    ctx = binding.Context(T, k, E, R, ns, um)
    ws, plan = ctx.new_workspace(), ctx.new_plan()
    src = synth.expert_state(E, elems, 7, dtype=torch.bfloat16, device=DEV)
    assert src.numel() * 2 > (1 << 34)                              # > 16 GiB: 64-bit offsets matter
    dst = torch.empty((R, ns, elems), dtype=torch.bfloat16, device=DEV)
    SENT = 0x5A5B
    for seed, through_balance in ((4242, True), (4243, False)):
        ids, lam, p = _fullsize_plan(ctx, c, seed)
        dst.view(torch.int16).fill_(SENT)
        count = torch.zeros(E, dtype=torch.int32, device=DEV)
        gate = synth.gates_uniform_renorm(T, k, 6, device=DEV)
        rep, rnk, off, og = ctx.new_outputs(gate)
        if through_balance:
            ctx.uep_balance(ids, gate, count, plan, rep, rnk, off, og, [src], [dst], ws)
        else:
            ctx.uep_histogram(ids, count, ws)
            ctx.uep_plan(count, plan, ws)
            ctx.uep_pack(plan, [src], [dst])
        torch.cuda.synchronize()
        assert np.array_equal(plan.host().slot_expert, p.slot_expert)
        n_used = 0
        for t in range(R):
            for q in range(ns):
                e = int(p.slot_expert[t, q])
                if e >= 0:
                    n_used += 1
                    assert torch.equal(dst[t, q].view(torch.int16), src[e].view(torch.int16)), (t, q, e)
                else:
                    assert bool((dst[t, q].view(torch.int16) == SENT).all()), (t, q)
        assert n_used == p.n_replicas


def test_grad_reduce_at_the_benchmarked_byte_size():
    """uep_grad_reduce over fp32 [E, 7168 x 2048] main gradients (15 GB) and [R, n_slot, 7168 x 2048]
    slot gradients (7.5 GB) — the size bench.py times.  On the device, expert by
    expert as the ORACLE's plan names them: main = the sequential fp32 sum in instance order (bit for
    bit), used slots zero, empty slots and unreplicated experts untouched; and on 4096 sampled
    columns the fp64 oracle O-5 within n_terms x 2^-24 x sum|terms|."""
    c = synth.CONFIGS["dsv3_prefill"]
    T, k, E, R, ns, um = c["T"], c["k"], c["E"], c["R"], c["n_slot"], c["u_min"]
    B = 7168 * 2048
    ctx = binding.Context(T, k, E, R, ns, um, gate_dtype=binding.GATE_NONE)
    ws, plan = ctx.new_workspace(), ctx.new_plan()
    ids, lam, p = _fullsize_plan(ctx, c, 99)
    count = torch.zeros(E, dtype=torch.int32, device=DEV)
    ctx.uep_histogram(ids, count, ws)
    ctx.uep_plan(count, plan, ws)
    main0 = synth.expert_state(E, B, 21, dtype=torch.float32, device=DEV, std=1.0)
    slot0 = synth.expert_state(R * ns, B, 22, dtype=torch.float32, device=DEV, std=1.0).view(R, ns, B)
    main, slot = main0.clone(), slot0.clone()
    ctx.uep_grad_reduce(plan, [main], [slot])
    torch.cuda.synchronize()
    assert np.array_equal(plan.host().inst_rank, p.inst_rank)
    used = np.zeros((R, ns), dtype=bool)
    for e in range(E):
        exp = main0[e]
        lo, hi = int(p.inst_off[e]), int(p.inst_off[e + 1])
        for i in range(lo + 1, hi):                                   # instance order (S11)
            t, q = int(p.inst_rank[i]), int(p.inst_phys[i]) - p.M
            exp = exp + slot0[t, q]
            used[t, q] = True
        assert torch.equal(main[e], exp), e
    assert used.sum() == p.n_replicas and np.array_equal(used, p.slot_expert >= 0)
    for t in range(R):
        for q in range(ns):
            if used[t, q]:
                assert not bool(slot[t, q].any()), (t, q)             # cleared in place
            else:
                assert torch.equal(slot[t, q], slot0[t, q]), (t, q)   # empty slots untouched
    # fp64 oracle on sampled columns (incl. the first and last element of the tensor)
    g = torch.Generator().manual_seed(1)
    cols = torch.cat([torch.tensor([0, B - 1]), torch.randint(0, B, (4094,), generator=g)]).to(DEV)
    m_s, s_s = main0[:, cols].cpu().numpy(), slot0[:, :, cols].cpu().numpy()
    m64, s_ref = oracle.grad_reduce(p, m_s, s_s)
    got = main[:, cols].cpu().numpy()
    mag, nterm = np.abs(m_s).astype(np.float64), np.ones(E)
    for t in range(R):
        for q in range(ns):
            e = int(p.slot_expert[t, q])
            if e >= 0:
                mag[e] += np.abs(s_s[t, q]); nterm[e] += 1
    assert (np.abs(got - m64) <= (nterm[:, None] * 2.0 ** -24) * mag + 1e-30).all()
    assert np.array_equal(slot[:, :, cols].cpu().numpy(), s_ref)


def test_balance_failure_mid_chain_leaves_stream_and_workspace_usable():
    """A stage that fails to launch part-way through uep_balance (here: uep_pack refuses a tensor
    with more tiles than its unit counter can index, after histogram, rank and plan were enqueued)
    must still join the internal side stream back into the caller's stream — inside a stream capture
    too, which has to end cleanly — and must leave the workspace's accumulator clean, so that the
    next call on the same workspace publishes exact counts."""
    import ctypes
    T, k, E, R, ns, um = 16384, 4, 64, 16, 2, 64
    ctx = binding.Context(T, k, E, R, ns, um, gate_dtype=binding.GATE_NONE)
    ws, plan = ctx.new_workspace(), ctx.new_plan()
    ids = synth.zipf_topk_ids(T, k, E, 1.3, 3)
    d_ids = ids.to(DEV)
    count = torch.zeros(E, dtype=torch.int32, device=DEV)
    rep, rnk, off, _ = ctx.new_outputs(None)
    src = torch.zeros((E, 16), dtype=torch.uint8, device=DEV)
    dst = torch.zeros((R, ns, 16), dtype=torch.uint8, device=DEV)
    L = binding.lib()

    def bad_call(stream):
        srcs = (ctypes.c_void_p * 1)(src.data_ptr())
        dsts = (ctypes.c_void_p * 1)(dst.data_ptr())
        bpe = (ctypes.c_size_t * 1)(1 << 46)             # 2^32 tiles per expert: launch_pack refuses
        return L.uep_balance(ctx._h, ctypes.c_void_p(d_ids.data_ptr()), None, ctypes.c_void_p(count.data_ptr()),
                             ctypes.byref(plan.c), ctypes.c_void_p(rep.data_ptr()), ctypes.c_void_p(rnk.data_ptr()),
                             ctypes.c_void_p(off.data_ptr()), None, 1, srcs, bpe, dsts,
                             ctypes.c_void_p(ws.data_ptr()), ctypes.c_void_p(stream.cuda_stream))

    st = torch.cuda.Stream()
    st.wait_stream(torch.cuda.current_stream())
    assert bad_call(st) == -2                             # UEP_ERR_UNSUPPORTED, eager
    torch.cuda.synchronize()
    lam, _ = oracle.histogram(ids.numpy(), E)
    with torch.cuda.stream(st):
        ctx.uep_balance(d_ids, None, count, plan, rep, rnk, off, None, [], [], ws)
    torch.cuda.synchronize()
    assert np.array_equal(count.cpu().numpy(), lam)       # not doubled by the aborted call
    g = torch.cuda.CUDAGraph()                            # the same inside a capture
    with torch.cuda.stream(st):
        with torch.cuda.graph(g, stream=st):
            assert bad_call(st) == -2
            ctx.uep_balance(d_ids, None, count, plan, rep, rnk, off, None, [], [], ws)
    count.fill_(-1)
    for _ in range(2):
        g.replay()
    torch.cuda.synchronize()
    assert np.array_equal(count.cpu().numpy(), lam)
    o = oracle_chain(ids, None, E, R, ns, um)
    assert np.array_equal(rep.cpu().numpy(), o[2]) and np.array_equal(off.cpu().numpy(), o[4])


def test_many_replays_with_changing_ids_on_one_workspace_full_size():
    """The lookup reads rank_kernel's outputs (packed ranks, chunk counts) in its prologue, before its
    griddepcontrol.wait: that rests on rank_kernel's grid being complete (prefix_kernel waits for it
    before it lets the lookup start) and on loads that bypass L1.  Stress it: ONE graph of three
    different calls (uep_balance, uep_remap, uep_balance) on ONE workspace at the DeepSeek-V3 shape,
    replayed six times with the ids and gates rewritten before every replay, each result checked
    against the oracle — a stale read of the previous replay's ranks or counts would show."""
    c = synth.CONFIGS["dsv3_prefill"]
    T, k, E, R, ns, um = c["T"], c["k"], c["E"], c["R"], c["n_slot"], c["u_min"]
    ctx = binding.Context(T, k, E, R, ns, um)
    ws = ctx.new_workspace()
    d_ids = [torch.zeros((T, k), dtype=torch.int32, device=DEV) for _ in range(3)]
    d_gate = [torch.zeros((T, k), dtype=torch.float32, device=DEV) for _ in range(3)]
    outs = []
    for b in range(3):
        rep, rnk, off, og = ctx.new_outputs(d_gate[b])
        outs.append(dict(count=torch.zeros(E, dtype=torch.int32, device=DEV), plan=ctx.new_plan(), rep=rep, rnk=rnk,
                         off=off, og=og))
    stream = torch.cuda.Stream()
    stream.wait_stream(torch.cuda.current_stream())

    def run_all():
        for b in (0, 1, 2):
            o = outs[b]
            if b == 1:                                   # remap alone, on the plan of its own ids
                ctx.uep_histogram(d_ids[b], o["count"], ws)
                ctx.uep_plan(o["count"], o["plan"], ws)
                ctx.uep_remap(d_ids[b], d_gate[b], o["plan"], o["rep"], o["rnk"], o["off"], o["og"], ws)
            else:
                ctx.uep_balance(d_ids[b], d_gate[b], o["count"], o["plan"], o["rep"], o["rnk"], o["off"], o["og"],
                                [], [], ws)

    with torch.cuda.stream(stream):
        run_all()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=stream):
            run_all()
    torch.cuda.synchronize()
    for it in range(6):
        host = []
        for b in range(3):
            ids = synth.zipf_topk_ids(T, k, E, 0.6 + 0.25 * ((it + b) % 5), 5000 + 10 * it + b, device=DEV)
            gate = synth.gates_uniform_renorm(T, k, 70 + 10 * it + b, device=DEV)
            d_ids[b].copy_(ids); d_gate[b].copy_(gate)
            host.append((ids.cpu(), gate.cpu()))
        torch.cuda.synchronize()
        graph.replay()
        torch.cuda.synchronize()
        for b in range(3):
            lam, p, rep, rnk, off, og = oracle_chain(host[b][0], host[b][1], E, R, ns, um)
            o = outs[b]
            assert np.array_equal(o["count"].cpu().numpy(), lam), (it, b)
            assert np.array_equal(o["rep"].cpu().numpy(), rep), (it, b)
            assert np.array_equal(o["rnk"].cpu().numpy(), rnk), (it, b)
            assert np.array_equal(o["off"].cpu().numpy(), off), (it, b)
            nv = int(p.rank_base[-1])
            assert np.array_equal(o["og"].cpu().view(torch.int32).numpy().view(np.uint32)[:nv], og[:nv]), (it, b)
