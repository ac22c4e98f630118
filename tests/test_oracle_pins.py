"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU, no CUDA path).

Every test here would fail on a plausible oracle mistake (dropped term, wrong tie-break,
wrong rounding, wrong floor predicate, transposed index):
  * hand-worked examples A/B (tests/golden, derived by hand from Alg. 1)
  * closed form for all-slots-to-one-expert
  * identity / degenerate cases, strict == tolerant at u_min = 1
  * the paper's constraints as invariants on Zipf workloads over a shape grid
  * numpy bincount (histogram), numpy STABLE argsort (remap), numpy fancy indexing (pack)
  * exhaustive optimum over all placements on the tiny config (Hall bound, cross-checked
    against scipy max-flow)
"""
import itertools
import os

import numpy as np
import pytest

import oracle
from paper_2606_04101_b200 import synth
import uep_checks as ck

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _read_golden(name):
    d = {}
    with open(os.path.join(GOLD, name)) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            k, v = line.split(":", 1)
            d[k.strip()] = v.strip()
    return d


@pytest.mark.parametrize("name", ["example_A.txt", "example_B_strict.txt",
                                  "example_B_tolerant.txt"])
def test_worked_examples(name):
    g = _read_golden(name)
    lam = np.array(g["lambda"].split(), dtype=np.int32)
    bn, bd = (int(x) for x in g["beta"].split("/"))
    probes = [(int(a), b == "F") for a, b in (x.split(":") for x in g["probes"].split())]
    transfers = []
    for x in g["transfers"].split():
        et, d = x.split(":")
        e, t = et.split(">")
        transfers.append((int(e), int(t), int(d)))
    for mode in g["modes"].split():
        fm = oracle.FLOOR_STRICT if mode == "strict" else oracle.FLOOR_TOLERANT
        p = oracle.plan(lam, int(g["R"]), int(g["n_slot"]), int(g["u_min"]), bn, bd, fm)
        assert p.trace == probes
        assert p.tau == int(g["tau"])
        assert p.rank_load.tolist() == [int(x) for x in g["rank_load"].split()]
        got = []
        for e in range(p.E):
            lo, hi = p.inst_off[e], p.inst_off[e + 1]
            q = np.diff(np.concatenate([[0], p.inst_cum[lo:hi]]))
            got += [(e, int(p.inst_rank[lo + i]), int(q[i])) for i in range(1, hi - lo)]
        assert got == transfers
        assert p.inst_cum[p.inst_off[0]:p.inst_off[1]].tolist() == \
            [int(x) for x in g["cum_e0"].split()]
        # S13: local physical slot of every instance (main: index among E_h(e); replica: M + slot)
        assert p.M == int(g["M"])
        assert p.inst_phys[:p.inst_off[-1]].tolist() == [int(x) for x in g["inst_phys"].split()]
        assert p.main_phys.tolist() == [p.inst_phys[p.inst_off[e]] for e in range(p.E)]
        ck.check_plan(lam, p, int(g["u_min"]), bn, bd, fm)


def test_all_to_one_closed_form():
    """All S slots on one expert: the other R-1 ranks have slack tau each, so the probe takes
    tau-sized bites, lowest rank id first.  S=2^21, R=64, beta=1.01, u_min=1024:
    tau = floor(1.01*32768) = 33095, 63 replicas: 62 of 33095 and one of 12167."""
    E, R, S = 256, 64, 2097152
    for hot in (0, 37, 255):
        lam = np.zeros(E, dtype=np.int32)
        lam[hot] = S
        p = oracle.plan(lam, R, 2, 1024)
        h = hot * R // E
        assert p.tau == 33095 and p.n_replicas == 63 and int(p.scalars[3]) == 64
        lo, hi = p.inst_off[hot], p.inst_off[hot + 1]
        q = np.diff(np.concatenate([[0], p.inst_cum[lo:hi]]))
        assert q[0] == 33095 and (q[1:63] == 33095).all() and q[63] == 12167
        assert 63 * 33095 + 12167 == S
        others = [t for t in range(R) if t != h]
        assert p.inst_rank[lo + 1:hi].tolist() == others          # lowest rank id first
        assert all(ok for _, ok in p.trace)                       # monotone: every mid feasible
        ck.check_plan(lam, p, 1024)
    # general closed form (tolerant): tau = tau_lo whenever tau_lo >= ceil(S/R)
    for S2, R2, um in [(100000, 8, 100), (999983, 16, 500), (4096, 4, 64)]:
        lam = np.zeros(32, dtype=np.int32)
        lam[5] = S2
        p = oracle.plan(lam, R2, 1, um)
        tau = (-(-S2 // R2)) * 101 // 100
        assert p.tau == tau
        bites = (S2 - tau) // tau
        rem = (S2 - tau) - bites * tau
        assert p.n_replicas == bites + (1 if rem >= um else 0)
        ck.check_plan(lam, p, um)


def test_identity_and_degenerate_cases():
    rng = np.random.default_rng(0)
    # balanced: max l <= tau_lo -> loop never runs (S4)
    lam = np.full(64, 1000, dtype=np.int32)
    p = oracle.plan(lam, 16, 2, 16)
    assert p.n_replicas == 0 and p.trace == [] and p.tau == 4000 and (p.slot_expert == -1).all()
    assert (p.rank_load == 4000).all()
    # n_slot = 0: probes run, none can move load -> identity, tau = max l
    lam = rng.integers(0, 5000, 64).astype(np.int32)
    p = oracle.plan(lam, 16, 0, 16, floor_mode=oracle.FLOOR_STRICT)
    ell = ck.initial_rank_load(lam, p.home, 16)
    assert p.n_replicas == 0 and p.tau == ell.max() and (p.rank_load == ell).all()
    ck.check_plan(lam, p, 16, floor_mode=ck.STRICT)
    # tolerant (S8): with no transfer possible a probe is feasible iff max l - tau < u_min,
    # which is monotone, so bisection must find exactly max l - u_min + 1
    p = oracle.plan(lam, 16, 0, 16)
    assert p.n_replicas == 0 and p.tau == ell.max() - 16 + 1 and (p.rank_load == ell).all()
    ck.check_plan(lam, p, 16)
    # R = 1
    p = oracle.plan(lam, 1, 2, 16)
    assert p.n_replicas == 0 and p.rank_load[0] == lam.sum()
    # empty load
    p = oracle.plan(np.zeros(16, np.int32), 4, 1, 8)
    assert p.n_replicas == 0 and p.tau == 0 and (p.rank_load == 0).all()
    # E < R (S2): ranks without a main expert are pure absorbers
    lam = rng.integers(1000, 90000, 64).astype(np.int32)
    p = oracle.plan(lam, 256, 1, 64)
    assert p.M == 1 and (np.bincount(p.home, minlength=256) <= 1).all()
    ck.check_plan(lam, p, 64)
    assert p.n_replicas > 0
    # explicit home map
    home = rng.integers(0, 8, 64).astype(np.int32)
    p = oracle.plan(lam, 8, 3, 256, home=home)
    assert (p.home == home).all()
    ck.check_plan(lam, p, 256)


def test_strict_equals_tolerant_at_u_min_1():
    for seed in range(6):
        ids = synth.zipf_topk_ids(2048, 4, 64, 0.6 + 0.3 * seed, seed).numpy()
        lam, _ = oracle.histogram(ids, 64)
        a = oracle.plan(lam, 16, 2, 1, floor_mode=oracle.FLOOR_STRICT)
        b = oracle.plan(lam, 16, 2, 1, floor_mode=oracle.FLOOR_TOLERANT)
        assert a.trace == b.trace and (a.U == b.U).all() and (a.slot_expert == b.slot_expert).all()
        ck.check_plan(lam, a, 1, floor_mode=ck.STRICT)
        # with u_min = 1 every overloaded rank that can be drained is: load <= tau exactly
        assert a.rank_load.max() <= a.tau


GRID = [  # (T, k, E, R, n_slot, s)
    (4096, 2, 16, 4, 1, 1.2), (8192, 8, 128, 32, 2, 0.6), (8192, 8, 128, 32, 2, 1.4),
    (16384, 8, 256, 64, 2, 1.0), (16384, 4, 512, 256, 4, 2.0), (4096, 1, 64, 8, 1, 0.0),
    (8192, 8, 160, 40, 4, 1.0), (2048, 4, 64, 256, 1, 1.0), (16384, 8, 512, 8, 3, 1.6),
]


@pytest.mark.parametrize("T,k,E,R,n_slot,s", GRID)
@pytest.mark.parametrize("mode", [oracle.FLOOR_STRICT, oracle.FLOOR_TOLERANT])
def test_plan_invariants_and_remap_on_zipf(T, k, E, R, n_slot, s, mode):
    ids = synth.zipf_topk_ids(T, k, E, s, seed=T + E + R).numpy()
    lam, bad = oracle.histogram(ids, E)
    assert bad == 0 and (lam == np.bincount(ids.ravel(), minlength=E)).all()   # library pin
    u_min = synth.stress_u_min(T * k, R)
    p = oracle.plan(lam, R, n_slot, u_min, floor_mode=mode)
    ck.check_plan(lam, p, u_min, floor_mode=mode)
    gate = synth.gates_uniform_renorm(T, k, 3).numpy()
    rep, rnk, off, og = oracle.remap(ids, gate, p)
    ck.check_remap(ids, p, rep, rnk, off, gate, og)


def test_histogram_invalid_ids_and_remap_skip():
    rng = np.random.default_rng(5)
    ids = rng.integers(-3, 20, size=(3000, 4)).astype(np.int32)       # ids in [-3, 19], E = 16
    lam, bad = oracle.histogram(ids, 16)
    valid = (ids >= 0) & (ids < 16)
    assert bad == (~valid).sum() and (lam == np.bincount(ids[valid], minlength=16)).all()
    p = oracle.plan(lam, 4, 1, 32, S_total=ids.size)
    assert int(p.scalars[5]) == bad
    gate = rng.standard_normal(ids.shape).astype(np.float32)
    rep, rnk, off, og = oracle.remap(ids, gate, p)
    ck.check_remap(ids, p, rep, rnk, off, gate, og)


def test_remap_duplicate_ids_in_token_and_gate_bits():
    """S15 duplicates inside a token; S17 gates are raw bit copies (NaN payloads, -0.0, denormals)."""
    ids = synth.one_expert_ids(2048, 4, 3).numpy()
    lam, _ = oracle.histogram(ids, 16)
    p = oracle.plan(lam, 4, 1, 64)
    bits = np.arange(ids.size, dtype=np.uint32) * np.uint32(2654435761)
    bits[:8] = [0x7FC00001, 0xFFC12345, 0x80000000, 0x00000001, 0x807FFFFF, 0x7F800000,
                0xFF800000, 0x7FA00000]
    gate = bits.view(np.float32).reshape(ids.shape)
    rep, rnk, off, og = oracle.remap(ids, gate, p)
    pos = ck.check_remap(ids, p, rep, rnk, off, gate, og)
    assert sorted(og.view(np.uint32).tolist()) == sorted(bits.tolist())
    # contiguous ranges in global stable order: slot j of expert 3 -> instance by cum
    cum = p.inst_cum[p.inst_off[3]:p.inst_off[4]]
    j = np.arange(ids.size)
    assert (rep.ravel() == np.searchsorted(cum, j, side="right")).all()
    # bf16-sized gates
    g16 = (np.arange(ids.size) % 65536).astype(np.uint16)
    _, _, _, og16 = oracle.remap(ids, g16, p)
    assert (og16[pos] == g16).all()


def test_pack_matches_numpy_indexing():
    rng = np.random.default_rng(1)
    ids = synth.zipf_topk_ids(4096, 2, 16, 1.2, 9).numpy()
    lam, _ = oracle.histogram(ids, 16)
    p = oracle.plan(lam, 4, 2, 64)
    assert p.n_replicas > 0
    src = rng.integers(0, 65536, size=(16, 1000)).astype(np.uint16)
    sent = rng.integers(0, 65536, size=(4, 2, 1000)).astype(np.uint16)
    dst = sent.copy()
    oracle.pack(p.slot_expert, src, dst)
    X = p.slot_expert
    ref = np.where((X >= 0)[..., None], src[np.maximum(X, 0)], sent)
    assert np.array_equal(dst, ref)
    ck.check_pack(X, src, dst, sent)


def _hall_min_max(lam, home, placements, R):
    """Exact optimum of min-max rank load with splittable expert load for each placement:
    max over non-empty rank subsets B of ceil(load confined to B / |B|) (max-flow/min-cut)."""
    lam = np.asarray(lam, dtype=np.int64)
    E = lam.size
    N = placements.shape[0]
    best = np.zeros(N, dtype=np.int64)
    e_idx = np.arange(E)
    for mask in range(1, 1 << R):
        inB = np.array([(mask >> t) & 1 for t in range(R)], dtype=bool)
        conf = np.broadcast_to(inB[home][None, :], (N, E)).copy()      # home in B
        for t in range(R):
            if not inB[t]:                                             # replica outside B
                conf &= placements[:, t][:, None] != e_idx[None, :]
        load = (conf * lam[None, :]).sum(axis=1)
        nb = int(inB.sum())
        best = np.maximum(best, -(-load // nb))
    return best


def test_tiny_config_bruteforce_optimum_bound():
    """tiny config: enumerate all 13^4 placements (each rank's slot: empty or one of the 12
    non-home experts); OPT (ignoring u_min, hence a lower bound) <= oracle's max load."""
    from scipy.sparse import csr_matrix
    from scipy.sparse.csgraph import maximum_flow
    c = synth.CONFIGS["tiny"]
    E, R = c["E"], c["R"]
    ids = synth.zipf_topk_ids(c["T"], c["k"], E, c["zipf_s"], 2024).numpy()
    lam, _ = oracle.histogram(ids, E)
    home, _, _ = oracle.layout(E, R)
    opts = []
    for t in range(R):
        opts.append([-1] + [e for e in range(E) if home[e] != t])
    placements = np.array(list(itertools.product(*opts)), dtype=np.int64)
    assert placements.shape == (13 ** 4, 4)
    best = _hall_min_max(lam, home, placements, R)
    # cross-check the Hall formula against scipy max-flow on a few placements
    rng = np.random.default_rng(0)
    for i in rng.integers(0, placements.shape[0], 12):
        tau = int(best[i])
        for cap, want in ((tau, True), (tau - 1, False)):
            n = E + R + 2
            g = np.zeros((n, n), dtype=np.int32)
            for e in range(E):
                g[0, 1 + e] = lam[e]
                g[1 + e, 1 + E + home[e]] = lam[e]
                for t in range(R):
                    if placements[i, t] == e:
                        g[1 + e, 1 + E + t] = lam[e]
            for t in range(R):
                g[1 + E + t, n - 1] = cap
            flow = maximum_flow(csr_matrix(g), 0, n - 1).flow_value
            assert (flow == lam.sum()) == want
    opt = int(best.min())
    mean_ceil = -(-int(lam.sum()) // R)
    assert opt >= mean_ceil
    for mode in (oracle.FLOOR_STRICT, oracle.FLOOR_TOLERANT):
        p = oracle.plan(lam, R, c["n_slot"], c["u_min"], floor_mode=mode)
        ck.check_plan(lam, p, c["u_min"], floor_mode=mode)
        assert opt <= int(p.rank_load.max())
        # the heuristic should land close to the optimum on this instance (plausibility)
        assert int(p.rank_load.max()) <= opt + c["u_min"] + mean_ceil // 50


def test_dsv3_shape_plausibility_against_table3():
    """Table 3 aggregates are plausibility only: post-balance imbalance
    within [1.00, beta + u_min/mean], a few dozen replicas, single-digit-ish fan-out."""
    c = synth.CONFIGS["dsv3_prefill"]
    for seed in (1, 2):
        ids = synth.zipf_topk_ids(c["T"], c["k"], c["E"], 1.0, seed).numpy()
        lam, _ = oracle.histogram(ids, c["E"])
        p = oracle.plan(lam, c["R"], c["n_slot"], c["u_min"])
        ck.check_plan(lam, p, c["u_min"])
        mean = lam.sum() / c["R"]
        imb = p.rank_load.max() / mean
        assert 1.0 <= imb <= 1.01 + 1024 / mean + 1e-9
        assert 20 <= p.n_replicas <= 128 and int(p.scalars[3]) <= 16
        assert 12 <= int(p.scalars[4]) <= 24


def test_grad_reduce_and_inverse_remap_pins():
    """O-5 / O-6 against what the paper fixes: on worked example A (expert 0 replicated on ranks
    1, 2, 3) with integer-valued gradients the reduction is a closed form; the total over all
    buffers is conserved ("preserves equivalence with the no-replica formulation");
    empty slots are untouched; the inverse remap composed with the forward map is the identity
    and equals a library stable argsort of the destination index."""
    lam = np.array([400, 100, 50, 50, 120, 80, 60, 140], np.int32)
    p = oracle.plan(lam, 4, 1, 10)
    assert p.slot_expert.reshape(-1).tolist() == [-1, 0, 0, 0]
    B = 6
    main = np.arange(8 * B, dtype=np.float32).reshape(8, B)
    slot = np.stack([np.full((1, B), 1000.0 * (t + 1), np.float32) for t in range(4)])
    m2, s2 = oracle.grad_reduce(p, main, slot)
    assert np.array_equal(m2[0], main[0] + 2000.0 + 3000.0 + 4000.0)       # closed form
    assert np.array_equal(m2[1:], main[1:].astype(np.float64))             # no replica: unchanged
    assert np.array_equal(s2[0], slot[0]) and not s2[1:].any()             # empty untouched, used cleared
    assert m2.sum() + s2.sum() == main.astype(np.float64).sum() + slot.astype(np.float64).sum() - 0.0
    # inverse remap on a random routing of that plan
    rng = np.random.default_rng(3)
    ids = np.repeat(np.arange(8, dtype=np.int32), lam)
    rng.shuffle(ids)
    rep, rnk, off, _ = oracle.remap(ids.reshape(-1, 1), None, p)
    src = oracle.inverse_remap(p, rnk, off)
    dest = p.rank_base[rnk.reshape(-1)] + off.reshape(-1)
    assert np.array_equal(dest[src], np.arange(ids.size))                  # forward o inverse = id
    assert np.array_equal(src, np.argsort(dest, kind="stable").astype(np.int32))
    ids2 = ids.copy(); ids2[::7] = -1                                      # invalid slots drop out
    rep, rnk, off, _ = oracle.remap(ids2.reshape(-1, 1), None, oracle.plan(
        np.bincount(ids2[ids2 >= 0], minlength=8).astype(np.int32), 4, 1, 10, S_total=ids2.size))
    pl2 = oracle.plan(np.bincount(ids2[ids2 >= 0], minlength=8).astype(np.int32), 4, 1, 10, S_total=ids2.size)
    src2 = oracle.inverse_remap(pl2, rnk, off)
    nv = int((ids2 >= 0).sum())
    assert (src2[nv:] == -1).all() and sorted(src2[:nv].tolist()) == np.flatnonzero(ids2 >= 0).tolist()


def test_relay_plan_pins():
    """O-7 against what §6.2 fixes: frontier = sqrt(f) to nearest; only experts with more than 4
    replicas get a tree; every replica has one parent in {home} U relays(e), relays hang off the
    home rank, leaves off relays; a rank's final send volume = the number of children it has;
    the all-to-one-expert closed form (f = 63: 8 relays, source fan-out 8 instead of 63, leaves
    7,7,7,7,7,7,7,6 because all relay volumes tie and ties go to the lower rank id)."""
    assert [oracle.relay_frontier(f) for f in (5, 6, 7, 8, 9, 12, 13, 16, 20, 21, 63, 255)] == \
        [2, 2, 3, 3, 3, 3, 4, 4, 4, 5, 8, 16]
    E, R, S = 256, 64, 2097152
    lam = np.zeros(E, np.int32); lam[0] = S
    p = oracle.plan(lam, R, 2, 1024)
    assert p.n_replicas == 63
    parent, vol = oracle.relay_plan(p)
    lo, hi = p.inst_off[0], p.inst_off[1]
    kids = np.bincount(parent[lo + 1:hi], minlength=R)
    assert kids[0] == 8 and vol[0] == 8                        # the source pushes 8 copies, not 63
    relays = [r for r in range(1, R) if kids[r] > 0]
    assert relays == list(range(1, 9)) and kids[1:9].tolist() == [7, 7, 7, 7, 7, 7, 7, 6]
    assert vol.sum() == 63 and np.array_equal(vol, kids)
    # general invariants on skewed routing
    for s, seed in ((1.4, 1), (2.0, 2)):
        ids = synth.zipf_topk_ids(32768, 8, 128, s, seed).numpy()
        lam, _ = oracle.histogram(ids, 128)
        p = oracle.plan(lam, 32, 2, 64)
        parent, vol = oracle.relay_plan(p)
        kids = np.zeros(32, np.int64)
        for e in range(128):
            lo, hi = p.inst_off[e], p.inst_off[e + 1]
            f = hi - lo - 1
            assert parent[lo] == -1
            reps = list(range(lo + 1, hi))
            par = parent[lo + 1:hi]
            np.add.at(kids, par, 1)
            if f <= oracle.RELAY_THRESHOLD:
                assert (par == p.home[e]).all()
                continue
            relay_ranks = {int(p.inst_rank[q]) for q in reps if parent[q] == p.home[e]}
            assert len(relay_ranks) == oracle.relay_frontier(f)
            assert all(int(x) == p.home[e] or int(x) in relay_ranks for x in par)
            assert all(parent[q] != p.inst_rank[q] for q in reps)          # nobody relays to itself
        assert np.array_equal(kids, vol) and vol.sum() == p.n_replicas
        assert (parent[p.inst_off[-1]:] == -1).all()


@pytest.mark.parametrize("name", ["example_local_A.txt", "example_local_B.txt"])
def test_local_remap_worked_examples_per_token(name):
    """O-8a + O-8b against hand-worked per-token literals (tests/golden/README.md): the split Q,
    and (replica, rank, offset) of EVERY slot, including a source that spills to a remote replica
    and two sources landing in one instance (reading S25 fixes their order), invalid ids, the gate
    placement and the in-flight counts."""
    import types
    g = _read_golden(name)
    ints = lambda key: [int(x) for x in g[key].split()]
    E, R, T, k = int(g["E"]), int(g["R"]), int(g["T"]), int(g["k"])
    P = len(ints("phys_base")) // R
    pl = types.SimpleNamespace(
        E=E, R=R, n_slot=int(g["n_slot"]), inst_off=np.array(ints("inst_off"), np.int32),
        inst_rank=np.array(ints("inst_rank"), np.int32), inst_phys=np.array(ints("inst_phys"), np.int32),
        inst_cum=np.array(ints("inst_cum"), np.int32),
        phys_base=np.array(ints("phys_base"), np.int32).reshape(R, P),
        rank_base=np.array(ints("rank_base"), np.int32))
    ids = np.array(ints("ids"), np.int32).reshape(T, k)
    Lam = np.array(ints("Lambda")).reshape(R, E)
    qs = oracle.reroute_split(Lam, pl)
    for e in range(E):
        assert qs[e].reshape(-1).tolist() == ints(f"q_e{e}"), e
    gate = (np.arange(T * k, dtype=np.uint32) * np.uint32(2654435761) + np.uint32(7)).reshape(T, k)
    rep, rnk, off, og, qs2, infl = oracle.remap_local(ids, gate, pl)
    assert rep.reshape(-1).tolist() == ints("replica")
    assert rnk.reshape(-1).tolist() == ints("rank")
    assert off.reshape(-1).tolist() == ints("offset")
    assert infl.tolist() == ints("n_inflight")
    assert all(np.array_equal(a, b) for a, b in zip(qs, qs2))       # Lambda counted from the ids
    want = np.zeros(T * k, np.uint32)                                # gates land at rank_base + offset
    for s, (t, o) in enumerate(zip(ints("rank"), ints("offset"))):
        if t >= 0:
            want[ints("rank_base")[t] + o] = gate.reshape(-1)[s]
    assert np.array_equal(og, want)
    v = ck.remap_local_vectorised(ids, pl, qs)                       # the sort-based cross-check agrees
    assert all(np.array_equal(a, b) for a, b in zip(v, (rep, rnk, off)))


def test_reroute_split_and_local_remap_pins():
    """O-8 against what the paper fixes: the hand-worked split below; both marginals of Q (Table 1,
    PAPER.md:133-135: sum_t q = lambda_{r,e}, sum_r q = u_{e,t}); local quota consumed first
    (Alg. 1 line 29); (rank, offset) a bijection onto the receive buffers with every instance
    receiving exactly its quota; no replicas => identical to the global remap; and locality can only
    lower the in-flight token count on the skewed example."""
    # hand example: E=2 experts on R=2 ranks, expert 0 (home rank 0) split main 3 + replica@rank1 3
    import types
    pl = types.SimpleNamespace(E=2, R=2, inst_off=np.array([0, 2, 3]), inst_rank=np.array([0, 1, 1, -1]),
                               inst_cum=np.array([3, 6, 2, 0]))
    Lam = np.array([[4, 1], [2, 1]])
    q0, q1 = oracle.reroute_split(Lam, pl)
    assert q0.tolist() == [[3, 1], [0, 2]]      # r0: 3 local + 1 spills to the replica; r1: 2 local
    assert q1.tolist() == [[1], [1]]
    for s, seed in ((1.0, 5), (2.0, 6)):
        T, k, E, R, ns = 8192, 4, 64, 16, 2
        ids = synth.zipf_topk_ids(T, k, E, s, seed).numpy()
        lam, _ = oracle.histogram(ids, E)
        p = oracle.plan(lam, R, ns, 64)
        assert p.n_replicas > 0
        rep, rnk, off, _, qs, infl = oracle.remap_local(ids, None, p)
        src = np.repeat(oracle.source_rank(T, R), k)
        for e in range(E):
            lo, hi = p.inst_off[e], p.inst_off[e + 1]
            u = np.diff(np.concatenate([[0], p.inst_cum[lo:hi]]))
            lam_re = np.bincount(src[ids.reshape(-1) == e], minlength=R)
            assert np.array_equal(qs[e].sum(axis=1), lam_re) and np.array_equal(qs[e].sum(axis=0), u)
            for i in range(hi - lo):
                t = p.inst_rank[lo + i]
                assert qs[e][t, i] >= min(lam_re[t], u[i])
        dest = p.rank_base[rnk.reshape(-1)] + off.reshape(-1)      # bijection onto the receive buffers
        assert np.array_equal(np.sort(dest), np.arange(ids.size))
        for e in range(E):                                          # every instance receives its quota,
            lo, hi = p.inst_off[e], p.inst_off[e + 1]               # in its own segment of its rank
            sel = ids.reshape(-1) == e
            u = np.diff(np.concatenate([[0], p.inst_cum[lo:hi]]))
            assert np.array_equal(np.bincount(rep.reshape(-1)[sel], minlength=hi - lo), u)
            for i in range(hi - lo):
                m = sel & (rep.reshape(-1) == i)
                t = p.inst_rank[lo + i]
                b0 = p.phys_base[t, p.inst_phys[lo + i]]
                assert (rnk.reshape(-1)[m] == t).all()
                assert np.array_equal(np.sort(off.reshape(-1)[m]), b0 + np.arange(u[i]))
        v = ck.remap_local_vectorised(ids, p, qs)                  # sort-based cross-check of the loop
        assert all(np.array_equal(a, b) for a, b in zip(v, (rep, rnk, off)))
        g_rep, g_rnk, g_off, _ = oracle.remap(ids, None, p)
        assert infl.sum() == (rnk.reshape(-1) != src).sum()
        assert infl.sum() <= (g_rnk.reshape(-1) != src).sum()
    ids = synth.zipf_topk_ids(4096, 2, 16, 0.0, 9).numpy()            # balanced: no replicas
    lam, _ = oracle.histogram(ids, 16)
    p = oracle.plan(lam, 4, 1, 4096)
    assert p.n_replicas == 0
    a = oracle.remap_local(ids, None, p)
    b = oracle.remap(ids, None, p)
    assert all(np.array_equal(x, y) for x, y in zip(a[:3], b[:3]))
