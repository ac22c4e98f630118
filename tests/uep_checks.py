"""Size-independent property checkers (numpy only) for plans and remaps.

They encode what the PAPER fixes, independently of any implementation:
constraints §4.3, Table 1 identities, threshold
semantics §5.1 and the token-assignment rule §5.2.
Used on oracle output (pins) and on CUDA output at full benchmark sizes.
`p` is any object with the plan arrays as numpy attributes (oracle.Plan or a host copy of
the device plan).
"""
import numpy as np

STRICT, TOLERANT = 0, 1


def initial_rank_load(lam, home, R):
    ell = np.zeros(R, dtype=np.int64)
    np.add.at(ell, np.asarray(home), np.asarray(lam, dtype=np.int64))
    return ell


def check_plan(lam, p, u_min, beta_num=101, beta_den=100, floor_mode=TOLERANT):
    lam = np.asarray(lam, dtype=np.int64)
    E, R, n_slot, M, P = p.E, p.R, p.n_slot, p.M, p.P
    home = np.asarray(p.home)
    ell = initial_rank_load(lam, home, R)
    S = int(lam.sum())
    tau = int(p.scalars[0])
    tau_lo0 = (-(-S // R)) * beta_num // beta_den
    tau_hi0 = int(ell.max()) if R else 0
    assert int(p.scalars[6]) == tau_lo0 and int(p.scalars[7]) == tau_hi0
    # (v) tau range
    assert min(tau_lo0, tau_hi0) <= tau <= tau_hi0, (tau_lo0, tau, tau_hi0)

    inst_off = np.asarray(p.inst_off)
    assert inst_off[0] == 0 and inst_off.shape == (E + 1,)
    n_inst = np.diff(inst_off)
    assert (n_inst >= 1).all()
    n_rep_total = int(n_inst.sum()) - E
    assert n_rep_total == int(p.scalars[1])
    assert int(p.scalars[3]) == int(n_inst.max())
    assert int(p.scalars[8]) == int((n_inst > 1).sum())

    U = np.zeros((E, R), dtype=np.int64)
    used = np.zeros(R, dtype=np.int64)
    X = np.asarray(p.slot_expert).reshape(R, n_slot) if n_slot else np.zeros((R, 0), int)
    seen_slot = np.zeros((R, max(n_slot, 1)), dtype=bool)
    for e in range(E):
        lo, hi = inst_off[e], inst_off[e + 1]
        ranks = p.inst_rank[lo:hi]
        phys = p.inst_phys[lo:hi]
        cum = np.asarray(p.inst_cum[lo:hi], dtype=np.int64)
        q = np.diff(np.concatenate([[0], cum]))
        # (iv) main placement immutable: entry 0 is the home instance in its main slot
        assert ranks[0] == home[e] and phys[0] == p.main_phys[e]
        # (i) sum_t u_{e,t} = lambda_e
        assert cum[-1] == lam[e], (e, cum, lam[e])
        assert (q >= 0).all()
        # (iii) no expert twice on a rank, never a replica on its own home
        assert len(set(ranks.tolist())) == len(ranks)
        # (ii) every replica carries at least u_min
        assert (q[1:] >= u_min).all(), (e, q)
        for i in range(1, hi - lo):
            t, s = int(ranks[i]), int(phys[i]) - M
            assert 0 <= s < n_slot
            assert X[t, s] == e and not seen_slot[t, s]
            seen_slot[t, s] = True
            used[t] += 1
        U[e, ranks] = q
        assert p.phys_count[home[e], p.main_phys[e]] == q[0]
        for i in range(1, hi - lo):
            assert p.phys_count[ranks[i], phys[i]] == q[i]
    # X holds exactly the replicas, used slots are a prefix (S10), budget respected
    assert ((X >= 0) == seen_slot[:, :n_slot]).all()
    for t in range(R):
        assert used[t] <= n_slot
        assert (X[t, :used[t]] >= 0).all() and (X[t, used[t]:] == -1).all()
    if getattr(p, "U", None) is not None:
        assert (np.asarray(p.U, dtype=np.int64) == U).all()
    load = U.sum(axis=0)
    assert (np.asarray(p.rank_load, dtype=np.int64) == load).all()
    assert (np.asarray(p.phys_count, dtype=np.int64).sum(axis=1) == load).all()
    pb = np.asarray(p.phys_base, dtype=np.int64)
    pc = np.asarray(p.phys_count, dtype=np.int64)
    assert (pb == np.cumsum(pc, axis=1) - pc).all()
    rb = np.asarray(p.rank_base, dtype=np.int64)
    assert rb[0] == 0 and (np.diff(rb) == load).all() and rb[-1] == S
    assert int(p.scalars[2]) == int(load.max())
    # (v) load bound, (vi) absorbers never exceed tau, (vii) never worse than doing nothing
    bound = tau if floor_mode == STRICT else tau + u_min - 1
    assert load.max() <= bound, (load.max(), bound)
    under = ell <= tau
    assert (load[under] <= tau).all()
    assert (load[~under] <= ell[~under]).all()
    assert load.max() <= ell.max()
    return U, load


def check_remap(ids, p, replica, rank, offset, gate=None, out_gate=None):
    """(rank, offset) is a bijection onto U_t {t} x [0, rank_load[t]); per instance the
    received count is its quota; inside an expert the instance index is non-decreasing in
    stable order; the dispatch order equals numpy's STABLE argsort by (rank, phys)."""
    ids = np.asarray(ids).reshape(-1).astype(np.int64)
    replica, rank, offset = (np.asarray(a).reshape(-1).astype(np.int64)
                             for a in (replica, rank, offset))
    E, P = p.E, p.P
    valid = (ids >= 0) & (ids < E)
    assert (replica[~valid] == -1).all() and (rank[~valid] == -1).all() \
        and (offset[~valid] == -1).all()
    v_ids, v_rep, v_rank, v_off = ids[valid], replica[valid], rank[valid], offset[valid]
    inst = np.asarray(p.inst_off, dtype=np.int64)[v_ids] + v_rep
    assert (v_rep >= 0).all() and (inst < np.asarray(p.inst_off)[v_ids + 1]).all()
    assert (np.asarray(p.inst_rank)[inst] == v_rank).all()
    phys = np.asarray(p.inst_phys, dtype=np.int64)[inst]
    # per-instance received count == quota
    cum = np.asarray(p.inst_cum, dtype=np.int64)
    n_tot = int(p.inst_off[-1])
    got = np.bincount(inst, minlength=n_tot)
    quota = cum[:n_tot].copy()
    first = np.zeros(n_tot, dtype=bool)
    first[np.asarray(p.inst_off[:-1])] = True
    quota[~first] -= cum[:n_tot][np.flatnonzero(~first) - 1]
    assert (got == quota).all()
    # bijection onto the receive buffers
    rb = np.asarray(p.rank_base, dtype=np.int64)
    pos = rb[v_rank] + v_off
    assert (v_off >= 0).all() and (v_off < np.asarray(p.rank_load, dtype=np.int64)[v_rank]).all()
    assert np.unique(pos).size == pos.size == int(rb[-1])
    # stable: sorting slots by dispatch position == stable sort by (rank, phys)
    key = v_rank * P + phys
    assert (np.argsort(pos, kind="stable") == np.argsort(key, kind="stable")).all()
    # contiguous ranges per expert: instance index non-decreasing in slot order
    order = np.argsort(v_ids, kind="stable")
    same = v_ids[order][1:] == v_ids[order][:-1]
    assert (np.diff(v_rep[order])[same] >= 0).all()
    if gate is not None:
        g = np.asarray(gate).reshape(-1)
        og = np.asarray(out_gate).reshape(-1)
        bits = {2: np.uint16, 4: np.uint32}[g.itemsize]
        assert (og.view(bits)[pos] == g.view(bits)[valid]).all()
    return pos


def check_pack(slot_expert, src, dst, sentinel_dst):
    """dst slot == src expert for filled slots; untouched sentinel for empty ones."""
    X = np.asarray(slot_expert)
    R, n_slot = X.shape
    d = dst.reshape(R, n_slot, -1)
    s0 = sentinel_dst.reshape(R, n_slot, -1)
    s = src.reshape(src.shape[0], -1)
    for t in range(R):
        for k in range(n_slot):
            e = X[t, k]
            ref = s[e] if e >= 0 else s0[t, k]
            assert np.array_equal(d[t, k].view(np.uint8), ref.view(np.uint8)), (t, k, e)


def remap_local_vectorised(ids, pl, qs):
    """Cross-check of the oracle's per-slot loop O-8b (oracle.remap_local): the same assignment
    computed the way a fast implementation would (stable argsort over (source rank, expert),
    searchsorted per group).  qs = oracle.reroute_split's list.  Returns (replica, rank, offset)."""
    ids32 = np.ascontiguousarray(ids, dtype=np.int32)
    T, k = ids32.shape
    E, R = pl.E, pl.R
    flat = ids32.reshape(-1)
    S = flat.size
    src = np.repeat((np.arange(T, dtype=np.int64) * R // max(T, 1)), k)
    valid = (flat >= 0) & (flat < E)
    rep = np.full(S, -1, np.int32); rnk = np.full(S, -1, np.int32); off = np.full(S, -1, np.int32)
    inst_base = np.asarray(pl.phys_base).reshape(R, -1)
    order = np.argsort(np.where(valid, src * E + flat, np.int64(R) * E), kind="stable")
    keys = (src * E + flat)[order]
    nv = int(valid.sum())
    bounds = np.flatnonzero(np.diff(np.concatenate([[-1], keys[:nv]]))).tolist() + [nv]
    for a, b in zip(bounds[:-1], bounds[1:]):
        r, e = divmod(int(keys[a]), E)
        lo = int(pl.inst_off[e])
        q = qs[e]
        cum = np.cumsum(q[r])
        j = np.arange(b - a)
        i = np.searchsorted(cum, j, side="right")
        before = np.concatenate([[0], cum])[i]
        srcpre = q[:r].sum(axis=0)
        sl = order[a:b]
        rep[sl] = i
        rnk[sl] = pl.inst_rank[lo + i]
        off[sl] = inst_base[pl.inst_rank[lo + i], pl.inst_phys[lo + i]] + srcpre[i] + (j - before)
    return rep.reshape(ids32.shape), rnk.reshape(ids32.shape), off.reshape(ids32.shape)
