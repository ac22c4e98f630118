"""CPU oracle for the UltraEP balance-planning path — TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares no code with the CUDA
path (``paper_2606_04101_b200``) and never imports it.

The arithmetic of O-1..O-4 lives in ``uep_oracle.cpp`` (plain single-threaded C++, written
from reference/PAPER.md Algorithm 1 and §5.2); this module compiles it with g++ and marshals
numpy arrays through ctypes.  The backward-path definitions O-5 (gradient reduction, fp64) and
O-6 (inverse remap) are a few lines of numpy each, below; their pins are in
tests/test_oracle_pins.py::test_grad_reduce_and_inverse_remap_pins.  O-7 (relay trees) and O-8a
(the source-wise split Q of SolveReroute) are plain Python loops below; O-8b (the per-token
source-aware assignment) is the per-slot loop uep_oracle_remap_local in uep_oracle.cpp.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "uep_oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle.so")

FLOOR_STRICT = 0
FLOOR_TOLERANT = 1
N_SCALARS = 16
SC_TAU, SC_N_REPLICAS, SC_MAX_LOAD, SC_MAX_FANOUT, SC_N_PROBES, SC_N_INVALID, SC_TAU_LO0, \
    SC_TAU_HI0, SC_N_GROUPS = range(9)


def build(force: bool = False) -> str:
    """Compile the oracle (g++ -O2, single translation unit). Returns the .so path."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    tmp = _LIB + f".tmp{os.getpid()}"
    subprocess.check_call(["g++", "-O2", "-std=c++17", "-shared", "-fPIC", "-o", tmp, _SRC])
    os.replace(tmp, _LIB)
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        for name in ("uep_oracle_histogram", "uep_oracle_layout", "uep_oracle_plan",
                     "uep_oracle_remap", "uep_oracle_remap_local", "uep_oracle_pack"):
            getattr(_lib, name).restype = ctypes.c_int
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


@dataclass
class Plan:
    """Host copy of every plan array (names as in include/uep.h / DESIGN.md)."""
    E: int
    R: int
    n_slot: int
    M: int
    P: int
    home: np.ndarray
    main_phys: np.ndarray
    slot_expert: np.ndarray   # [R, n_slot]
    inst_off: np.ndarray      # [E+1]
    inst_rank: np.ndarray     # [E + R*n_slot]
    inst_phys: np.ndarray
    inst_cum: np.ndarray
    phys_count: np.ndarray    # [R, P]
    phys_base: np.ndarray     # [R, P]
    rank_load: np.ndarray     # [R]
    rank_base: np.ndarray     # [R+1]
    U: np.ndarray             # [E, R]
    scalars: np.ndarray       # [16]
    trace: list               # [(tau, feasible)] bisection sequence

    @property
    def tau(self):
        return int(self.scalars[SC_TAU])

    @property
    def n_replicas(self):
        return int(self.scalars[SC_N_REPLICAS])


def histogram(ids: np.ndarray, E: int):
    """O-1. Returns (count[E] int32, n_invalid)."""
    ids = _i32(ids).reshape(-1)
    count = np.zeros(E, dtype=np.int32)
    bad = ctypes.c_int64(0)
    rc = _load().uep_oracle_histogram(_p(ids), ctypes.c_int64(ids.size), ctypes.c_int32(E),
                                      _p(count), ctypes.byref(bad))
    assert rc == 0
    return count, int(bad.value)


def layout(E: int, R: int, home=None):
    """Static layout: (home[E], main_phys[E], M)."""
    home_in = None if home is None else _i32(home)
    home_out = np.zeros(E, dtype=np.int32)
    main_phys = np.zeros(E, dtype=np.int32)
    M = ctypes.c_int32(0)
    rc = _load().uep_oracle_layout(ctypes.c_int32(E), ctypes.c_int32(R), _p(home_in),
                                   _p(home_out), _p(main_phys), ctypes.byref(M))
    if rc != 0:
        raise ValueError("home rank outside [0, R)")
    return home_out, main_phys, int(M.value)


def plan(lam: np.ndarray, R: int, n_slot: int, u_min: int, beta_num: int = 101,
         beta_den: int = 100, floor_mode: int = FLOOR_TOLERANT, home=None,
         S_total: int | None = None) -> Plan:
    """O-2 SolveReplication (Alg. 1 lines 1-25)."""
    lam = _i32(lam).reshape(-1)
    E = lam.size
    home_arr, main_phys, M = layout(E, R, home)
    P = M + n_slot
    cap = E + R * n_slot
    z = lambda n: np.zeros(n, dtype=np.int32)
    slot_expert, inst_off = z(max(R * n_slot, 1)), z(E + 1)
    inst_rank, inst_phys, inst_cum = z(cap), z(cap), z(cap)
    phys_count, phys_base = z(R * P), z(R * P)
    rank_load, rank_base, U, scalars = z(R), z(R + 1), z(E * R), z(N_SCALARS)
    trace_tau = np.zeros(128, dtype=np.int64)
    trace_feas = z(128)
    home_in = None if home is None else _i32(home)
    if S_total is None:
        S_total = int(lam.astype(np.int64).sum())
    rc = _load().uep_oracle_plan(
        _p(lam), ctypes.c_int32(E), ctypes.c_int32(R), ctypes.c_int32(n_slot),
        ctypes.c_int32(u_min), ctypes.c_int32(beta_num), ctypes.c_int32(beta_den),
        ctypes.c_int32(floor_mode), _p(home_in), ctypes.c_int64(S_total),
        _p(slot_expert), _p(inst_off), _p(inst_rank), _p(inst_phys), _p(inst_cum),
        _p(phys_count), _p(phys_base), _p(rank_load), _p(rank_base), _p(U), _p(scalars),
        _p(trace_tau), _p(trace_feas), ctypes.c_int32(128))
    if rc != 0:
        raise ValueError(f"uep_oracle_plan rc={rc}")
    n = int(scalars[SC_N_PROBES])
    trace = [(int(trace_tau[i]), bool(trace_feas[i])) for i in range(min(n, 128))]
    return Plan(E, R, n_slot, M, P, home_arr, main_phys,
                slot_expert[:R * n_slot].reshape(R, n_slot), inst_off, inst_rank, inst_phys,
                inst_cum, phys_count.reshape(R, P), phys_base.reshape(R, P), rank_load,
                rank_base, U.reshape(E, R), scalars, trace)


def remap(ids: np.ndarray, gate: np.ndarray | None, pl: Plan):
    """O-3 token assignment. gate is any array with 2- or 4-byte items (raw byte copy).
    Returns (replica, rank, offset, out_gate) with the shapes of ids / a flat gate array."""
    ids32 = _i32(ids)
    flat = ids32.reshape(-1)
    S = flat.size
    rep, rnk, off = (np.empty(S, dtype=np.int32) for _ in range(3))
    if gate is not None:
        gate = np.ascontiguousarray(gate).reshape(-1)
        assert gate.size == S and gate.itemsize in (2, 4)
        out_gate = np.zeros(S, dtype=gate.dtype)
        gbytes = gate.itemsize
    else:
        out_gate, gbytes = None, 0
    rc = _load().uep_oracle_remap(
        _p(flat), _p(gate), ctypes.c_int32(gbytes), ctypes.c_int64(S), ctypes.c_int32(pl.E),
        ctypes.c_int32(pl.P), _p(pl.inst_off), _p(pl.inst_rank), _p(pl.inst_phys),
        _p(pl.inst_cum), _p(np.ascontiguousarray(pl.phys_base).reshape(-1)), _p(pl.rank_base),
        _p(rep), _p(rnk), _p(off), _p(out_gate))
    if rc != 0:
        raise ValueError(f"uep_oracle_remap rc={rc}")
    shp = ids32.shape
    return rep.reshape(shp), rnk.reshape(shp), off.reshape(shp), out_gate


def pack(slot_expert: np.ndarray, src: np.ndarray, dst: np.ndarray) -> None:
    """O-4. src: [E, ...] contiguous per expert; dst: [R, n_slot, ...] written in place."""
    se = _i32(slot_expert)
    R, n_slot = se.shape
    assert src.flags.c_contiguous and dst.flags.c_contiguous and dst.flags.writeable
    B = src.nbytes // src.shape[0]
    assert dst.nbytes == R * n_slot * B
    rc = _load().uep_oracle_pack(_p(se.reshape(-1)), ctypes.c_int32(R), ctypes.c_int32(n_slot),
                                 _p(src), ctypes.c_int64(B), _p(dst))
    assert rc == 0


def grad_reduce(pl: Plan, main_grad: np.ndarray, slot_grad: np.ndarray):
    """O-5 backward gradient reduction ("every main expert aggregates the gradients
    contributed by all of its remote replicas into the main gradient buffer"; PAPER.md:341
    "accumulated into the local gradient buffer of main experts, and then cleared in place").

    main_grad [E, B], slot_grad [R, n_slot, B] (any float dtype).  Returns (main_out float64 [E, B],
    slot_out like slot_grad): main_out[e] = main[e] + sum over the replicas of e of their slot
    buffer, accumulated in fp64 (the plain definition; a sum has no order in exact arithmetic);
    slot buffers of USED redundant slots are zero afterwards, empty slots are untouched."""
    main64 = np.asarray(main_grad, dtype=np.float64).copy()
    slot_out = np.array(slot_grad, copy=True)
    R, n_slot = pl.R, pl.n_slot
    for t in range(R):
        for s in range(n_slot):
            e = int(pl.slot_expert[t, s])
            if e < 0:
                continue
            main64[e] += np.asarray(slot_grad[t, s], dtype=np.float64)
            slot_out[t, s] = 0
    return main64, slot_out


def inverse_remap(pl: Plan, rank: np.ndarray, offset: np.ndarray) -> np.ndarray:
    """O-6 reverse reroute ("a scatter-to-gather inversion of the forward assignment",
    PAPER.md:164-166): src[rank_base[rank[s]] + offset[s]] = s for every valid slot s (flat slot
    index); positions past the number of valid slots are -1."""
    rank = np.asarray(rank).reshape(-1)
    offset = np.asarray(offset).reshape(-1)
    src = np.full(rank.size, -1, dtype=np.int32)
    for s in range(rank.size):
        if rank[s] >= 0:
            src[int(pl.rank_base[rank[s]]) + int(offset[s])] = s
    return src


RELAY_THRESHOLD = 4          # "experts whose replica count exceeds the relay threshold (set to 4)"


def relay_frontier(f: int) -> int:
    """Relay frontier "chosen near sqrt(|H(e)|-1)": sqrt(f) rounded to nearest,
    in integers: k = floor(sqrt(f)), +1 if f > k*k + k."""
    k = int(np.floor(np.sqrt(f)))
    while k * k > f:
        k -= 1
    while (k + 1) * (k + 1) <= f:
        k += 1
    return k + 1 if f > k * k + k else k


def relay_plan(pl: Plan):
    """O-7 load-aware relay scheduling, topology only (§6.2), step by step:
      1. send volume of every rank = number of replica copies its main experts must push;
      2. relay-eligible experts (replica count f > 4), one by one in ascending expert id
         (the paper gives no order; S24);
      3. first-stage relays = the k = relay_frontier(f) replica ranks of e with the smallest
         sending volume (ties -> lower rank id);
      4. every remaining replica, in instance order, is attached to the relay whose sending volume
         would remain smallest after taking it (ties -> lower rank id);
      5. volumes updated: the source now sends k copies instead of f, each relay its leaves.
    Returns (parent[E + R*n_slot] int32 aligned with the plan's CSR: -1 for main instances and
    unused entries, else the rank that sends this replica its copy; send_volume[R] int32)."""
    E, R = pl.E, pl.R
    parent = np.full(pl.inst_rank.size, -1, dtype=np.int32)
    vol = np.zeros(R, dtype=np.int64)
    for e in range(E):
        lo, hi = int(pl.inst_off[e]), int(pl.inst_off[e + 1])
        vol[pl.home[e]] += hi - lo - 1
        parent[lo + 1:hi] = pl.home[e]                      # direct sends unless a relay tree replaces them
    for e in range(E):
        lo, hi = int(pl.inst_off[e]), int(pl.inst_off[e + 1])
        f = hi - lo - 1
        if f <= RELAY_THRESHOLD:
            continue
        k = relay_frontier(f)
        reps = list(range(lo + 1, hi))                      # CSR indices of the replicas, instance order
        order = sorted(reps, key=lambda p: (vol[pl.inst_rank[p]], pl.inst_rank[p]))
        relays = order[:k]
        relay_set = set(relays)
        leaves_of = {p: 0 for p in relays}
        for p in reps:
            if p in relay_set:
                continue
            best = min(relays, key=lambda q: (vol[pl.inst_rank[q]] + leaves_of[q] + 1, pl.inst_rank[q]))
            parent[p] = pl.inst_rank[best]
            leaves_of[best] += 1
        vol[pl.home[e]] += k - f
        for q in relays:
            vol[pl.inst_rank[q]] += leaves_of[q]
    return parent, vol.astype(np.int32)


def source_rank(T: int, R: int) -> np.ndarray:
    """S1: token i is routed by source rank floor(i*R/T) ("each rank computes gating for its local
    tokens")."""
    return (np.arange(T, dtype=np.int64) * R // max(T, 1)).astype(np.int32)


def reroute_split(Lam: np.ndarray, pl: Plan):
    """O-8a SolveReroute (Alg. 1 lines 26-36; §5.2).  Lam[R,E] =
    lambda_{r,e}.  Returns a list over experts of q_e[R, n_e] (n_e instances in the plan's CSR
    order [main, replicas...]):
      line 29   q[t,e,t] = min(lambda[t,e], u[e,t]) for every host rank t of e  (consume local quota)
      lines 30-31   residual demand and residual quota
      lines 32-34   the residual demand of every source is split over the residual quotas.  The
                paper's round(lambda^ * u^/sum u^) cannot keep both marginals; reading S18: lay the
                residual demands (ascending source rank) and the residual quotas (instance order)
                on one number line and give q[r,e,t] the length of the overlap.  Both marginals
                hold exactly and the split is deterministic."""
    R, E = Lam.shape
    out = []
    for e in range(E):
        lo, hi = int(pl.inst_off[e]), int(pl.inst_off[e + 1])
        n = hi - lo
        host = pl.inst_rank[lo:hi].astype(np.int64)
        cum = pl.inst_cum[lo:hi].astype(np.int64)
        u = np.diff(np.concatenate([[0], cum]))
        lam = Lam[:, e].astype(np.int64)
        q = np.zeros((R, n), dtype=np.int64)
        lam_hat, u_hat = lam.copy(), u.copy()
        for i in range(n):                                  # line 29
            t = host[i]
            q[t, i] = min(lam[t], u[i])
            lam_hat[t] -= q[t, i]
            u_hat[i] -= q[t, i]
        d0 = np.concatenate([[0], np.cumsum(lam_hat)])      # number line of residual demands
        u0 = np.concatenate([[0], np.cumsum(u_hat)])        # ... and of residual quotas
        for r in range(R):
            for i in range(n):
                q[r, i] += max(0, min(d0[r + 1], u0[i + 1]) - max(d0[r], u0[i]))
        out.append(q)
    return out


def remap_local(ids: np.ndarray, gate: np.ndarray | None, pl: Plan):
    """O-8b source-aware token assignment (§5.2 "Token Assignment"): "the j-th local
    token of pair (r, e) is sent to the first physical instance whose cumulative quota covers j",
    cumulative over q[r,e,.] in instance order.  Receive order inside an instance (the paper leaves
    it to the dispatch library; reading S25): by source rank ascending, then local order, so
    offset = inst_base + sum_{r'<r} q[r',e,i] + (j - cumulative before i).

    The split Q is O-8a (reroute_split, above) on Lambda[r,e] counted here slot by slot; the
    assignment itself is the plain per-slot loop uep_oracle_remap_local in uep_oracle.cpp (next to
    O-3, same shape).  Returns (replica, rank, offset, out_gate, q_list, n_inflight[R])."""
    ids32 = _i32(ids)
    T, k = ids32.shape
    E, R = pl.E, pl.R
    flat = ids32.reshape(-1)
    S = flat.size
    src = np.repeat(source_rank(T, R), k)                    # S1: source rank of every slot
    valid = (flat >= 0) & (flat < E)
    Lam = np.zeros((R, E), dtype=np.int64)                   # lambda_{r,e}: a plain count
    np.add.at(Lam, (src[valid], flat[valid]), 1)
    qs = reroute_split(Lam, pl)
    cap = int(np.asarray(pl.inst_rank).size)
    q = np.zeros((R, cap), dtype=np.int64)                   # q[r][CSR entry]
    for e in range(E):
        lo, hi = int(pl.inst_off[e]), int(pl.inst_off[e + 1])
        q[:, lo:hi] = qs[e]
    rep, rnk, off = (np.empty(S, dtype=np.int32) for _ in range(3))
    infl = np.zeros(R, dtype=np.int32)
    if gate is not None:
        gate = np.ascontiguousarray(gate).reshape(-1)
        assert gate.size == S and gate.itemsize in (2, 4)
        out_gate = np.zeros(S, dtype=gate.dtype)
        gbytes = gate.itemsize
    else:
        out_gate, gbytes = None, 0
    P = int(np.asarray(pl.phys_base).reshape(R, -1).shape[1])
    rc = _load().uep_oracle_remap_local(
        _p(flat), _p(gate), ctypes.c_int32(gbytes), ctypes.c_int64(T), ctypes.c_int32(k),
        ctypes.c_int32(E), ctypes.c_int32(R), ctypes.c_int32(P), ctypes.c_int32(cap),
        _p(_i32(pl.inst_off)), _p(_i32(pl.inst_rank)), _p(_i32(pl.inst_phys)), _p(q),
        _p(np.ascontiguousarray(pl.phys_base, dtype=np.int32).reshape(-1)), _p(_i32(pl.rank_base)),
        _p(rep), _p(rnk), _p(off), _p(out_gate), _p(infl))
    if rc != 0:
        raise ValueError(f"uep_oracle_remap_local rc={rc}")
    shp = ids32.shape
    return rep.reshape(shp), rnk.reshape(shp), off.reshape(shp), out_gate, qs, infl
