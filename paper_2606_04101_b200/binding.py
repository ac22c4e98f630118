"""Thin ctypes binding of libuep.so — same names as include/uep.h, argument marshalling only.

PyTorch is used for device memory and streams; every step of the path runs in the CUDA
kernels behind the C ABI.  There is no CPU fallback: if the shared library is missing the
first call raises, and every non-zero return code raises ``UepError``.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass, field

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libuep.so")

FLOOR_STRICT, FLOOR_TOLERANT = 0, 1
GATE_F32, GATE_BF16, GATE_NONE = 0, 1, 2
N_SCALARS = 16
MAX_TENSORS = 8
SC_TAU, SC_N_REPLICAS, SC_MAX_LOAD, SC_MAX_FANOUT, SC_N_PROBES, SC_N_INVALID, SC_TAU_LO0, \
    SC_TAU_HI0, SC_N_GROUPS = range(9)

EXPORTS = ["uep_create", "uep_destroy", "uep_workspace_bytes", "uep_workspace_init",
           "uep_plan_bytes", "uep_histogram", "uep_plan", "uep_plan_batched", "uep_remap", "uep_remap_local",
           "uep_remap_rank", "uep_shard_count", "uep_shard_rows", "uep_shard_finish",
           "uep_remap_lookup", "uep_remap_inverse", "uep_relay_plan", "uep_pack", "uep_grad_reduce",
           "uep_balance",
           "uep_balance_host", "uep_strerror", "uep_last_cuda_error", "uep_get_launch_info",
           "uep_launch_count", "uep_histogram_static", "uep_histogram_static_setup",
           "uep_static_last_error"]
STATIC_MAX_SLOTS = 1 << 24


class UepError(RuntimeError):
    pass


class _Config(ctypes.Structure):
    _fields_ = [(n, ctypes.c_int32) for n in
                ("T", "k", "E", "R", "n_slot", "u_min", "beta_num", "beta_den", "floor_mode",
                 "gate_dtype")] + [("home_rank", ctypes.POINTER(ctypes.c_int32))]


class _PlanSizes(ctypes.Structure):
    _fields_ = [(n, ctypes.c_int32) for n in
                ("slot_expert", "inst_off", "inst_cap", "phys", "rank_load", "rank_base", "U",
                 "scalars", "M", "P")]


_PLAN_FIELDS = ("slot_expert", "inst_off", "inst_rank", "inst_phys", "inst_cum", "inst_base", "phys_count",
                "phys_base", "rank_load", "rank_base", "scalars", "U")


class _PlanOut(ctypes.Structure):
    _fields_ = [(n, ctypes.c_void_p) for n in _PLAN_FIELDS]


class _LaunchInfo(ctypes.Structure):
    _fields_ = [(n, ctypes.c_int32) for n in
                ("n_chunks", "chunk_len", "hist_threads", "remap_threads", "plan_threads",
                 "pack_ctas", "pack_tile_bytes", "sm_count", "r_chunks", "r_chunk_len",
                 "plan_cluster")]


_lib = None


def lib():
    """Load libuep.so (built in-tree by paper_2606_04101_b200.build). Raises if missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise UepError(f"{LIB_PATH} not built: run `python -m paper_2606_04101_b200.build` "
                           "(there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        for n in EXPORTS:
            getattr(L, n)                      # every declared symbol must be exported
        L.uep_workspace_bytes.restype = ctypes.c_size_t
        L.uep_strerror.restype = ctypes.c_char_p
        L.uep_last_cuda_error.restype = ctypes.c_char_p
        L.uep_destroy.restype = None
        L.uep_launch_count.restype = ctypes.c_ulonglong
        L.uep_static_last_error.restype = ctypes.c_char_p
        _lib = L
    return _lib


def _check(rc: int):
    if rc != 0:
        L = lib()
        msg = L.uep_strerror(rc).decode()
        if rc == -3:
            msg += " — " + L.uep_last_cuda_error().decode()
        raise UepError(f"libuep rc={rc}: {msg}")


def _check_static(rc: int):
    if rc != 0:
        L = lib()
        msg = L.uep_static_last_error().decode() or L.uep_strerror(rc).decode()
        if rc == -3:
            msg += " — " + L.uep_last_cuda_error().decode()
        raise UepError(f"libuep rc={rc}: {msg}")


def uep_histogram_static_setup():
    """Resolve the static scratch on the current device (once per device, outside capture)."""
    _check_static(lib().uep_histogram_static_setup())


def uep_histogram_static(topk_ids, E, expert_count, stream=None, n_slots=None):
    """lambda_e without context or workspace; the library allocates nothing (include/uep.h).
    topk_ids: int32 device tensor (or None with n_slots=0); expert_count: int32 [E] device tensor."""
    n = (0 if topk_ids is None else topk_ids.numel()) if n_slots is None else int(n_slots)
    _check_static(lib().uep_histogram_static(_ptr(topk_ids), ctypes.c_longlong(n), ctypes.c_int32(E),
                                             _ptr(expert_count), _stream(stream)))
    return expert_count


def _ptr(t):
    return ctypes.c_void_p(0 if t is None else t.data_ptr())


def _stream(stream):
    if stream is None:
        stream = torch.cuda.current_stream()
    return ctypes.c_void_p(stream.cuda_stream)


@dataclass
class Plan:
    """Device-resident plan arrays (torch int32 tensors) + the C struct that points at them."""
    E: int
    R: int
    n_slot: int
    M: int
    P: int
    slot_expert: torch.Tensor
    inst_off: torch.Tensor
    inst_rank: torch.Tensor
    inst_phys: torch.Tensor
    inst_cum: torch.Tensor
    inst_base: torch.Tensor
    phys_count: torch.Tensor
    phys_base: torch.Tensor
    rank_load: torch.Tensor
    rank_base: torch.Tensor
    scalars: torch.Tensor
    U: torch.Tensor | None
    c: _PlanOut = field(default=None, repr=False)
    batch: int = 1

    def host(self, b: int = 0):
        """Host (numpy) copy of instance b with the attribute names the checkers use."""
        import types
        h = types.SimpleNamespace(E=self.E, R=self.R, n_slot=self.n_slot, M=self.M, P=self.P)
        for n in _PLAN_FIELDS:
            t = getattr(self, n)
            if t is not None:
                per = t.numel() // self.batch
                t = t[b * per:(b + 1) * per]
            setattr(h, n, None if t is None else t.cpu().numpy())
        h.slot_expert = h.slot_expert[:self.R * self.n_slot].reshape(self.R, self.n_slot)
        h.phys_count = h.phys_count.reshape(self.R, self.P)
        h.phys_base = h.phys_base.reshape(self.R, self.P)
        if h.U is not None:
            h.U = h.U.reshape(self.E, self.R)
        return h


class Context:
    """uep_ctx wrapper. Shapes are static; see include/uep.h for every argument."""

    def __init__(self, T, k, E, R, n_slot, u_min, beta_num=101, beta_den=100,
                 floor_mode=FLOOR_TOLERANT, gate_dtype=GATE_F32, home_rank=None, device=None):
        self.device = torch.device("cuda", torch.cuda.current_device()) if device is None \
            else torch.device(device)
        cfg = _Config(T, k, E, R, n_slot, u_min, beta_num, beta_den, floor_mode, gate_dtype, None)
        if home_rank is not None:
            arr = (ctypes.c_int32 * E)(*[int(x) for x in home_rank])
            cfg.home_rank = ctypes.cast(arr, ctypes.POINTER(ctypes.c_int32))
        self._h = ctypes.c_void_p()
        with torch.cuda.device(self.device):
            _check(lib().uep_create(ctypes.byref(cfg), ctypes.byref(self._h)))
        self.T, self.k, self.E, self.R, self.n_slot = T, k, E, R, n_slot
        self.S = T * k
        self.gate_dtype = gate_dtype
        sz = _PlanSizes()
        _check(lib().uep_plan_bytes(self._h, ctypes.byref(sz)))
        self.sizes = sz
        self.M, self.P = sz.M, sz.P
        li = _LaunchInfo()
        _check(lib().uep_get_launch_info(self._h, ctypes.byref(li)))
        self.launch_info = {n: getattr(li, n) for n, _ in _LaunchInfo._fields_}

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            lib().uep_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def uep_launch_count(self) -> int:
        """Kernels launched through this context so far (host-side count kept by the library)."""
        return int(lib().uep_launch_count(self._h))

    # ---- allocation helpers (PyTorch = device memory only) ------------------------------
    def workspace_bytes(self) -> int:
        return int(lib().uep_workspace_bytes(self._h))

    def new_workspace(self, stream=None) -> torch.Tensor:
        ws = torch.empty(self.workspace_bytes(), dtype=torch.uint8, device=self.device)
        _check(lib().uep_workspace_init(self._h, _ptr(ws), _stream(stream)))
        return ws

    def new_plan(self, dense_U=False, batch: int = 1) -> Plan:
        """Plan arrays for `batch` instances (uep_plan_batched layout: instance b of every array
        starts b * its element count after instance 0)."""
        sz = self.sizes
        z = lambda n: torch.zeros(max(int(n), 1) * batch, dtype=torch.int32, device=self.device)
        p = Plan(self.E, self.R, self.n_slot, sz.M, sz.P, z(sz.slot_expert), z(sz.inst_off),
                 z(sz.inst_cap), z(sz.inst_cap), z(sz.inst_cap), z(sz.inst_cap), z(sz.phys), z(sz.phys),
                 z(sz.rank_load), z(sz.rank_base), z(sz.scalars), z(sz.U) if dense_U else None)
        p.c = _PlanOut(*[_ptr(getattr(p, n)).value or 0 for n in _PLAN_FIELDS])
        p.batch = batch
        return p

    def new_outputs(self, gate: torch.Tensor | None = None):
        o = [torch.empty((self.T, self.k), dtype=torch.int32, device=self.device) for _ in range(3)]
        og = None if gate is None else torch.zeros(self.S, dtype=gate.dtype, device=self.device)
        return o[0], o[1], o[2], og

    # ---- the C ABI, one method per entry point ---------------------------------------------
    def uep_histogram(self, topk_ids, expert_count, ws, stream=None):
        _check(lib().uep_histogram(self._h, _ptr(topk_ids), _ptr(expert_count), _ptr(ws),
                                   _stream(stream)))

    def uep_plan(self, expert_count, plan: Plan, ws=None, stream=None):
        _check(lib().uep_plan(self._h, _ptr(expert_count), ctypes.byref(plan.c), _ptr(ws),
                              _stream(stream)))

    def uep_remap(self, topk_ids, gate, plan: Plan, out_replica, out_rank, out_offset, out_gate,
                  ws, stream=None):
        _check(lib().uep_remap(self._h, _ptr(topk_ids), _ptr(gate), ctypes.byref(plan.c),
                               _ptr(out_replica), _ptr(out_rank), _ptr(out_offset), _ptr(out_gate),
                               _ptr(ws), _stream(stream)))

    def uep_plan_batched(self, n_inst: int, expert_count, plan: Plan, stream=None):
        assert plan.batch >= n_inst and expert_count.numel() >= n_inst * self.E
        _check(lib().uep_plan_batched(self._h, int(n_inst), _ptr(expert_count), ctypes.byref(plan.c),
                                      _stream(stream)))

    def uep_remap_local(self, topk_ids, gate, plan: Plan, out_replica, out_rank, out_offset, out_gate,
                        n_inflight, ws, stream=None):
        _check(lib().uep_remap_local(self._h, _ptr(topk_ids), _ptr(gate), ctypes.byref(plan.c),
                                     _ptr(out_replica), _ptr(out_rank), _ptr(out_offset),
                                     _ptr(out_gate), _ptr(n_inflight), _ptr(ws), _stream(stream)))

    # ---- token-sharded path (uep.h: uep_shard_*): GPU `shard` of `n_shards` --------------------
    def uep_shard_count(self, shard: int, n_shards: int, topk_ids_local, ws, stream=None):
        _check(lib().uep_shard_count(self._h, int(shard), int(n_shards), _ptr(topk_ids_local), _ptr(ws),
                                     _stream(stream)))

    def uep_shard_rows(self, shard: int, n_shards: int) -> tuple[int, int]:
        """(byte offset inside ws, byte count) of the shard's rows of the count table."""
        off, n = ctypes.c_size_t(0), ctypes.c_size_t(0)
        _check(lib().uep_shard_rows(self._h, int(shard), int(n_shards), ctypes.byref(off), ctypes.byref(n)))
        return int(off.value), int(n.value)

    def uep_shard_finish(self, shard: int, n_shards: int, gate_local, expert_count, plan: Plan,
                         out_replica_local, out_rank_local, out_offset_local, out_gate, n_inflight, ws,
                         stream=None):
        _check(lib().uep_shard_finish(self._h, int(shard), int(n_shards), _ptr(gate_local),
                                      _ptr(expert_count), ctypes.byref(plan.c), _ptr(out_replica_local),
                                      _ptr(out_rank_local), _ptr(out_offset_local), _ptr(out_gate),
                                      _ptr(n_inflight), _ptr(ws), _stream(stream)))

    def uep_remap_rank(self, topk_ids, ws, stream=None):
        _check(lib().uep_remap_rank(self._h, _ptr(topk_ids), _ptr(ws), _stream(stream)))

    def uep_remap_lookup(self, gate, plan: Plan, out_replica, out_rank, out_offset, out_gate, ws,
                         stream=None):
        _check(lib().uep_remap_lookup(self._h, _ptr(gate), ctypes.byref(plan.c), _ptr(out_replica),
                                      _ptr(out_rank), _ptr(out_offset), _ptr(out_gate), _ptr(ws),
                                      _stream(stream)))

    @staticmethod
    def _tensor_lists(src, dst):
        n = len(src)
        assert n == len(dst) and n <= MAX_TENSORS
        srcs = (ctypes.c_void_p * max(n, 1))(*[s.data_ptr() for s in src])
        dsts = (ctypes.c_void_p * max(n, 1))(*[d.data_ptr() for d in dst])
        bpe = (ctypes.c_size_t * max(n, 1))(*[s.nbytes // s.shape[0] for s in src])
        return n, srcs, bpe, dsts

    def uep_pack(self, plan: Plan, src, dst, stream=None):
        """src[j]: [E, ...] contiguous; dst[j]: [R, n_slot, ...] contiguous."""
        n, srcs, bpe, dsts = self._tensor_lists(src, dst)
        _check(lib().uep_pack(self._h, ctypes.byref(plan.c), n, srcs, bpe, dsts, _stream(stream)))

    def uep_grad_reduce(self, plan: Plan, main_grad, slot_grad, stream=None):
        """main_grad[j] [E, ...] fp32 += replicas' slot_grad[j] [R, n_slot, ...]; used slots cleared."""
        n, mains, bpe, slots = self._tensor_lists(main_grad, slot_grad)
        _check(lib().uep_grad_reduce(self._h, ctypes.byref(plan.c), n, mains, bpe, slots,
                                     _stream(stream)))

    def uep_relay_plan(self, plan: Plan, relay_parent, send_volume, stream=None):
        _check(lib().uep_relay_plan(self._h, ctypes.byref(plan.c), _ptr(relay_parent),
                                    _ptr(send_volume), _stream(stream)))

    def uep_remap_inverse(self, out_rank, out_offset, plan: Plan, out_src, stream=None):
        _check(lib().uep_remap_inverse(self._h, _ptr(out_rank), _ptr(out_offset),
                                       ctypes.byref(plan.c), _ptr(out_src), _stream(stream)))

    def uep_balance(self, topk_ids, gate, expert_count, plan: Plan, out_replica, out_rank,
                    out_offset, out_gate, src, dst, ws, stream=None):
        n, srcs, bpe, dsts = self._tensor_lists(src, dst)
        _check(lib().uep_balance(self._h, _ptr(topk_ids), _ptr(gate), _ptr(expert_count),
                                 ctypes.byref(plan.c), _ptr(out_replica), _ptr(out_rank),
                                 _ptr(out_offset), _ptr(out_gate), n, srcs, bpe, dsts, _ptr(ws),
                                 _stream(stream)))

    def uep_balance_host(self, ids_host, gate_host, dev_ids, dev_gate, expert_count, plan: Plan,
                         out_replica, out_rank, out_offset, out_gate, h_replica, h_rank, h_offset,
                         h_gate, h_scalars, src, dst, ws, stream=None):
        """End-to-end leg: HOST (pinned) inputs in, HOST outputs back, synchronises."""
        n, srcs, bpe, dsts = self._tensor_lists(src, dst)
        _check(lib().uep_balance_host(
            self._h, _ptr(ids_host), _ptr(gate_host), _ptr(dev_ids), _ptr(dev_gate),
            _ptr(expert_count), ctypes.byref(plan.c), _ptr(out_replica), _ptr(out_rank),
            _ptr(out_offset), _ptr(out_gate), _ptr(h_replica), _ptr(h_rank), _ptr(h_offset),
            _ptr(h_gate), _ptr(h_scalars), n, srcs, bpe, dsts, _ptr(ws), _stream(stream)))
