"""Seeded synthetic inputs shaped like the paper's workloads.

This module serves BOTH the oracle-side tests and the CUDA path and therefore holds none
of the method's arithmetic: no histogram, no planning, no remap.  It only draws routing
ids, gate weights and expert-state bytes.  Everything that decides an integer is done in
int64 with a counter-based hash, so the same (seed, shape) gives the same bytes on CPU and
on CUDA; the oracle and the kernels are always handed the same tensors anyway.

The paper's routing traces, models and corpus are not available; its own Fig. 15 uses a
synthetic power-law load.  Zipf(s) top-k routing stands in for them.
"""
from __future__ import annotations

import numpy as np
import torch

_M64 = (1 << 64) - 1


def _s64(x: int) -> int:
    """Python int -> the int64 with the same low 64 bits."""
    x &= _M64
    return x - (1 << 64) if x >= (1 << 63) else x


_C1 = _s64(0xBF58476D1CE4E5B9)
_C2 = _s64(0x94D049BB133111EB)
_G = _s64(0x9E3779B97F4A7C15)


def _lsr(x: torch.Tensor, n: int) -> torch.Tensor:
    return (x >> n) & ((1 << (64 - n)) - 1)


def _mix(x: torch.Tensor) -> torch.Tensor:
    """splitmix64 finaliser on int64 tensors (wrapping arithmetic)."""
    x = (x ^ _lsr(x, 30)) * _C1
    x = (x ^ _lsr(x, 27)) * _C2
    return x ^ _lsr(x, 31)


def _mix_int(x: int) -> int:
    x &= _M64
    x = ((x ^ (x >> 30)) * 0xBF58476D1CE4E5B9) & _M64
    x = ((x ^ (x >> 27)) * 0x94D049BB133111EB) & _M64
    return x ^ (x >> 31)


def instance_seed(base: int, layer: int, microbatch: int) -> int:
    """seed of one (layer, microbatch) instance = hash(base, layer, microbatch)."""
    return _mix_int(_mix_int(_mix_int(base) + layer * 0x9E3779B97F4A7C15) + microbatch + 1) >> 1


def _stream(seed: int, n: int, lane: int, device) -> torch.Tensor:
    """n non-negative 63-bit hashes: counter = element index, keyed by (seed, lane)."""
    key = _s64(_mix_int(_mix_int(seed) + lane * 0x9E3779B97F4A7C15))
    idx = torch.arange(n, dtype=torch.int64, device=device)
    return _lsr(_mix(_mix(idx * _G + key) + key), 1)


def zipf_weights(E: int, s: float) -> np.ndarray:
    """Integer popularity weights w_p ∝ 1/p^s (p = 1..E), scaled to sum ≈ 2^40, each >= 1."""
    w = 1.0 / np.power(np.arange(1, E + 1, dtype=np.float64), float(s))
    return np.maximum(1, np.rint(w / w.sum() * float(1 << 40))).astype(np.int64)


def expert_permutation(E: int, seed: int) -> np.ndarray:
    """Seeded permutation: popularity position p -> expert id."""
    h = _stream(seed, E, 7, "cpu").numpy()
    return np.argsort(h, kind="stable").astype(np.int64)


def zipf_topk_ids(T: int, k: int, E: int, s: float, seed: int, device="cpu") -> torch.Tensor:
    """topk_ids[T,k] int32: per token, k distinct experts drawn WITHOUT replacement with
    probability ∝ Zipf(s) weights assigned to experts through a seeded permutation.
    s = 0 is the uniform distribution.  Exact sequential sampling: draw d takes a hash
    u in [0, remaining mass) and skips the intervals of the experts already chosen."""
    assert 1 <= k <= E
    iw = zipf_weights(E, s)
    hi = torch.from_numpy(np.cumsum(iw)).to(device)            # inclusive CDF over positions
    lo = hi - torch.from_numpy(iw).to(device)
    w = torch.from_numpy(iw).to(device)
    perm = torch.from_numpy(expert_permutation(E, seed)).to(device)
    total = int(iw.sum())
    chosen = torch.empty((T, 0), dtype=torch.int64, device=device)   # positions, ascending
    order = torch.empty((T, k), dtype=torch.int64, device=device)    # positions, draw order
    removed = torch.zeros(T, dtype=torch.int64, device=device)
    for d in range(k):
        u = _stream(seed, T, 100 + d, device) % (total - removed)
        for c in range(d):                                     # ascending position order
            pc = chosen[:, c]
            u = torch.where(u >= lo[pc], u + w[pc], u)
        pos = torch.searchsorted(hi, u, right=True).clamp_(max=E - 1)
        order[:, d] = pos
        removed += w[pos]
        chosen = torch.sort(torch.cat([chosen, pos[:, None]], dim=1), dim=1).values
    return perm[order].to(torch.int32).contiguous()


def one_expert_ids(T: int, k: int, e: int, device="cpu") -> torch.Tensor:
    """Adversarial routing: every slot goes to expert e (duplicates inside a token)."""
    return torch.full((T, k), int(e), dtype=torch.int32, device=device)


def gates_uniform_renorm(T: int, k: int, seed: int, device="cpu") -> torch.Tensor:
    """fp32 gate weights: uniform(0,1) per slot, renormalised to sum 1 per token."""
    u = (_lsr(_stream(seed, T * k, 200, device), 39).to(torch.float32) + 0.5) * (2.0 ** -24)
    u = u.view(T, k)
    return (u / u.sum(dim=1, keepdim=True)).contiguous()


def gates_softmax_bf16(T: int, k: int, seed: int, device="cpu") -> torch.Tensor:
    """bf16 gate weights: softmax over k seeded N(0,1) logits per token."""
    g = torch.Generator(device=device)
    g.manual_seed(seed & 0x7FFFFFFF)
    logits = torch.randn((T, k), generator=g, device=device, dtype=torch.float32)
    return torch.softmax(logits, dim=1).to(torch.bfloat16).contiguous()


def expert_state(E: int, elems_per_expert: int, seed: int, dtype=torch.bfloat16,
                 device="cpu", std: float = 0.02) -> torch.Tensor:
    """[E, elems_per_expert] tensor ~ N(0, std) (any byte pattern serves the pack)."""
    g = torch.Generator(device=device)
    g.manual_seed(seed & 0x7FFFFFFF)
    out = torch.empty((E, elems_per_expert), dtype=dtype, device=device)
    step = max(1, (1 << 28) // max(1, elems_per_expert))       # bound the fp32 temporary
    for a in range(0, E, step):
        b = min(E, a + step)
        out[a:b] = (torch.randn((b - a, elems_per_expert), generator=g, device=device,
                                dtype=torch.float32) * std).to(dtype)
    return out


# The five BASELINE.json configs (SURVEY.md §8 size table). u_min / beta per S23.
CONFIGS = {
    "tiny": dict(T=4096, k=2, E=16, R=4, n_slot=1, u_min=64, zipf_s=1.2, gate="f32",
                 state=[("w", 256 * 512, "bf16")]),
    "glm_air": dict(T=65536, k=8, E=128, R=32, n_slot=2, u_min=1024, zipf_s=1.0, gate="bf16",
                    state=[("gate_up_down", 3 * 4096 * 1408, "bf16")]),
    "dsv3_prefill": dict(T=262144, k=8, E=256, R=64, n_slot=2, u_min=1024, zipf_s=1.0,
                         gate="f32", state=[("gate_up_down", 3 * 7168 * 2048, "bf16")]),
    "dsv3_train": dict(T=262144, k=8, E=256, R=64, n_slot=2, u_min=1024, zipf_s=None,
                       gate="f32", layers=58, microbatches=4,
                       state=[("w", 7168 * 2048, "bf16"), ("grad", 7168 * 2048, "f32"),
                              ("adam_m", 7168 * 2048, "f32"), ("adam_v", 7168 * 2048, "f32")]),
}


def stress_u_min(S: int, R: int) -> int:
    """S23: u_min = max(1, (S/R)/32) keeps the paper's 1024 : 32768 ratio."""
    return max(1, (S // R) // 32)


def train_sweep_s(base_seed: int, layer: int, microbatch: int) -> float:
    """dsv3_train: Zipf s ~ U[0.6, 1.6] per (layer, microbatch)."""
    h = instance_seed(base_seed ^ 0x5EED, layer, microbatch)
    return 0.6 + (h % 1000001) / 1000000.0
