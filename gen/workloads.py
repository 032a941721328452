"""Synthetic DepthWeave-KV caches: shapes, tier routing and value distributions of BASELINE.json configs[0..4].

Recipe (SURVEY.md §8d "Generation rules", restated in DESIGN.md §5). Everything is seeded from BASE_SEED;
metadata (tier / flag per token) is drawn with numpy on the host, tensors with a torch.Generator on the
requested device (CPU for the oracle tests and small parity cases, CUDA for the full-size bench fill).
Tensors are returned already rounded to their storage type (bf16 / fp32), so the oracle and the CUDA
library consume the same bytes.

No method arithmetic lives here: no reconstruction of K-hat/V-hat for attention, no softmax, no int4 quantiser.
`make_dense_kv_chunk` builds "low-rank plus noise" K/V vectors as *inputs* for append/compress; that is an
input distribution, not the compression method.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace
from typing import Optional, Sequence, Tuple

import numpy as np
import torch

BASE_SEED = 260706523

# tensor ids for seed sub-streams
_TID_BASIS, _TID_GATES, _TID_Q, _TID_COEF, _TID_RESID, _TID_ROUTE, _TID_DENSE, _TID_LEN, _TID_OMEGA = range(9)


@dataclass(frozen=True)
class Workload:
    """One BASELINE.json config. Symbols as in SURVEY.md §8: L layers, w layers per group, H_kv KV heads,
    G query heads per KV head, d head dim, tier_ranks ascending (last == basis rank r)."""
    name: str
    index: int                      # BASELINE.json configs[] index (seed sub-stream)
    L: int
    w: int
    H_kv: int
    G: int
    d: int
    tier_ranks: Tuple[int, ...]
    tier_frac: Tuple[float, ...]    # fraction of tokens per tier, low -> high
    resid_frac: float               # fraction of tokens carrying the int4 residual (subset of the top tier)
    S0: int                         # leading tokens that are always top tier (and flagged first)
    T: Tuple[int, ...]              # cached tokens per sequence
    isolated: Optional[Tuple[float, float]] = None   # cfg 4: fraction range of isolated top-tier single tokens
    patterns: Tuple[str, ...] = ()  # per-sequence routing pattern override: "", "all_low", "all_top_flag", "alternating", "mix"
    n_append: int = 0               # cfg 5: tokens appended per sequence per step

    @property
    def r(self) -> int:
        return self.tier_ranks[-1]

    @property
    def M(self) -> int:
        return self.L // self.w

    @property
    def H_q(self) -> int:
        return self.H_kv * self.G

    @property
    def n_seq(self) -> int:
        return len(self.T)

    def with_batch(self, n: int) -> "Workload":
        return replace(self, T=tuple([self.T[0]] * n), name=f"{self.name.rsplit('_b', 1)[0]}_b{n}")


def _ragged_lengths() -> Tuple[int, ...]:
    rng = np.random.Generator(np.random.PCG64([BASE_SEED, 4, _TID_LEN]))
    T = [1, 12347] + [int(x) for x in rng.integers(1024, 32769, size=30)]
    return tuple(T)


WORKLOADS = {
    # BASELINE.json configs[0]: tiny CPU-checkable cache
    "tiny": Workload("tiny", 0, L=2, w=2, H_kv=2, G=2, d=64, tier_ranks=(8, 16), tier_frac=(0.7, 0.3),
                     resid_frac=0.10, S0=32, T=(512,)),
    # configs[1]: Llama-3-8B shape, batch 8, T=16384, flag on the whole top tier
    "llama8b_16k_b8": Workload("llama8b_16k_b8", 1, L=32, w=2, H_kv=8, G=4, d=128, tier_ranks=(8, 16, 32),
                               tier_frac=(0.6, 0.3, 0.1), resid_frac=0.10, S0=128, T=(16384,) * 8),
    # configs[2]: the paper's headline 64K setting, batch 1 / 4 / 8
    "llama8b_64k_b1": Workload("llama8b_64k_b1", 2, L=32, w=2, H_kv=8, G=4, d=128, tier_ranks=(8, 16, 32),
                               tier_frac=(0.65, 0.25, 0.10), resid_frac=0.08, S0=128, T=(65536,)),
    # configs[3]: Llama-3-70B shape
    "llama70b_128k_b1": Workload("llama70b_128k_b1", 3, L=80, w=4, H_kv=8, G=8, d=128, tier_ranks=(8, 24, 48),
                                 tier_frac=(0.6, 0.3, 0.1), resid_frac=0.10, S0=128, T=(131072,),
                                 isolated=(0.01, 0.03)),
    # configs[4]: ragged / adversarial sweep, 32 sequences, +64 appended tokens per step
    "ragged32": Workload("ragged32", 4, L=32, w=2, H_kv=8, G=4, d=128, tier_ranks=(8, 16, 32),
                         tier_frac=(0.6, 0.3, 0.1), resid_frac=0.10, S0=128, T=_ragged_lengths(),
                         patterns=("", "", "all_low", "all_top_flag", "alternating") + ("mix",) * 27,
                         n_append=64),
}
WORKLOADS["llama8b_64k_b4"] = WORKLOADS["llama8b_64k_b1"].with_batch(4)
WORKLOADS["llama8b_64k_b8"] = WORKLOADS["llama8b_64k_b1"].with_batch(8)


def class_of(tier: np.ndarray, flag: np.ndarray) -> np.ndarray:
    """Class id of a token = 2*tier + flag (SURVEY.md §8 symbols). Pure bookkeeping."""
    return (2 * tier.astype(np.int32) + flag.astype(np.int32)).astype(np.int32)


def expected_bytes_per_lht(wl: Workload, tier: np.ndarray, flag: np.ndarray) -> float:
    """Compressed bytes per (layer, kv head, token) for this routing: 4*r_t + f_t*2*(d/2 + d/8)."""
    ranks = np.asarray(wl.tier_ranks)[tier]
    return float(np.mean(4.0 * ranks + flag * 2.0 * (wl.d / 2 + wl.d / 8)))


# ----------------------------------------------------------------------------------------------------------
# routing metadata (host, numpy)
# ----------------------------------------------------------------------------------------------------------

def _mark_spans(rng, assigned: np.ndarray, target: int, T: int, S0: int, order: list) -> None:
    """Mark contiguous spans (start ~ U[S0,T), length ~ U{16..64}) over still-unassigned tokens until `target`
    tokens are marked; the last span is trimmed. `order` receives the marked token ids in generation order."""
    count = int(assigned.sum())
    guard = 0
    while count < target and guard < 100 * T + 1000:
        guard += 1
        lo = min(S0, T - 1)
        start = int(rng.integers(lo, T))
        length = int(rng.integers(16, 65))
        for t in range(start, min(T, start + length)):
            if count >= target:
                break
            if not assigned[t]:
                assigned[t] = True
                order.append(t)
                count += 1


def make_routing(wl: Workload, seq: int = 0, T: Optional[int] = None) -> Tuple[np.ndarray, np.ndarray]:
    """tier[T] (uint8 tier index, 0 = lowest rank) and flag[T] (uint8 residual flag) for sequence `seq`.

    SURVEY.md §8d: tokens 0..S0-1 top tier; seeded contiguous spans of 16..64 tokens for the top tier until
    ceil(f_top*T) tokens, then the same for each lower-middle tier over unassigned tokens; the rest lowest.
    Residual flags: tokens 0..S0-1 first, then top-tier tokens in generation order until ceil(f_res*T)."""
    T = int(wl.T[seq] if T is None else T)
    K = len(wl.tier_ranks)
    rng = np.random.Generator(np.random.PCG64([BASE_SEED, wl.index, _TID_ROUTE, seq]))
    pattern = wl.patterns[seq] if seq < len(wl.patterns) else ""
    tier = np.zeros(T, dtype=np.uint8)
    flag = np.zeros(T, dtype=np.uint8)
    if pattern == "all_low":
        return tier, flag
    if pattern == "all_top_flag":
        tier[:] = K - 1
        flag[:] = 1
        return tier, flag
    if pattern == "alternating":
        tier[:] = (np.arange(T) % K).astype(np.uint8)
        flag[:] = (tier == K - 1).astype(np.uint8) * (np.arange(T) % 2 == 0)
        return tier, flag
    frac = list(wl.tier_frac)
    f_res = wl.resid_frac
    if pattern == "mix":          # cfg 5: per-sequence tier mix
        f_top = float(rng.uniform(0.02, 0.3))
        f_mid = float(rng.uniform(0.1, 0.4))
        frac = [1.0 - f_top - f_mid, f_mid, f_top]
        f_res = f_top
    assigned = np.zeros(T, dtype=bool)
    top_order: list = []
    S0 = wl.S0
    n0 = min(S0, T)
    assigned[:n0] = True
    top_order.extend(range(n0))
    n_top = max(n0, math.ceil(frac[-1] * T))
    if wl.isolated is not None:   # cfg 4: isolated single high-tier tokens, counted inside the top fraction
        u = float(rng.uniform(*wl.isolated))
        n_iso = min(math.ceil(u * T), max(0, n_top - n0))
        cand = rng.permutation(np.arange(n0, T))[:n_iso]
        for t in np.sort(cand):
            assigned[t] = True
            top_order.append(int(t))
    _mark_spans(rng, assigned, n_top, T, S0, top_order)
    tier[assigned] = K - 1
    # middle tiers, from the second highest down to tier 1
    for k in range(K - 2, 0, -1):
        before = assigned.copy()
        target = int(before.sum()) + math.ceil(frac[k] * T)
        target = min(target, T)
        order_k: list = []
        _mark_spans(rng, assigned, target, T, S0, order_k)
        tier[assigned & ~before] = k
    n_res = min(math.ceil(f_res * T), len(top_order))
    if n_res > 0:
        flag[np.asarray(top_order[:n_res], dtype=np.int64)] = 1
    return tier, flag


# ----------------------------------------------------------------------------------------------------------
# tensors (torch; device selectable)
# ----------------------------------------------------------------------------------------------------------

def _gen(device, *stream) -> torch.Generator:
    g = torch.Generator(device=device)
    s = BASE_SEED
    for x in stream:
        s = (s * 6364136223846793005 + int(x) + 1442695040888963407) % (1 << 63)
    g.manual_seed(s)
    return g


def make_basis(wl: Workload, device="cpu") -> Tuple[torch.Tensor, torch.Tensor]:
    """BK, BV: bf16 [M, H_kv, r, d], rows orthonormal before bf16 rounding (QR of a seeded N(0,1) d x r matrix)."""
    out = []
    for z in range(2):
        g = _gen("cpu", wl.index, _TID_BASIS, z)
        a = torch.randn(wl.M, wl.H_kv, wl.d, wl.r, generator=g, dtype=torch.float64)
        qm, _ = torch.linalg.qr(a)                       # columns orthonormal: [M,H,d,r]
        out.append(qm.transpose(-1, -2).contiguous().to(torch.bfloat16).to(device))
    return out[0], out[1]


def make_gates(wl: Workload, device="cpu") -> Tuple[torch.Tensor, torch.Tensor]:
    """gK, gV: bf16 [L, H_kv, d] ~ U(0.5, 1.5)."""
    out = []
    for z in range(2):
        g = _gen("cpu", wl.index, _TID_GATES, z)
        u = torch.rand(wl.L, wl.H_kv, wl.d, generator=g, dtype=torch.float64) + 0.5
        out.append(u.to(torch.bfloat16).to(device))
    return out[0], out[1]


def make_q(wl: Workload, step: int = 0, device="cpu", gain: float = 1.0, n_seq: Optional[int] = None) -> torch.Tensor:
    """q: bf16 [n_seq, L, H_q, d] ~ N(0,1) * gain (gain 8 / 64 = the peaked-softmax stress variants, pin P12)."""
    n = wl.n_seq if n_seq is None else n_seq
    g = _gen("cpu", wl.index, _TID_Q, step)
    q = torch.randn(n, wl.L, wl.H_q, wl.d, generator=g, dtype=torch.float32) * gain
    return q.to(torch.bfloat16).to(device)


def make_coef_chunk(wl: Workload, seq: int, t0: int, tier: np.ndarray, device="cpu",
                    layers: Optional[Sequence[int]] = None) -> Tuple[torch.Tensor, torch.Tensor]:
    """Coefficients for tokens [t0, t0+len(tier)): bf16 [n, L, H_kv, r], c_j ~ N(0, var=1/(1+j)) for j < r_t,
    exactly zero for j >= r_t. K and V drawn independently."""
    n = len(tier)
    ranks = torch.as_tensor(np.asarray(wl.tier_ranks, dtype=np.int64)[tier], device=device)       # [n]
    j = torch.arange(wl.r, device=device)
    std = (1.0 / (1.0 + j.to(torch.float32))).sqrt()
    mask = (j[None, :] < ranks[:, None])                                                          # [n, r]
    out = []
    for z in range(2):
        g = _gen(device, wl.index, _TID_COEF, z, seq, t0)
        c = torch.randn(n, wl.L, wl.H_kv, wl.r, generator=g, device=device, dtype=torch.float32)
        c = c * std
        c = torch.where(mask[:, None, None, :], c, torch.zeros((), device=device))
        out.append(c.to(torch.bfloat16))
    return out[0], out[1]


def make_resid_chunk(wl: Workload, seq: int, t0: int, n_flagged: int, device="cpu") -> Tuple[torch.Tensor, torch.Tensor]:
    """Residual vectors for the flagged tokens of a chunk: fp32 [n_flagged, L, H_kv, d] ~ N(0, 0.05^2)."""
    out = []
    for z in range(2):
        g = _gen(device, wl.index, _TID_RESID, z, seq, t0)
        x = torch.randn(n_flagged, wl.L, wl.H_kv, wl.d, generator=g, device=device, dtype=torch.float32) * 0.05
        out.append(x)
    return out[0], out[1]


def make_dense_kv_chunk(wl: Workload, seq: int, t0: int, n: int, BK, BV, gK, gV, device="cpu") -> Tuple[torch.Tensor, torch.Tensor]:
    """Dense K/V inputs for append/compress (cfg 5): bf16 [n, L, H_kv, d], low-rank-plus-noise vectors
    x = gate * (c @ B) + e with c ~ N(0, 1/(1+j)) full rank and e ~ N(0, 0.05^2)."""
    j = torch.arange(wl.r, device=device)
    std = (1.0 / (1.0 + j.to(torch.float32))).sqrt()
    lay_group = torch.arange(wl.L, device=device) // wl.w
    out = []
    for z, (B, gt) in enumerate(((BK, gK), (BV, gV))):
        g = _gen(device, wl.index, _TID_DENSE, z, seq, t0)
        c = torch.randn(n, wl.L, wl.H_kv, wl.r, generator=g, device=device, dtype=torch.float32) * std
        e = torch.randn(n, wl.L, wl.H_kv, wl.d, generator=g, device=device, dtype=torch.float32) * 0.05
        Bl = B.to(device=device, dtype=torch.float32)[lay_group]                       # [L,H,r,d]
        x = torch.einsum("nlhr,lhrd->nlhd", c, Bl) * gt.to(device=device, dtype=torch.float32)[None] + e
        out.append(x.to(torch.bfloat16))
    return out[0], out[1]


def make_omega(wl: Workload, n: int, n_sketch: int, device="cpu") -> torch.Tensor:
    """Random test matrix of the basis sketch (an INPUT of dwkv_build_basis): bf16 [w, n_sketch, n] ~ N(0, 1)."""
    g = _gen(device, wl.index, _TID_OMEGA, n_sketch)
    return torch.randn(wl.w, n_sketch, n, generator=g, device=device, dtype=torch.float32).to(torch.bfloat16)
