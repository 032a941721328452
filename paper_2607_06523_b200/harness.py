"""Harness helpers shared by tests, bench.py and smoke(): create a cache for a gen.Workload and fill it from the seeded
generators through dwkv_append_raw. No method arithmetic and no oracle here."""
from __future__ import annotations

from typing import Dict, Iterable, Optional, Tuple

import numpy as np
import torch

import gen
from . import binding

PAGE_LH_BYTES = 64 * 1024


def class_block_bytes(rank: int, flag: int, d: int) -> int:
    return 2 * (rank // 8) * 512 + flag * 40 * d


def arena_bytes_for(wl: gen.Workload, routings, slack_pages_per_class: int = 1, slack_tokens: int = 0) -> int:
    """Pages needed for the given per-sequence (tier, flag) routings, plus slack for appended tokens: `slack_pages_per_class` pages
    per (sequence, class), and room for `slack_tokens` more tokens per sequence in whichever class they fall."""
    page = wl.L * wl.H_kv * PAGE_LH_BYTES
    pages = 0
    for tier, flag in routings:
        cls = gen.class_of(tier, flag)
        for k in range(2 * len(wl.tier_ranks)):
            tpp = (PAGE_LH_BYTES // class_block_bytes(wl.tier_ranks[k >> 1], k & 1, wl.d)) * 32
            n = int((cls == k).sum())
            pages += (n + tpp - 1) // tpp + slack_pages_per_class + (slack_tokens + tpp - 1) // tpp
    return pages * page


def make_cache(wl: gen.Workload, n_seqs: Optional[int] = None, max_tokens: Optional[int] = None, arena_bytes: int = 0,
               device: int = 0, softmax_scale: float = 0.0, coef_int8: bool = False):
    n_seqs = wl.n_seq if n_seqs is None else n_seqs
    max_tokens = (max(wl.T) + 4096) if max_tokens is None else max_tokens
    cache = binding.DwkvCache(wl.L, wl.w, wl.H_kv, wl.H_q, wl.d, list(wl.tier_ranks), n_seqs, max_tokens,
                              softmax_scale=softmax_scale, device=device, arena_bytes=arena_bytes)
    if coef_int8:       # 8-bit coefficient planes (dwkv.h option "coef_int8"): must be chosen while the cache is empty
        cache.set_option("coef_int8", 1)
    dev = torch.device("cuda", device)
    BK, BV = gen.make_basis(wl, device=dev)
    gK, gV = gen.make_gates(wl, device=dev)
    cache.set_basis(BK, BV)
    cache.set_gates(gK, gV)
    return cache, (BK, BV, gK, gV)


def fill_sequence(cache, wl: gen.Workload, seq: int, seq_id: int, tier: np.ndarray, flag: np.ndarray, device: int = 0,
                  chunk: int = 4096, keep: Iterable[Tuple[int, int]] = ()) -> Dict:
    """Generate the sequence chunk by chunk on the GPU and load it with dwkv_append_raw (mode A: fp32 residuals, the
    library quantises). `keep` lists (layer, kv head) slices whose *generator outputs* are copied to the host so a
    checker can recompute them independently. Returns {(l,h): dict(cK, cV, rK, rV)} of host tensors."""
    dev = torch.device("cuda", device)
    keep = list(keep)
    kept = {lh: dict(cK=[], cV=[], rK=[], rV=[]) for lh in keep}
    T = len(tier)
    for t0 in range(0, T, chunk):
        t1 = min(T, t0 + chunk)
        tr, fl = tier[t0:t1], flag[t0:t1]
        cK, cV = gen.make_coef_chunk(wl, seq, t0, tr, device=dev)
        nf = int(fl.sum())
        rK = rV = None
        if nf:
            rK, rV = gen.make_resid_chunk(wl, seq, t0, nf, device=dev)
        cache.append_raw(seq_id, tr, fl, cK, cV, residK=rK, residV=rV)
        for (l, h) in keep:
            kept[(l, h)]["cK"].append(cK[:, l, h].cpu())
            kept[(l, h)]["cV"].append(cV[:, l, h].cpu())
            if nf:
                kept[(l, h)]["rK"].append(rK[:, l, h].cpu())
                kept[(l, h)]["rV"].append(rV[:, l, h].cpu())
        torch.cuda.current_stream().synchronize()   # generator tensors are freed after each chunk
    out = {}
    for lh, v in kept.items():
        out[lh] = {k: (torch.cat(x) if len(x) else None) for k, x in v.items()}
    return out
