"""Test helpers: build an oracle cache (and the matching raw inputs) from a gen.Workload. No method arithmetic."""
import numpy as np
import torch

import gen
from oracle import dwkv_oracle as orc


def f64(t: torch.Tensor) -> np.ndarray:
    return t.detach().to("cpu", torch.float64).numpy()


def workload_inputs(wl, seq=0, T=None, device="cpu"):
    """All raw inputs of one sequence, token-ordered (torch tensors on `device` + numpy metadata)."""
    tier, flag = gen.make_routing(wl, seq, T)
    cK, cV = gen.make_coef_chunk(wl, seq, 0, tier, device=device)
    nf = int(flag.sum())
    rK, rV = gen.make_resid_chunk(wl, seq, 0, nf, device=device)
    return dict(tier=tier, flag=flag, cK=cK, cV=cV, rK=rK, rV=rV)


def make_oracle(wl, softmax_scale=None):
    BK, BV = gen.make_basis(wl)
    gK, gV = gen.make_gates(wl)
    oc = orc.OracleCache(wl.L, wl.w, wl.H_kv, wl.G, wl.d, wl.tier_ranks, f64(BK), f64(BV), f64(gK), f64(gV),
                         softmax_scale=softmax_scale)
    return oc, (BK, BV, gK, gV)


def oracle_load(oc, seq, inp):
    nf = int(inp["flag"].sum())
    oc.append_raw(seq, inp["tier"], inp["flag"], f64(inp["cK"]), f64(inp["cV"]),
                  residK=inp["rK"].cpu().numpy() if nf else None,
                  residV=inp["rV"].cpu().numpy() if nf else None)


def rel_l2(a, b):
    a = np.asarray(a, np.float64); b = np.asarray(b, np.float64)
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))
