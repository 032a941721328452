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


def oracle_slice_from_kept(wl, consts, tier, flag, kept_lh, q_lh, l, h, scale=None):
    """Oracle attention for one (layer, kv head) from the generator outputs kept on the host.
    Returns (o [G,d], V-hat [T,d], (codeK, scaleK, codeV, scaleV) full-length arrays)."""
    BK, BV, gK, gV = consts
    T = len(tier)
    ranks = np.asarray(wl.tier_ranks)[tier]
    d = wl.d
    cK_ = np.zeros((T, d), np.int8); cV_ = np.zeros((T, d), np.int8)
    sK_ = np.zeros((T, d // 16), np.float16); sV_ = np.zeros((T, d // 16), np.float16)
    idx = np.nonzero(flag)[0]
    if len(idx):
        cK_[idx], sK_[idx] = orc.quantize_int4_g16(kept_lh["rK"].numpy())
        cV_[idx], sV_[idx] = orc.quantize_int4_g16(kept_lh["rV"].numpy())
    scale = (1.0 / np.sqrt(d)) if scale is None else scale
    o, _, V = orc.attention_slice(f64(kept_lh["cK"]), f64(kept_lh["cV"]), ranks, flag, cK_, sK_, cV_, sV_,
                                  f64(BK)[l // wl.w, h], f64(BV)[l // wl.w, h], f64(gK)[l, h], f64(gV)[l, h],
                                  q_lh, scale)
    return o, V, (cK_, sK_, cV_, sV_)


def check_output(o_gpu, o_ref, vmax, what=""):
    """BASELINE.json north_star tolerance: max-abs <= 2e-3 * max|V-hat| and relative L2 <= 5e-3."""
    err = float(np.abs(np.asarray(o_gpu, np.float64) - o_ref).max())
    rel = rel_l2(o_gpu, o_ref)
    assert err <= 2e-3 * vmax, f"{what}: max-abs {err:.3e} > 2e-3*{vmax:.3e}"
    assert rel <= 5e-3, f"{what}: rel-L2 {rel:.3e} > 5e-3"
    return err, rel
