"""CPU oracle for the 8-bit blockwise-quantised coefficient format.  TEST INFRASTRUCTURE ONLY.

Only `tests/`, `__graft_entry__.smoke()` and bench.py's `cpu_baseline` / `--impl reference` legs may import this module;
the product never does and shares no code, constants or layout with it.

PAPER.md:56: "The coefficient vector A_{l,h,t}^Z is produced by projecting the original cache vector onto the current basis
and is stored in 8-bit blockwise quantized form."  The paper fixes neither the block nor the scale format; DESIGN.md reading
A27 does:

    block  = 32 consecutive rank columns j of ONE token's coefficient vector of one (layer, kv head, Z); a tier rank r_t
             that is not a multiple of 32 ends in a partial block (r_t = 8, 16: one block; r_t = 48: blocks of 32 and 16)
    scale  = 2^e, a power of two shared by the block (one signed byte e), e the SMALLEST integer with amax <= 127 * 2^e
             where amax = max_j |c_j| over the block; e is clamped to [E_MIN, E_MAX] = [-126, 127]; amax == 0 -> e = E_MIN
    code_j = clamp( rint( c_j / 2^e ), -127, 127 )        (int8, round half to even; -128 is never produced)
    deq_j  = code_j * 2^e

Every step is exact in binary floating point (division by a power of two, rint of an exact quotient), so there is no rounding
order to fix: the quantiser is a function of its fp32 input alone.  deq_j has at most 7 significant bits, so it is EXACTLY a
bfloat16 value: a cache in this format is a special case of the bf16-coefficient cache of Eq. (1) as BASELINE.json reads it,
and everything downstream (reconstruction, attention, footprint closed forms) is `oracle/dwkv_oracle.py` fed with deq.

Append / compress in this format (readings A13, A14 with the quantiser in place of the bf16 rounding):
    c32 = fp32( B[:r_t] @ (x / g) )   (fp64 dot, one rounding to fp32) ; (code, e) = quantise(c32) ; c = deq(code, e)
    residual e = x - g * (c @ B[:r_t])  uses the DEQUANTISED coefficients (it absorbs the quantisation error), then A14.

Bytes per (layer, kv head, token): 2 * (r_t + ceil(r_t / 32)) + f_t * 2 * (d/2 + d/8).

Pins: tests/test_coef8_oracle_pins.py (hand vectors, exact bf16 representability, error bound amax/127 per element,
idempotence, power-of-two covariance, brute-force search of e, footprint closed form).
"""
from __future__ import annotations

import numpy as np

BLOCK = 32
E_MIN, E_MAX = -126, 127


def block_exponent(amax) -> np.ndarray:
    """Smallest integer e with amax <= 127 * 2^e, clamped to [E_MIN, E_MAX]; amax == 0 -> E_MIN.

    Exact: amax = m * 2^x with m in [0.5, 1) (frexp). 127 * 2^e = (127/128) * 2^(e+7), so e = x - 7 if m <= 127/128
    else x - 6."""
    amax = np.asarray(amax, dtype=np.float64)
    m, x = np.frexp(amax)
    e = np.where(m <= 127.0 / 128.0, x - 7, x - 6)
    e = np.where(amax == 0.0, E_MIN, e)
    return np.clip(e, E_MIN, E_MAX).astype(np.int64)


def quantize_coef_i8(c, rank: int | None = None):
    """c [..., r] (fp32 values; only the leading `rank` columns are used, default all).
    Returns (codes int8 [..., r] zero beyond rank, exps int8 [..., ceil(r/32)] with E_MIN for blocks beyond rank)."""
    c = np.asarray(c, dtype=np.float32).astype(np.float64)
    r = c.shape[-1]
    rank = r if rank is None else int(rank)
    nb = (r + BLOCK - 1) // BLOCK
    codes = np.zeros(c.shape, dtype=np.int8)
    exps = np.full(c.shape[:-1] + (nb,), E_MIN, dtype=np.int8)
    for b in range(nb):
        lo, hi = b * BLOCK, min((b + 1) * BLOCK, rank)
        if hi <= lo:
            continue
        blk = c[..., lo:hi]
        e = block_exponent(np.max(np.abs(blk), axis=-1))
        q = np.rint(blk / np.exp2(e.astype(np.float64))[..., None])
        codes[..., lo:hi] = np.clip(q, -127, 127).astype(np.int8)
        exps[..., b] = e.astype(np.int8)
    return codes, exps


def dequant_coef_i8(codes, exps) -> np.ndarray:
    """deq[..., j] = code[..., j] * 2^exps[..., j // 32], exact, float64."""
    codes = np.asarray(codes)
    r = codes.shape[-1]
    scale = np.exp2(np.asarray(exps).astype(np.float64))
    return codes.astype(np.float64) * np.repeat(scale, BLOCK, axis=-1)[..., :r]


def project_quantise(x, B_lead, gate):
    """Append/compress of one vector in this format (header): returns (codes, exps, c = deq, residual fp32).
    x [d] bf16 values, B_lead [r_t, d] leading rows of the shared basis, gate [d]."""
    x = np.asarray(x, np.float64); B_lead = np.asarray(B_lead, np.float64); gate = np.asarray(gate, np.float64)
    c32 = (B_lead @ (x / gate)).astype(np.float32)
    codes, exps = quantize_coef_i8(c32)
    c = dequant_coef_i8(codes, exps)
    resid = (x - gate * (c @ B_lead)).astype(np.float32)
    return codes, exps, c, resid


def append_compress_i8(oc, s, k_new, v_new, tier, flag) -> None:
    """Append/compress in this format into an `oracle.dwkv_oracle.OracleCache` `oc` (token by token, header formulas):
    the cache receives the dequantised coefficients (exact bf16 values) and the fp32 residuals of the flagged tokens."""
    tier = np.asarray(tier, np.uint8); flag = np.asarray(flag, np.uint8)
    n, L, H, d, r = len(tier), oc.L, oc.H, oc.d, oc.r
    coef = {z: np.zeros((n, L, H, r)) for z in "KV"}
    resid = {z: np.zeros((n, L, H, d), np.float32) for z in "KV"}
    for z, x_all, B_all, g_all in (("K", k_new, oc.BK, oc.gK), ("V", v_new, oc.BV, oc.gV)):
        x_all = np.asarray(x_all, np.float64)
        for t in range(n):
            rt = oc.tier_ranks[tier[t]]
            for l in range(L):
                for h in range(H):
                    _, _, c, e = project_quantise(x_all[t, l, h], B_all[l // oc.w, h, :rt, :], g_all[l, h])
                    coef[z][t, l, h, :rt] = c
                    resid[z][t, l, h] = e
    fidx = np.nonzero(flag)[0]
    oc.append_raw(s, tier, flag, coef["K"], coef["V"],
                  residK=resid["K"][fidx] if len(fidx) else None, residV=resid["V"][fidx] if len(fidx) else None)


def footprint_bytes_i8(tier, flag, tier_ranks, d, L, H) -> int:
    """Compressed bytes of one sequence with int8 coefficients: per (layer, kv head, token)
    2*(r_t + ceil(r_t/32)) (codes + one exponent byte per block, K and V) + f_t * 2*(d/2 + d/8)."""
    ranks = np.asarray(tier_ranks, np.int64)[np.asarray(tier)]
    per = 2 * (ranks + (ranks + BLOCK - 1) // BLOCK) + np.asarray(flag).astype(np.int64) * 2 * (d // 2 + d // 8)
    return int(per.sum()) * L * H
