"""Pins for the CPU oracle. CPU only.

The paper prints no worked numeric example of the decode-attention path, so the oracle is pinned to what the
paper and the mathematics fix: special cases that reduce to a library routine (torch SDPA in float64), closed
forms, invariants, a hand-derived brute-force case, and hand-derived quantiser vectors.
"""
import math
import os

import numpy as np
import pytest
import torch

import gen
from oracle import dwkv_oracle as orc
from helpers import f64, make_oracle, oracle_load, workload_inputs, rel_l2


def sdpa64(q, K, V, scale):
    """Independent routine: torch.nn.functional.scaled_dot_product_attention in float64 on CPU."""
    qt = torch.tensor(q, dtype=torch.float64)[None]          # [1,G,d]
    Kt = torch.tensor(K, dtype=torch.float64)[None]
    Vt = torch.tensor(V, dtype=torch.float64)[None]
    return torch.nn.functional.scaled_dot_product_attention(qt, Kt, Vt, scale=scale)[0].numpy()


def small_cache(rng, T=37, L=2, w=2, H=2, G=2, d=32, ranks=(8, 16), identity=False, unit_gates=False, resid=True):
    r = ranks[-1]
    M = L // w
    if identity:
        assert r == d
        BK = np.broadcast_to(np.eye(d), (M, H, d, d)).copy()
        BV = BK.copy()
    else:
        BK = np.stack([[np.linalg.qr(rng.standard_normal((d, r)))[0].T for _ in range(H)] for _ in range(M)])
        BV = np.stack([[np.linalg.qr(rng.standard_normal((d, r)))[0].T for _ in range(H)] for _ in range(M)])
    gK = np.ones((L, H, d)) if unit_gates else rng.uniform(0.5, 1.5, (L, H, d))
    gV = np.ones((L, H, d)) if unit_gates else rng.uniform(0.5, 1.5, (L, H, d))
    oc = orc.OracleCache(L, w, H, G, d, ranks, BK, BV, gK, gV)
    tier = rng.integers(0, len(ranks), T).astype(np.uint8)
    flag = (rng.random(T) < 0.3).astype(np.uint8) if resid else np.zeros(T, np.uint8)
    cK = rng.standard_normal((T, L, H, r))
    cV = rng.standard_normal((T, L, H, r))
    nf = int(flag.sum())
    rK = (rng.standard_normal((nf, L, H, d)) * 0.05).astype(np.float32)
    rV = (rng.standard_normal((nf, L, H, d)) * 0.05).astype(np.float32)
    oc.append_raw(0, tier, flag, cK, cV, residK=rK if nf else None, residV=rV if nf else None)
    return oc, dict(tier=tier, flag=flag, cK=cK, cV=cV, rK=rK, rV=rV, BK=BK, BV=BV, gK=gK, gV=gV)


# P1 -------------------------------------------------------------------------------------------------------
def test_p1_identity_basis_equals_dense_attention():
    """r = d, B = I, unit gates, no residual  ==  uncompressed attention on K = cK, V = cV (BASELINE north_star)."""
    rng = np.random.default_rng(1)
    d = 32
    oc, x = small_cache(rng, T=53, d=d, ranks=(d,), identity=True, unit_gates=True, resid=False)
    q = rng.standard_normal((oc.H * oc.G, d))
    for l in range(oc.L):
        o = oc.decode_attention(l, 0, q)
        for h in range(oc.H):
            ref = sdpa64(q[h * oc.G:(h + 1) * oc.G], x["cK"][:, l, h], x["cV"][:, l, h], 1.0 / math.sqrt(d))
            np.testing.assert_allclose(o[h * oc.G:(h + 1) * oc.G], ref, rtol=1e-12, atol=1e-14)


# P2 -------------------------------------------------------------------------------------------------------
def test_p2_exact_low_rank_dense_equivalence():
    """Dense K = gate * (C_lead @ B) + deq built independently with einsum/loops, SDPA vs the oracle."""
    rng = np.random.default_rng(2)
    oc, x = small_cache(rng, T=41, d=32, ranks=(8, 16))
    ranks = np.asarray(oc.tier_ranks)[x["tier"]]
    q = rng.standard_normal((oc.H * oc.G, oc.d))
    fidx = np.cumsum(x["flag"]) - 1
    for l in range(oc.L):
        o = oc.decode_attention(l, 0, q)
        for h in range(oc.H):
            K = np.zeros((41, oc.d)); V = np.zeros((41, oc.d))
            for t in range(41):
                for j in range(ranks[t]):
                    K[t] += x["cK"][t, l, h, j] * x["BK"][l // oc.w, h, j]
                    V[t] += x["cV"][t, l, h, j] * x["BV"][l // oc.w, h, j]
                K[t] *= x["gK"][l, h]; V[t] *= x["gV"][l, h]
                if x["flag"][t]:
                    for z, X, R in (("K", K, x["rK"]), ("V", V, x["rV"])):
                        e = R[fidx[t], l, h]
                        for g0 in range(0, oc.d, 16):
                            grp = e[g0:g0 + 16]
                            s = np.float16(min(np.float32(np.max(np.abs(grp))) / np.float32(7), np.float32(65504)))
                            if float(s) != 0.0:
                                code = np.clip(np.rint(grp / np.float32(s)), -7, 7)
                                X[t, g0:g0 + 16] += code.astype(np.float64) * float(s)
            ref = sdpa64(q[h * oc.G:(h + 1) * oc.G], K, V, 1.0 / math.sqrt(oc.d))
            np.testing.assert_allclose(o[h * oc.G:(h + 1) * oc.G], ref, rtol=1e-11, atol=1e-13)


# P3 -------------------------------------------------------------------------------------------------------
def test_p3_softmax_shift_invariance():
    """Adding the same vector a (support j < r_0) to every token's cK shifts all scores equally: o unchanged."""
    rng = np.random.default_rng(3)
    oc, x = small_cache(rng, T=64)
    q = rng.standard_normal((oc.H * oc.G, oc.d)) * 4
    o1 = np.stack([oc.decode_attention(l, 0, q) for l in range(oc.L)])
    a = np.zeros(oc.r); a[:oc.tier_ranks[0]] = rng.standard_normal(oc.tier_ranks[0]) * 30
    oc.seqs[0]["cK"] = oc.seqs[0]["cK"] + a
    o2 = np.stack([oc.decode_attention(l, 0, q) for l in range(oc.L)])
    np.testing.assert_allclose(o1, o2, rtol=1e-9, atol=1e-12)


# P4 -------------------------------------------------------------------------------------------------------
def test_p4_convex_combination_bounds():
    rng = np.random.default_rng(4)
    oc, _ = small_cache(rng, T=80)
    q = rng.standard_normal((oc.H * oc.G, oc.d)) * 3
    for l in range(oc.L):
        o = oc.decode_attention(l, 0, q)
        for h in range(oc.H):
            _, V = oc.khat_vhat(0, l, h)
            for g in range(oc.G):
                row = o[h * oc.G + g]
                assert np.all(row <= V.max(axis=0) + 1e-12) and np.all(row >= V.min(axis=0) - 1e-12)


# P5 -------------------------------------------------------------------------------------------------------
def test_p5_zero_query_gives_mean_of_vhat():
    rng = np.random.default_rng(5)
    oc, x = small_cache(rng, T=33)
    q = np.zeros((oc.H * oc.G, oc.d))
    ranks = np.asarray(oc.tier_ranks)[x["tier"]]
    for l in range(oc.L):
        o = oc.decode_attention(l, 0, q)
        for h in range(oc.H):
            lead = np.arange(oc.r)[None] < ranks[:, None]
            V = x["gV"][l, h] * np.einsum("tj,jd->td", x["cV"][:, l, h] * lead, x["BV"][l // oc.w, h])
            codes, sc = orc.quantize_int4_g16(x["rV"][:, l, h])
            V[x["flag"].astype(bool)] += codes.reshape(-1, oc.d // 16, 16).astype(np.float64).__mul__(
                sc.astype(np.float64)[..., None]).reshape(-1, oc.d)
            np.testing.assert_allclose(o[h * oc.G:(h + 1) * oc.G], np.broadcast_to(V.mean(0), (oc.G, oc.d)),
                                       rtol=1e-11, atol=1e-13)


# P6 -------------------------------------------------------------------------------------------------------
def test_p6_single_token_and_identical_tokens():
    rng = np.random.default_rng(6)
    oc, _ = small_cache(rng, T=1)
    q = rng.standard_normal((oc.H * oc.G, oc.d)) * 5
    for l in range(oc.L):
        o = oc.decode_attention(l, 0, q)
        for h in range(oc.H):
            _, V = oc.khat_vhat(0, l, h)
            np.testing.assert_allclose(o[h * oc.G:(h + 1) * oc.G], np.broadcast_to(V[0], (oc.G, oc.d)), rtol=0, atol=1e-15)
    # all tokens identical -> o = V-hat[0] for any q
    oc2, x = small_cache(rng, T=1, resid=False)
    S = oc2.seqs[0]
    for k in ("cK", "cV", "codeK", "codeV", "scaleK", "scaleV", "tier", "flag", "cls", "slot"):
        S[k] = np.repeat(S[k], 9, axis=0)
    o = oc2.decode_attention(0, 0, q)
    _, V = oc2.khat_vhat(0, 0, 1)
    np.testing.assert_allclose(o[oc2.G:2 * oc2.G], np.broadcast_to(V[0], (oc2.G, oc2.d)), rtol=1e-13, atol=1e-15)


# P7 -------------------------------------------------------------------------------------------------------
def test_p7_token_permutation_invariance():
    rng = np.random.default_rng(7)
    oc, x = small_cache(rng, T=50)
    q = rng.standard_normal((oc.H * oc.G, oc.d)) * 2
    o1 = oc.decode_attention(1, 0, q)
    perm = rng.permutation(50)
    fl = x["flag"].astype(bool)
    fidx = np.cumsum(x["flag"]) - 1
    order_f = [fidx[t] for t in perm if fl[t]]
    oc2 = orc.OracleCache(oc.L, oc.w, oc.H, oc.G, oc.d, oc.tier_ranks, x["BK"], x["BV"], x["gK"], x["gV"])
    oc2.append_raw(0, x["tier"][perm], x["flag"][perm], x["cK"][perm], x["cV"][perm],
                   residK=x["rK"][order_f], residV=x["rV"][order_f])
    np.testing.assert_allclose(oc2.decode_attention(1, 0, q), o1, rtol=1e-11, atol=1e-14)


# P8 -------------------------------------------------------------------------------------------------------
def test_p8_tier_and_flag_semantics():
    """tier-r0 token == same token at the top tier with zeros beyond r0; flagged token with all-zero codes == unflagged
    ("represented solely by the shared basis component")."""
    rng = np.random.default_rng(8)
    oc, x = small_cache(rng, T=40, resid=False)
    q = rng.standard_normal((oc.H * oc.G, oc.d))
    o1 = oc.decode_attention(0, 0, q)
    ranks = np.asarray(oc.tier_ranks)[x["tier"]]
    lead = (np.arange(oc.r)[None] < ranks[:, None])[:, None, None, :]
    oc2 = orc.OracleCache(oc.L, oc.w, oc.H, oc.G, oc.d, oc.tier_ranks, x["BK"], x["BV"], x["gK"], x["gV"])
    T = 40
    top = np.full(T, len(oc.tier_ranks) - 1, np.uint8)
    flag = np.ones(T, np.uint8)
    zc = np.zeros((T, oc.L, oc.H, oc.d), np.int8)
    zs = np.ones((T, oc.L, oc.H, oc.d // 16), np.float16)
    oc2.append_raw(0, top, flag, x["cK"] * lead, x["cV"] * lead, codeK=zc, scaleK=zs, codeV=zc, scaleV=zs)
    np.testing.assert_allclose(oc2.decode_attention(0, 0, q), o1, rtol=1e-12, atol=1e-15)


# P9 -------------------------------------------------------------------------------------------------------
def test_p9_hand_derived_case():
    """d=32, r=8, tier ranks (4, 8), T=3, G=1, softmax scale 1/4. Derivation (by hand):
      BK[j] = e_j, BV[j] = e_{31-j}; gK = 2 at ch 0, 0.5 at ch 1, else 1; gV = 2 at ch >= 16, else 1.
      tok0: tier 1, cK = e_0           -> K0 = 2 e_0 ;            cV = e_0 -> V0 = 2 e_31
      tok1: tier 0 (r_t=4), cK = (0,2,0,0,9,9,9,9) -> K1 = e_1 (9s ignored); cV = (0,0,0,3,5,0,0,0) -> V1 = 6 e_28
      tok2: tier 1, flagged, cK = 0, codesK: ch0 = 4 (scale g0 = 0.5), ch17 = 7 (scale g1 = 1.0) -> K2 = 2 e_0 + 7 e_17
            cV = e_7 -> 2 e_24 ; codesV: ch3 = 6 (scale g0 = 0.5), ch20 = -3 (scale g1 = 0.25) -> V2 = 2 e_24 + 3 e_3 - 0.75 e_20
      q = 2 ln2 e_0 + 1 e_4 - (4 ln2 / 7) e_17
      s0 = (2 ln2 * 2)/4 = ln2 ; s1 = 0 (q_1 = 0, and the ignored 9 at j=4 would give 9/4) ; s2 = (4 ln2 - 4 ln2)/4 = 0
      p = (2,1,1)/4 ;  o = 0.5 V0 + 0.25 V1 + 0.25 V2 = e_31 + 1.5 e_28 + 0.5 e_24 + 0.75 e_3 - 0.1875 e_20."""
    d, r = 32, 8
    BK = np.zeros((1, 1, r, d)); BV = np.zeros((1, 1, r, d))
    for j in range(r):
        BK[0, 0, j, j] = 1.0
        BV[0, 0, j, 31 - j] = 1.0
    gK = np.ones((1, 1, d)); gK[0, 0, 0] = 2.0; gK[0, 0, 1] = 0.5
    gV = np.ones((1, 1, d)); gV[0, 0, 16:] = 2.0
    oc = orc.OracleCache(1, 1, 1, 1, d, (4, 8), BK, BV, gK, gV, softmax_scale=0.25)
    cK = np.zeros((3, 1, 1, r)); cV = np.zeros((3, 1, 1, r))
    cK[0, 0, 0, 0] = 1; cK[1, 0, 0] = [0, 2, 0, 0, 9, 9, 9, 9]
    cV[0, 0, 0, 0] = 1; cV[1, 0, 0] = [0, 0, 0, 3, 5, 0, 0, 0]; cV[2, 0, 0, 7] = 1
    codeK = np.zeros((1, 1, 1, d), np.int8); codeK[0, 0, 0, 0] = 4; codeK[0, 0, 0, 17] = 7
    codeV = np.zeros((1, 1, 1, d), np.int8); codeV[0, 0, 0, 3] = 6; codeV[0, 0, 0, 20] = -3
    scaleK = np.array([0.5, 1.0], np.float16).reshape(1, 1, 1, 2)
    scaleV = np.array([0.5, 0.25], np.float16).reshape(1, 1, 1, 2)
    oc.append_raw(0, [1, 0, 1], [0, 0, 1], cK, cV, codeK=codeK, scaleK=scaleK, codeV=codeV, scaleV=scaleV)
    q = np.zeros((1, d)); q[0, 0] = 2 * math.log(2); q[0, 4] = 1.0; q[0, 17] = -4 * math.log(2) / 7
    o = oc.decode_attention(0, 0, q)
    exp = np.zeros(d)          # the hand-derived output, stored with its derivation under tests/golden/
    for line in open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "p9_hand_case.txt")):
        if line.strip() and not line.startswith("#"):
            ch, val = line.split()
            exp[int(ch)] = float(val)
    assert np.count_nonzero(exp) == 5 and exp[31] == 1.0 and exp[20] == -0.1875
    np.testing.assert_allclose(o[0], exp, rtol=0, atol=1e-14)


# P10 ------------------------------------------------------------------------------------------------------
def test_p10_quantiser_hand_vectors():
    z = np.zeros(16, np.float32)
    c, s = orc.quantize_int4_g16(z)                         # all-zero group
    assert float(s[0]) == 0.0 and not c.any()
    e = z.copy(); e[5] = 7.0                                 # single spike: scale 1, code 7
    c, s = orc.quantize_int4_g16(e)
    assert float(s[0]) == 1.0 and c[5] == 7 and c.sum() == 7
    e = z.copy(); e[:7] = [3.5, 1.25, 1.75, -0.25, -0.75, 0.74, -3.5]   # scale 0.5; ties to even
    c, s = orc.quantize_int4_g16(e)
    assert float(s[0]) == 0.5
    assert list(c[:7]) == [7, 2, 4, 0, -2, 1, -7]            # 2.5->2, 3.5->4, -0.5->-0, -1.5->-2, 1.48->1
    e = z.copy(); e[0] = 7 * 2.0 ** -20; e[1] = -3 * 2.0 ** -20        # fp16-subnormal scale 2^-20
    c, s = orc.quantize_int4_g16(e)
    assert float(s[0]) == 2.0 ** -20 and c[0] == 7 and c[1] == -3
    e = z.copy(); e[0] = 7 * 2.0 ** -26                       # scale rounds to fp16 zero -> all codes 0
    c, s = orc.quantize_int4_g16(e)
    assert float(s[0]) == 0.0 and not c.any()
    e = z.copy(); e[0] = 1e6; e[1] = -2e5                     # saturated scale 65504; clamp acts
    c, s = orc.quantize_int4_g16(e)
    assert float(s[0]) == 65504.0 and c[0] == 7 and c[1] == -3   # -2e5/65504 = -3.05
    e = np.concatenate([np.full(16, 0.07, np.float32), np.full(16, -14.0, np.float32)])   # two groups
    c, s = orc.quantize_int4_g16(e)
    assert float(s[1]) == 2.0 and (c[16:] == -7).all() and (c[:16] == 7).all()
    # dequant: code * scale, -8 decodes as -8*s
    dq = orc.dequant_int4_g16(np.array([-8] + [1] * 15, np.int8), np.array([0.25], np.float16))
    assert dq[0] == -2.0 and dq[1] == 0.25
    # round trip error bound |e - deq| <= s/2 in the normal range
    rng = np.random.default_rng(10)
    e = (rng.standard_normal((200, 64)) * 0.05).astype(np.float32)
    c, s = orc.quantize_int4_g16(e)
    err = np.abs(orc.dequant_int4_g16(c, s) - e).reshape(200, 4, 16)
    assert np.all(err <= s.astype(np.float32)[..., None] * 0.5 * (1 + 1e-3)) and np.abs(c).max() == 7


# P12 ------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("gain", [8.0, 64.0])
def test_p12_peaked_scores_match_sdpa(gain):
    rng = np.random.default_rng(12)
    oc, _ = small_cache(rng, T=70)
    q = rng.standard_normal((oc.H * oc.G, oc.d)) * gain
    for h in range(oc.H):
        K, V = oc.khat_vhat(0, 1, h)
        ref = sdpa64(q[h * oc.G:(h + 1) * oc.G], K, V, oc.scale)
        np.testing.assert_allclose(oc.decode_attention(1, 0, q)[h * oc.G:(h + 1) * oc.G], ref, rtol=1e-10, atol=1e-13)


# P13 ------------------------------------------------------------------------------------------------------
def test_p13_footprint_closed_form_matches_paper_ratio():
    """BASELINE.json configs[2] mix: 62.4 B per (layer, head, token) vs 512 B dense bf16 -> 8.205x (paper: 8.3x)."""
    wl = gen.WORKLOADS["llama8b_64k_b1"]
    tier, flag = gen.make_routing(wl, 0)
    fp = orc.footprint_bytes(tier, flag, wl.tier_ranks, wl.d, wl.L, wl.H_kv)
    per = fp / (wl.L * wl.H_kv * len(tier))
    assert abs(per - 62.4) < 0.01
    dense = 2 * wl.d * 2
    assert abs(dense / per - 8.205) < 0.01
    assert abs(dense / per - 8.3) / 8.3 < 0.02          # within 2 % of the paper's headline ratio
    wl = gen.WORKLOADS["tiny"]
    tier, flag = gen.make_routing(wl, 0)
    per = orc.footprint_bytes(tier, flag, wl.tier_ranks, wl.d, 1, 1) / len(tier)
    assert abs(per - 49.6) < 0.3


# routing, bf16 rounding, append/compress ------------------------------------------------------------------
def test_route_slots_counts_earlier_tokens():
    tier = np.array([1, 0, 1, 1, 0, 1], np.uint8); flag = np.array([1, 0, 0, 1, 0, 1], np.uint8)
    cls, slot, counts = orc.route_slots(tier, flag, 2)
    assert list(cls) == [3, 0, 2, 3, 0, 3] and list(slot) == [0, 0, 0, 1, 1, 2] and list(counts) == [2, 0, 1, 3]
    cls2, slot2, counts2 = orc.route_slots([0, 1], [0, 1], 2, counts)
    assert list(slot2) == [2, 3] and list(counts2) == [3, 0, 1, 4]


def test_round_to_bf16_matches_torch_and_breaks_double_rounding():
    rng = np.random.default_rng(0)
    x = rng.standard_normal(20000) * np.exp(rng.uniform(-20, 20, 20000))
    x32 = x.astype(np.float32).astype(np.float64)      # fp32-representable: torch's float->bf16 is a single rounding
    ref = torch.tensor(x32, dtype=torch.float32).to(torch.bfloat16).to(torch.float64).numpy()
    np.testing.assert_array_equal(orc.round_to_bf16(x32), ref)
    # a value just above a bf16 tie that fp32 rounding would push onto the tie (-> even): direct rounding goes up
    y = 1.0 + 2.0 ** -8 + 2.0 ** -40
    assert orc.round_to_bf16(np.array([y]))[0] == 1.0 + 2.0 ** -7
    assert orc.round_to_bf16(np.array([1.0 + 2.0 ** -8]))[0] == 1.0           # exact tie -> even


def test_append_compress_identity_round_trip_and_projector():
    """PAPER.md:56 'projecting the original cache vector onto the current basis': with B = I (r = d) and unit gates the
    coefficients are the (bf16) input itself and the residual is zero; with orthonormal rows, compress(reconstruct)
    of an in-span vector returns its coefficients; the residual is orthogonal to the leading rows."""
    rng = np.random.default_rng(11)
    d = 32
    I = np.broadcast_to(np.eye(d), (1, 1, d, d)).copy()
    oc = orc.OracleCache(1, 1, 1, 1, d, (d,), I, I, np.ones((1, 1, d)), np.ones((1, 1, d)))
    x = orc.round_to_bf16(rng.standard_normal((5, 1, 1, d)))
    oc.append_compress(0, x, -x, np.zeros(5, np.uint8), np.ones(5, np.uint8))
    np.testing.assert_array_equal(oc.seqs[0]["cK"], x)
    assert not oc.seqs[0]["codeK"].any()
    K, V = oc.khat_vhat(0, 0, 0)
    np.testing.assert_array_equal(K, x[:, 0, 0]); np.testing.assert_array_equal(V, -x[:, 0, 0])
    # general basis + gates: residual before quantisation is orthogonal (in gate-normalised space) up to bf16 rounding of c
    r = 8
    B = np.linalg.qr(rng.standard_normal((d, r)))[0].T[None, None]
    g = rng.uniform(0.5, 1.5, (1, 1, d))
    oc = orc.OracleCache(1, 1, 1, 1, d, (4, r), B, B, g, g)
    c_true = orc.round_to_bf16(rng.standard_normal((3, r)))
    x = (g[0, 0] * (c_true @ B[0, 0]))[:, None, None, :]
    oc.append_compress(0, x, x, np.array([1, 1, 0], np.uint8), np.zeros(3, np.uint8))
    np.testing.assert_allclose(oc.seqs[0]["cK"][:2, 0, 0], c_true[:2], rtol=0, atol=1e-12)   # in-span: exact coefficients
    np.testing.assert_allclose(oc.seqs[0]["cK"][2, 0, 0, :4], c_true[2, :4], rtol=0, atol=1e-12)
    assert not oc.seqs[0]["cK"][2, 0, 0, 4:].any()
    K, _ = oc.khat_vhat(0, 0, 0)
    np.testing.assert_allclose(K[:2], x[:2, 0, 0], rtol=0, atol=1e-12)


def test_generated_tiny_workload_statistics():
    """The seeded tiny workload has the shapes / mixes BASELINE.json configs[0] states."""
    wl = gen.WORKLOADS["tiny"]
    inp = workload_inputs(wl)
    assert inp["cK"].shape == (512, 2, 2, 16) and inp["cK"].dtype == torch.bfloat16
    assert (inp["tier"][:32] == 1).all() and abs((inp["tier"] == 1).mean() - 0.3) < 0.01
    assert abs(inp["flag"].mean() - 0.1) < 0.01 and not (inp["flag"] & (inp["tier"] == 0)).any()
    assert not inp["cK"][torch.as_tensor(inp["tier"] == 0)][..., 8:].any()
    BK, BV = gen.make_basis(wl)
    Bf = BK.double()
    eye = torch.einsum("mhrd,mhsd->mhrs", Bf, Bf)
    assert (eye - torch.eye(16)).abs().max() < 0.02       # orthonormal up to bf16 rounding
    oc, _ = make_oracle(wl)
    oracle_load(oc, 0, inp)
    q = f64(gen.make_q(wl))[0]
    o = oc.decode_all_layers([0], q[None])
    assert np.isfinite(o).all() and o.shape == (1, 2, 4, 64)


def test_probe_error_eq3_closed_forms():
    """Eq. (3): hand values. ref = (3, 4) on one head, cmp = 0 -> 5 / (5 + eps); identical outputs -> 0; a
    uniformly scaled output (1 + delta) * ref -> delta * |ref| / (|ref| + eps); heads of different kv heads do not mix."""
    ref = np.zeros((1, 2, 2)); ref[0, 0] = [3.0, 4.0]; ref[0, 1] = [0.0, 12.0]
    cmp_ = np.zeros_like(ref); cmp_[0, 1] = [0.0, 12.0]
    e = orc.probe_error(ref, cmp_, G=1, eps=1.0)
    assert np.allclose(e, [5.0 / 6.0, 0.0])
    e2 = orc.probe_error(ref, cmp_, G=2, eps=0.0)                       # one kv head over both query heads
    assert np.allclose(e2, [5.0 / 13.0])
    rng = np.random.default_rng(0)
    a = rng.standard_normal((3, 4, 8))
    assert np.allclose(orc.probe_error(a, a, 2, 1e-6), 0.0)
    e3 = orc.probe_error(a, 1.25 * a, 2, 0.5)
    for h in range(2):
        nrm = np.linalg.norm(a[:, 2 * h:2 * h + 2])
        assert np.isclose(e3[h], 0.25 * nrm / (nrm + 0.5))
