"""Re-tiering of stored tokens (dwkv_retier_seq; reading A29): lowering a token's tier keeps the leading
coefficients of its stored vector, clearing its flag drops the int4 residual.

CPU part: pins of OracleCache.retier against things that do not go through it -- a fresh append at the lower tier (the coefficient
vector is nested: bit-identical), a closed form for the change of K-hat written out in the test, brute-force slot numbering.
GPU part: the library against the oracle, bit for bit on the stored bytes, within the north-star tolerance on the attention output."""
import dataclasses

import numpy as np
import pytest
import torch

import gen
from oracle import dwkv_oracle as orc
from helpers import f64, check_output


def _small(seed=0, L=4, w=2, H=2, d=32, ranks=(8, 16, 24)):
    rng = np.random.default_rng(seed)
    r = ranks[-1]
    B = {z: orc.round_to_bf16(rng.standard_normal((L // w, H, r, d)) / np.sqrt(d)) for z in "KV"}
    g = {z: orc.round_to_bf16(rng.uniform(0.5, 1.5, (L, H, d))) for z in "KV"}
    return rng, orc.OracleCache(L, w, H, 2, d, ranks, B["K"], B["V"], g["K"], g["V"]), B, g


# ---- CPU pins ----------------------------------------------------------------------------------------------------------
def test_retier_equals_fresh_append_at_the_lower_tier():
    """Unflagged tokens: the stored coefficients after lowering are bit-identical to what append_compress stores at that tier."""
    rng, oc, B, g = _small()
    n = 23
    x = {z: orc.round_to_bf16(rng.standard_normal((n, oc.L, oc.H, oc.d))) for z in "KV"}
    tier = rng.integers(1, 3, n).astype(np.uint8)
    oc.append_compress(0, x["K"], x["V"], tier, np.zeros(n, np.uint8))
    lower = (tier - rng.integers(0, 2, n)).astype(np.uint8)
    oc.retier(0, lower, np.zeros(n, np.uint8))
    fresh = orc.OracleCache(oc.L, oc.w, oc.H, oc.G, oc.d, oc.tier_ranks, B["K"], B["V"], g["K"], g["V"])
    fresh.append_compress(0, x["K"], x["V"], lower, np.zeros(n, np.uint8))
    for key in ("tier", "flag", "cls", "slot", "cK", "cV"):
        assert np.array_equal(oc.seqs[0][key], fresh.seqs[0][key]), key
    for l in range(oc.L):
        for h in range(oc.H):
            for a, b in zip(oc.khat_vhat(0, l, h), fresh.khat_vhat(0, l, h)):
                assert np.array_equal(a, b)


def test_retier_closed_form_slots_and_errors():
    rng, oc, B, g = _small(seed=1)
    n = 40
    x = {z: orc.round_to_bf16(rng.standard_normal((n, oc.L, oc.H, oc.d))) for z in "KV"}
    tier = rng.integers(0, 3, n).astype(np.uint8)
    flag = (rng.random(n) < 0.5).astype(np.uint8)
    oc.append_compress(0, x["K"], x["V"], tier, flag)
    before = {(l, h): oc.khat_vhat(0, l, h) for l in range(oc.L) for h in range(oc.H)}
    S = oc.seqs[0]
    cK, cV = S["cK"].copy(), S["cV"].copy()
    deq = {z: orc.dequant_int4_g16(S["code" + z], S["scale" + z]) for z in "KV"}
    # identity
    oc.retier(0, tier, flag)
    for (l, h), (K, V) in before.items():
        K2, V2 = oc.khat_vhat(0, l, h)
        assert np.array_equal(K, K2) and np.array_equal(V, V2)
    new_tier = np.minimum(tier, rng.integers(0, 3, n)).astype(np.uint8)
    new_flag = (flag & (rng.random(n) < 0.5)).astype(np.uint8)
    oc.retier(0, new_tier, new_flag)
    ranks_old, ranks_new = np.asarray(oc.tier_ranks)[tier], np.asarray(oc.tier_ranks)[new_tier]
    for (l, h), (K, V) in before.items():
        K2, V2 = oc.khat_vhat(0, l, h)
        for z, old, new, c, Ball, gate in (("K", K, K2, cK, oc.BK, oc.gK), ("V", V, V2, cV, oc.BV, oc.gV)):
            for t in range(n):
                # X-hat_new = X-hat_old - gate * (c[r':r] . B[r':r]) - (residual if its flag was cleared), written out
                drop = c[t, l, h, ranks_new[t]:ranks_old[t]] @ Ball[l // oc.w, h, ranks_new[t]:ranks_old[t]]
                want = old[t] - gate[l, h] * drop - (deq[z][t, l, h] if flag[t] and not new_flag[t] else 0.0)
                np.testing.assert_allclose(new[t], want, rtol=0, atol=1e-12)
    cnt = {}
    for t in range(n):                                   # slots: earlier tokens of the same NEW class, by brute force
        k = 2 * int(new_tier[t]) + int(new_flag[t])
        assert S["cls"][t] == k and S["slot"][t] == cnt.get(k, 0)
        cnt[k] = cnt.get(k, 0) + 1
    assert oc.footprint_bytes(0) == orc.footprint_bytes(new_tier, new_flag, oc.tier_ranks, oc.d, oc.L, oc.H)
    with pytest.raises(AssertionError):
        oc.retier(0, np.minimum(new_tier + 1, 2).astype(np.uint8), new_flag)        # a raised tier
    with pytest.raises(AssertionError):
        oc.retier(0, new_tier, np.ones(n, np.uint8))                                  # a raised flag


def test_retier_then_append_continues_the_slots_and_decode_matches_loop_built_attention():
    rng, oc, B, g = _small(seed=2)
    n = 30
    x = {z: orc.round_to_bf16(rng.standard_normal((n + 7, oc.L, oc.H, oc.d))) for z in "KV"}
    tier = rng.integers(0, 3, n + 7).astype(np.uint8)
    flag = (rng.random(n + 7) < 0.4).astype(np.uint8)
    oc.append_compress(0, x["K"][:n], x["V"][:n], tier[:n], flag[:n])
    nt = np.minimum(tier[:n], 1).astype(np.uint8); nf = np.zeros(n, np.uint8)
    oc.retier(0, nt, nf)
    oc.append_compress(0, x["K"][n:], x["V"][n:], tier[n:], flag[n:])
    S = oc.seqs[0]
    all_t, all_f = np.concatenate([nt, tier[n:]]), np.concatenate([nf, flag[n:]])
    cnt = {}
    for t in range(n + 7):
        k = 2 * int(all_t[t]) + int(all_f[t])
        assert S["slot"][t] == cnt.get(k, 0)
        cnt[k] = cnt.get(k, 0) + 1
    q = rng.standard_normal((oc.H * oc.G, oc.d))
    l = 3
    out = oc.decode_attention(l, 0, q)
    for h in range(oc.H):
        K, V = oc.khat_vhat(0, l, h)
        for gq in range(oc.G):
            s = (K @ q[h * oc.G + gq]) * oc.scale
            p = np.exp(s - s.max()); p /= p.sum()
            np.testing.assert_allclose(out[h * oc.G + gq], p @ V, rtol=1e-12, atol=1e-14)


# ---- GPU: the library against the oracle -------------------------------------------------------------------------------
@pytest.fixture(scope="module")
def mod():
    from paper_2607_06523_b200 import binding, harness
    return binding, harness


def _decode_codes(gc, shape):
    lo = (gc & 15).astype(np.int8); hi = (gc >> 4).astype(np.int8)
    lo = np.where(lo > 7, lo - 16, lo); hi = np.where(hi > 7, hi - 16, hi)
    return np.stack([lo, hi], axis=-1).reshape(shape)


@pytest.mark.gpu
@pytest.mark.parametrize("name", ["tiny", "g8_r48"])
def test_gpu_retier_against_oracle(mod, name):
    from test_gpu_parity import load
    from test_gpu_controller import oracle_from_kept
    binding, harness = mod
    if name == "tiny":
        wl = dataclasses.replace(gen.WORKLOADS["tiny"], T=(300, 1, 97), patterns=("", "all_top_flag", "alternating"))
    else:
        wl = dataclasses.replace(gen.WORKLOADS["llama70b_128k_b1"], L=4, T=(700,))
    routings = [gen.make_routing(wl, s) for s in range(wl.n_seq)]
    cache, consts, kept = load(harness, wl, routings, chunk=256)
    oc = oracle_from_kept(wl, consts, routings, kept)
    rng = np.random.default_rng(5)
    used0 = cache.footprint()["used_bytes"]
    q0 = gen.make_q(wl, device="cuda")
    for s, (tier, flag) in enumerate(routings):       # a probe before the move: the device-resident token table now holds the old places
        m = torch.zeros(len(tier), dtype=torch.float32, device="cuda"); sp = torch.zeros_like(m)
        cache.probe_token_stats(0, s, q0[s, 0].contiguous(), m, sp)
    for s, (tier, flag) in enumerate(routings):
        nt = np.minimum(tier, rng.integers(0, len(wl.tier_ranks), len(tier))).astype(np.uint8)
        nf = (flag & (rng.random(len(flag)) < 0.5)).astype(np.uint8)
        cache.retier_seq(s, nt, nf)
        oc.retier(s, nt, nf)
        T = len(tier)
        dump = cache.export_tokens(s, 0, T)
        S = oc.seqs[s]
        assert np.array_equal(dump["tier"].cpu().numpy(), S["tier"]) and np.array_equal(dump["flag"].cpu().numpy(), S["flag"])
        assert np.array_equal(dump["slot"].cpu().numpy(), S["slot"])
        for z in "KV":
            assert np.array_equal(dump["coef" + z].double().cpu().numpy(), S["c" + z]), (s, z)           # truncated, bit-exact
            assert np.array_equal(_decode_codes(dump["code" + z].cpu().numpy(), S["code" + z].shape), S["code" + z]), (s, z)
            assert np.array_equal(dump["scale" + z].cpu().numpy().view(np.uint16), S["scale" + z].view(np.uint16)), (s, z)
    fp = cache.footprint()
    assert fp["used_bytes"] == sum(oc.footprint_bytes(s) for s in range(wl.n_seq)) < used0
    ids = list(range(wl.n_seq))
    q = gen.make_q(wl, device="cuda")
    out = cache.decode_attention(-1, ids, q).double().cpu().numpy()
    ref = oc.decode_all_layers(ids, f64(q))
    for s in ids:
        for l in range(wl.L):
            check_output(out[s, l], ref[s, l], oc.max_abs_vhat(s, l), f"retier {name} seq {s} layer {l}")
    from test_gpu_controller import oracle_stats
    for s, (tier, flag) in enumerate(routings):       # ... and after it the table is rebuilt: statistics of the moved records
        m = torch.zeros(len(tier), dtype=torch.float32, device="cuda"); sp = torch.zeros_like(m)
        cache.probe_token_stats(wl.L - 1, s, q0[s, wl.L - 1].contiguous(), m, sp)
        m_o, sp_o = oracle_stats(oc, wl, s, wl.L - 1, f64(q0[s, wl.L - 1]))
        np.testing.assert_allclose(m.double().cpu().numpy(), m_o, rtol=3e-3, atol=1e-7)
        np.testing.assert_allclose(sp.double().cpu().numpy(), sp_o, rtol=3e-3, atol=1e-7)
    # a raised tier is refused and changes nothing; an identity call is a no-op
    tier0 = oc.seqs[0]["tier"].copy()
    if tier0.min() < len(wl.tier_ranks) - 1:
        bad = tier0.copy(); bad[int(np.argmin(tier0))] += 1
        with pytest.raises(binding.DwkvError):
            cache.retier_seq(0, bad, oc.seqs[0]["flag"])
    cache.retier_seq(0, tier0, oc.seqs[0]["flag"])
    out2 = cache.decode_attention(-1, ids, q).double().cpu().numpy()
    assert np.array_equal(out, out2)
    cache.destroy()


@pytest.mark.gpu
def test_gpu_retier_8bit_planes_equal_a_fresh_load(mod):
    """8-bit coefficient planes: re-tiering re-blocks the stored codes exactly, so the cache equals one loaded afresh with the same
    (already 8-bit representable) coefficients at the lower tiers: outputs bit-identical."""
    from test_gpu_coef8 import load8
    binding, harness = mod
    wl = dataclasses.replace(gen.WORKLOADS["tiny"], T=(257,))
    tier, flag = gen.make_routing(wl, 0)
    cache, consts, kept = load8(harness, wl, [(tier, flag)])
    rng = np.random.default_rng(7)
    nt = np.minimum(tier, rng.integers(0, len(wl.tier_ranks), len(tier))).astype(np.uint8)
    nf = (flag & (rng.random(len(flag)) < 0.5)).astype(np.uint8)
    T = len(tier)
    d0 = cache.export_tokens(0, 0, T)                     # dequantised coefficients (code * 2^e, exact in bf16), codes, scales
    cache.retier_seq(0, nt, nf)
    q = gen.make_q(wl, device="cuda")
    out = cache.decode_attention(-1, [0], q).clone()
    fresh, _ = harness.make_cache(wl, n_seqs=1, max_tokens=512, coef_int8=True)
    idx = torch.tensor(np.nonzero(nf)[0], device="cuda")
    fresh.append_raw(0, nt, nf, d0["coefK"], d0["coefV"],
                     codeK=d0["codeK"][idx].contiguous(), codeV=d0["codeV"][idx].contiguous(),
                     scaleK=d0["scaleK"][idx].contiguous(), scaleV=d0["scaleV"][idx].contiguous())
    out_f = fresh.decode_attention(-1, [0], q)
    assert torch.equal(out, out_f)
    assert cache.footprint()["used_bytes"] == fresh.footprint()["used_bytes"]
    cache.destroy(); fresh.destroy()


@pytest.mark.gpu
def test_gpu_budget_driven_retier_through_the_router(mod):
    """The budget loop of PAPER.md:63 on stored tokens: the router's budget-seeking thresholds (dwkv_router_thresholds) are tightened
    from the workload's tier mix to a leaner one, every stored token is re-routed with its features and LOWERED where the new
    routing is lower (tokens the new routing would raise keep their class: raising is impossible), the cache is re-tiered, and its
    footprint is the closed form of the new classes; routing bit-exact against the router oracle, attention against the oracle."""
    from test_gpu_parity import load
    from test_gpu_controller import oracle_from_kept
    from oracle import dwkv_router_oracle as ro
    binding, harness = mod
    wl = dataclasses.replace(gen.WORKLOADS["tiny"], T=(400,))
    tier, flag = gen.make_routing(wl, 0)
    cache, consts, kept = load(harness, wl, [(tier, flag)], chunk=256)
    oc = oracle_from_kept(wl, consts, [(tier, flag)], kept)
    rng = np.random.default_rng(11)
    T = len(tier)
    phi = rng.random((T, 4)).astype(np.float32)                      # stand-ins for the four features of Eq. (2)
    u = np.array([2.0, 1.5, 0.5, 1.0], np.float32)
    lean = [0.9, 0.1]                                                # budget: 90 % of the tokens at the lowest rank, 2 % flagged
    tau, tf = binding.router_thresholds(phi, u, lean, 0.02)
    tau_o, tf_o = ro.thresholds(phi, u, lean, 0.02)
    assert np.array_equal(np.asarray(tau, np.float32), np.asarray(tau_o, np.float32)) and np.float32(tf) == np.float32(tf_o)
    rt, rf = binding.route_tokens(phi, u, tau, tf, len(wl.tier_ranks))
    rt_o, rf_o = ro.route(phi, u, tau_o, tf_o)
    assert np.array_equal(rt, rt_o) and np.array_equal(rf, rf_o)
    nt, nf = np.minimum(tier, rt).astype(np.uint8), (flag & rf).astype(np.uint8)
    before = cache.footprint()["used_bytes"]
    cache.retier_seq(0, nt, nf)
    oc.retier(0, nt, nf)
    after = cache.footprint()["used_bytes"]
    assert after == orc.footprint_bytes(nt, nf, wl.tier_ranks, wl.d, wl.L, wl.H_kv) < before
    q = gen.make_q(wl, device="cuda")
    out = cache.decode_attention(-1, [0], q).double().cpu().numpy()
    ref = oc.decode_all_layers([0], f64(q))
    for l in range(wl.L):
        check_output(out[0, l], ref[0, l], oc.max_abs_vhat(0, l), f"budget retier layer {l}")
    cache.destroy()
