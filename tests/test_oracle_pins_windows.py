"""Pins for the two parts of the oracle that single-window / zero-residual cases cannot see (round-1 verdict): the depth-window
lookup m(l) = l // w (reading A1) in reconstruction AND in append/compress, and the residual arithmetic of
append/compress  e = x - g * (c_bf16 . B[:r_t])  (readings A13 / A14). CPU only.

  P14  hand-derived append case, expected values in tests/golden/append_hand_case.txt (two windows with different bases,
       non-unit gates, an out-of-span x, flag = 1, a coefficient that needs 10 significant bits)
  P15  >= 2 depth windows holding different bases: dense K-hat / V-hat built by the test's own loops that index B[l // w],
       SDPA in float64 as the independent attention routine
  P16  append/compress on a multi-window cache against the test's own loop (torch's bf16 rounding, own residual and quantiser),
       plus the property |x - X-hat| <= scale / 2 per group on flagged tokens
"""
import math
import os

import numpy as np
import torch

from oracle import dwkv_oracle as orc
from test_oracle_pins import sdpa64

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "append_hand_case.txt")


def _hand_case_constants():
    d, L, M = 16, 2, 2
    BK = np.zeros((M, 1, 2, d)); BV = np.zeros((M, 1, 2, d))
    for m in range(M):
        BK[m, 0, 0, 4 * m:4 * m + 4] = 0.5
        BK[m, 0, 1, 4 * m:4 * m + 4] = [0.5, -0.5, 0.5, -0.5]
    BV[0, 0, 0, 15] = 1.0; BV[0, 0, 1, 14] = 1.0
    BV[1, 0, 0, 0] = 1.0; BV[1, 0, 1, 1] = 1.0
    gK = np.ones((L, 1, d)); gK[0, 0, :4] = [2, 0.5, 4, 1]; gK[1, 0, 4:8] = [4, 2, 0.5, 1]
    gV = np.ones((L, 1, d)); gV[0] = 2.0; gV[1] = 0.5
    return d, L, BK, BV, gK, gV


def test_p14_hand_derived_append_case():
    d, L, BK, BV, gK, gV = _hand_case_constants()
    x = {z: np.zeros((2, L, 1, d)) for z in "KV"}
    c = {z: np.zeros((2, L, 1, 2)) for z in "KV"}
    code = {z: np.zeros((2, L, 1, d), np.int64) for z in "KV"}
    scale = {z: np.zeros((2, L, 1, 1)) for z in "KV"}
    hat = {z: np.zeros((2, L, d)) for z in "KV"}
    n_lines = 0
    for line in open(GOLDEN):
        f = line.split()
        if not f or f[0].startswith("#"):
            continue
        n_lines += 1
        kind, z, t, l = f[0], f[1], int(f[2]), int(f[3])
        if kind == "x":
            x[z][t, l, 0, int(f[4])] = float(f[5])
        elif kind == "c":
            c[z][t, l, 0, int(f[4])] = float(f[5])
        elif kind == "code":
            code[z][t, l, 0, int(f[4])] = int(f[5])
        elif kind == "scale":
            scale[z][t, l, 0, 0] = float(f[4])
        elif kind == "hat":
            hat[z][t, l, int(f[4])] = float(f[5])
        else:
            raise AssertionError(line)
    assert n_lines == 29 + 12 + 4 + 8 + 27
    oc = orc.OracleCache(L, 1, 1, 1, d, (1, 2), BK, BV, gK, gV)
    oc.append_compress(0, x["K"], x["V"], np.array([1, 0], np.uint8), np.array([1, 0], np.uint8))
    S = oc.seqs[0]
    for z in "KV":
        np.testing.assert_array_equal(S["c" + z], c[z])                      # rounded coefficients, leading r_t only
        np.testing.assert_array_equal(S["code" + z].astype(np.int64), code[z])
        np.testing.assert_array_equal(S["scale" + z].astype(np.float64), scale[z])
    for l in range(L):
        K, V = oc.khat_vhat(0, l, 0)
        np.testing.assert_array_equal(K, hat["K"][:, l])
        np.testing.assert_array_equal(V, hat["V"][:, l])
    assert list(S["cls"]) == [3, 0] and list(S["slot"]) == [0, 0]


def _multi_window_cache(rng, T, L=4, w=2, H=2, G=2, d=32, ranks=(8, 16)):
    r, M = ranks[-1], L // w
    BK = np.stack([[np.linalg.qr(rng.standard_normal((d, r)))[0].T for _ in range(H)] for _ in range(M)])
    BV = np.stack([[np.linalg.qr(rng.standard_normal((d, r)))[0].T for _ in range(H)] for _ in range(M)])
    assert np.abs(BK[0] - BK[1]).max() > 0.1          # the windows really hold different bases
    gK = rng.uniform(0.5, 1.5, (L, H, d)); gV = rng.uniform(0.5, 1.5, (L, H, d))
    tier = rng.integers(0, len(ranks), T).astype(np.uint8)
    flag = (rng.random(T) < 0.4).astype(np.uint8)
    flag[0] = 1
    return orc.OracleCache(L, w, H, G, d, ranks, BK, BV, gK, gV), dict(BK=BK, BV=BV, gK=gK, gV=gV, tier=tier, flag=flag)


def _quant_group_loop(e32):
    """The test's own int4 / group-16 quantiser (reading A14) on one fp32 vector; returns dequantised float64 values and scales."""
    out = np.zeros(len(e32)); scales = []
    for g0 in range(0, len(e32), 16):
        grp = e32[g0:g0 + 16]
        s = np.float16(min(np.float32(np.max(np.abs(grp))) / np.float32(7), np.float32(65504)))
        scales.append(float(s))
        if float(s) != 0.0:
            out[g0:g0 + 16] = np.clip(np.rint(grp / np.float32(s)), -7, 7).astype(np.float64) * float(s)
    return out, scales


def test_p15_two_windows_decode_against_loop_built_dense_cache():
    rng = np.random.default_rng(15)
    T = 29
    oc, x = _multi_window_cache(rng, T)
    r = oc.r
    cK = rng.standard_normal((T, oc.L, oc.H, r)); cV = rng.standard_normal((T, oc.L, oc.H, r))
    nf = int(x["flag"].sum())
    rK = (rng.standard_normal((nf, oc.L, oc.H, oc.d)) * 0.05).astype(np.float32)
    rV = (rng.standard_normal((nf, oc.L, oc.H, oc.d)) * 0.05).astype(np.float32)
    oc.append_raw(0, x["tier"], x["flag"], cK, cV, residK=rK, residV=rV)
    ranks = np.asarray(oc.tier_ranks)[x["tier"]]
    fidx = np.cumsum(x["flag"]) - 1
    q = rng.standard_normal((oc.H * oc.G, oc.d)) * 2
    for l in range(oc.L):
        o = oc.decode_attention(l, 0, q)
        m = l // 2                                                     # the test's own window index (w = 2)
        for h in range(oc.H):
            K = np.zeros((T, oc.d)); V = np.zeros((T, oc.d))
            for t in range(T):
                for j in range(ranks[t]):
                    K[t] += cK[t, l, h, j] * x["BK"][m, h, j]
                    V[t] += cV[t, l, h, j] * x["BV"][m, h, j]
                K[t] *= x["gK"][l, h]; V[t] *= x["gV"][l, h]
                if x["flag"][t]:
                    K[t] += _quant_group_loop(rK[fidx[t], l, h])[0]
                    V[t] += _quant_group_loop(rV[fidx[t], l, h])[0]
            ref = sdpa64(q[h * oc.G:(h + 1) * oc.G], K, V, 1.0 / math.sqrt(oc.d))
            np.testing.assert_allclose(o[h * oc.G:(h + 1) * oc.G], ref, rtol=1e-11, atol=1e-13)
    # and the outputs of the layers of different windows really differ when fed the same coefficients
    oc2, _ = _multi_window_cache(np.random.default_rng(15), T)
    same = np.broadcast_to(cK[:, :1], cK.shape).copy()
    oc2.append_raw(0, x["tier"], np.zeros(T, np.uint8), same, same)
    oc2.gK[:] = 1.0; oc2.gV[:] = 1.0
    assert np.abs(oc2.decode_attention(0, 0, q) - oc2.decode_attention(1, 0, q)).max() < 1e-12      # same window
    assert np.abs(oc2.decode_attention(0, 0, q) - oc2.decode_attention(2, 0, q)).max() > 1e-3       # other window


def test_p16_two_windows_append_compress_against_own_loop():
    rng = np.random.default_rng(16)
    T = 11
    oc, x = _multi_window_cache(rng, T)
    L, H, d = oc.L, oc.H, oc.d
    bf = lambda a: torch.tensor(a, dtype=torch.float64).to(torch.bfloat16).to(torch.float64).numpy()
    k_new = bf(rng.standard_normal((T, L, H, d))); v_new = bf(rng.standard_normal((T, L, H, d)))
    oc.append_compress(0, k_new, v_new, x["tier"], x["flag"])
    S = oc.seqs[0]
    ranks = np.asarray(oc.tier_ranks)[x["tier"]]
    for z, X, Ball, gall in (("K", k_new, x["BK"], x["gK"]), ("V", v_new, x["BV"], x["gV"])):
        for t in range(T):
            for l in range(L):
                for h in range(H):
                    B = Ball[l // 2, h][:ranks[t]]                      # own window index, leading r_t rows
                    g = gall[l, h]
                    c = np.zeros(oc.r)
                    c[:ranks[t]] = bf(np.array([float(np.dot(B[j], X[t, l, h] / g)) for j in range(ranks[t])]))
                    np.testing.assert_array_equal(S["c" + z][t, l, h], c)
                    rec = np.zeros(d)
                    for j in range(ranks[t]):
                        rec += c[j] * B[j]
                    hat = g * rec
                    got = orc.reconstruct(S["c" + z][t:t + 1, l, h], ranks[t:t + 1], x["flag"][t:t + 1],
                                          orc.dequant_int4_g16(S["code" + z][t:t + 1, l, h], S["scale" + z][t:t + 1, l, h]), Ball[l // 2, h], g)[0]
                    if x["flag"][t]:
                        e32 = (X[t, l, h] - hat).astype(np.float32)       # residual against the ROUNDED coefficients, gate applied
                        deq, scales = _quant_group_loop(e32)
                        np.testing.assert_array_equal(S["scale" + z][t, l, h].astype(np.float64), scales)
                        np.testing.assert_allclose(got, hat + deq, rtol=0, atol=1e-13)
                        err = np.abs(X[t, l, h] - got).reshape(-1, 16)
                        assert np.all(err <= np.asarray(scales)[:, None] * 0.5 * (1 + 1e-3) + 1e-12)     # |x - X-hat| <= scale / 2
                        assert np.abs(e32).max() > 0.05                   # x is far out of span: the residual matters
                    else:
                        np.testing.assert_allclose(got, hat, rtol=0, atol=1e-13)
                        assert not S["code" + z][t, l, h].any()
