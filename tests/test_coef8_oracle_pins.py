"""Pins for the 8-bit blockwise coefficient oracle (reading A27). CPU only.

The paper prints no worked example of its coefficient quantiser, so the oracle is pinned to what the reading fixes: hand-derived
vectors, an exhaustive search for the block exponent, the error bound and exact-bf16 property the format implies, invariants
(idempotence, power-of-two covariance), the footprint closed form, and the projector property of append/compress.
"""
import numpy as np

import gen
from oracle import dwkv_coef8_oracle as c8
from oracle import dwkv_oracle as orc
from helpers import make_oracle, workload_inputs, f64, rel_l2


def q1(v):
    codes, exps = c8.quantize_coef_i8(np.asarray(v, np.float32))
    return codes.tolist(), exps.tolist()


def test_hand_vectors():
    # amax = 127 fits e = 0 exactly; 0.5 and 1.5 are ties -> even; 2.5 -> 2
    assert q1([127.0, -127.0, 1.0, 0.5, 1.5, 2.5, -0.5, 0.0]) == ([127, -127, 1, 0, 2, 2, 0, 0], [0])
    # amax = 128 > 127 * 2^0 -> e = 1, codes halve (63.5 -> 64 tie to even)
    assert q1([128.0, -127.0, 3.0, 1.0]) == ([64, -64, 2, 0], [1])
    # the next fp32 above 127 already needs e = 1
    assert q1([np.nextafter(np.float32(127.0), np.float32(200.0)), 2.0])[1] == [1]
    # negative exponent: amax = 127/4 -> e = -2
    assert q1([31.75, -0.25, 0.125]) == ([127, -1, 0], [-2])        # 0.125 / 0.25 = 0.5 -> tie to even -> 0
    # all-zero block: codes 0, e = E_MIN
    assert q1([0.0] * 8) == ([0] * 8, [c8.E_MIN])
    # amax below 127 * 2^E_MIN: exponent clamps, codes stay small (here rint(2^-126 / 2^-126) = 1)
    assert q1([2.0 ** -126, 0.0]) == ([1, 0], [c8.E_MIN])
    # two blocks (rank 48 = 32 + 16) get independent exponents
    v = np.zeros(48, np.float32); v[0] = 1000.0; v[5] = 8.0; v[32] = 0.01; v[47] = -0.005
    codes, exps = c8.quantize_coef_i8(v)
    assert exps.tolist() == [3, -13]                                 # 1000/127 = 7.87 -> 2^3 ; 0.01/127 = 7.87e-5 -> 2^-13 = 1.22e-4
    assert codes[0] == 125 and codes[5] == 1 and codes[32] == 82 and codes[47] == -41
    # leading-rank semantics: columns beyond `rank` neither enter amax nor get codes
    codes, exps = c8.quantize_coef_i8(np.array([1.0, 2.0, 3.0, 4.0, 1e6, 1e6, 1e6, 1e6], np.float32), rank=4)
    assert codes.tolist() == [16, 32, 48, 64, 0, 0, 0, 0]
    assert exps.tolist() == [-4]                                     # 127 * 2^-5 = 3.97 < 4 <= 127 * 2^-4: step 1/16


def test_exponent_is_the_smallest_that_fits_brute_force():
    rng = np.random.default_rng(1)
    amax = np.concatenate([np.exp(rng.uniform(-40, 40, 2000)), 127.0 * 2.0 ** np.arange(-20, 20), 128.0 * 2.0 ** np.arange(-20, 20),
                           np.nextafter(127.0 * 2.0 ** np.arange(-20, 20), np.inf)]).astype(np.float32).astype(np.float64)
    e = c8.block_exponent(amax)
    for a, ee in zip(amax, e):
        k = -200
        while a > 127.0 * 2.0 ** k:      # plain search with exact fp64 arithmetic
            k += 1
        assert ee == max(k, c8.E_MIN), (a, ee, k)


def test_error_bound_and_exact_bf16():
    rng = np.random.default_rng(2)
    for r in (8, 16, 32, 48, 64):
        c = (rng.standard_normal((500, r)) / np.sqrt(1.0 + np.arange(r))).astype(np.float32)
        codes, exps = c8.quantize_coef_i8(c)
        deq = c8.dequant_coef_i8(codes, exps)
        assert np.abs(codes.astype(int)).max() <= 127
        for b in range(exps.shape[-1]):
            sl = slice(32 * b, min(32 * b + 32, r))
            amax = np.abs(c[:, sl].astype(np.float64)).max(axis=-1)
            step = 2.0 ** exps[:, b].astype(np.float64)
            assert np.all(step * 127 >= amax) and np.all(step * 127 < 2 * amax)            # smallest exponent that fits
            err = np.abs(deq[:, sl] - c[:, sl].astype(np.float64)).max(axis=-1)
            assert np.all(err <= step / 2) and np.all(err <= amax / 127)                   # half a step < amax / 127
            assert np.all(np.abs(codes[:, sl].astype(int)).max(axis=-1) >= 64)             # the block uses its top bit
        assert np.array_equal(orc.round_to_bf16(deq), deq)                                 # <= 7 significant bits: a bf16 value


def test_idempotent_and_power_of_two_covariant():
    rng = np.random.default_rng(3)
    c = rng.standard_normal((200, 48)).astype(np.float32)
    codes, exps = c8.quantize_coef_i8(c)
    deq = c8.dequant_coef_i8(codes, exps)
    codes2, exps2 = c8.quantize_coef_i8(deq.astype(np.float32))
    # re-quantising the dequantised block reproduces the values (the exponent may drop if the top code was < 64 after rounding)
    assert np.array_equal(c8.dequant_coef_i8(codes2, exps2), deq)
    for k in (-9, 5):
        ck, ek = c8.quantize_coef_i8((c.astype(np.float64) * 2.0 ** k).astype(np.float32))
        assert np.array_equal(ck, codes) and np.array_equal(ek.astype(int), exps.astype(int) + k)
    # sign symmetry
    cn, en = c8.quantize_coef_i8(-c)
    assert np.array_equal(cn, -codes) and np.array_equal(en, exps)


def test_footprint_closed_form():
    # BJ:9 mix (65/25/10 % at ranks 8/16/32, residual on 8 %), d = 128: 2*(12.4 + 1) + 0.08*160 = 39.6 B per (l, h, token)
    # against 512 B dense -> 12.93x (bf16 coefficients: 62.4 B -> 8.205x, pin P13)
    T = 100000
    tier = np.zeros(T, np.uint8); tier[:25000] = 1; tier[25000:35000] = 2
    flag = np.zeros(T, np.uint8); flag[25000:33000] = 1
    b = c8.footprint_bytes_i8(tier, flag, (8, 16, 32), 128, 1, 1)
    assert b == int(round(39.6 * T))
    assert abs(512.0 * T / b - 12.929) < 1e-3
    # rank 48 has two blocks: 2*(48 + 2) = 100 B
    assert c8.footprint_bytes_i8(np.zeros(1, np.uint8), np.zeros(1, np.uint8), (48,), 128, 1, 1) == 100


def test_project_quantise_is_a_projector_up_to_the_quantisation_step():
    rng = np.random.default_rng(4)
    d, r = 64, 16
    B = np.linalg.qr(rng.standard_normal((d, r)))[0].T
    gate = rng.uniform(0.5, 1.5, d)
    c_true = rng.standard_normal(r) / np.sqrt(1.0 + np.arange(r))
    x = orc.round_to_bf16(gate * (c_true @ B))
    codes, exps, c, resid = c8.project_quantise(x, B, gate)
    step = 2.0 ** float(exps[0])
    assert np.abs(c - c_true).max() <= step / 2 + 2e-2 * np.abs(c_true).max()      # bf16 rounding of x on top of half a step
    # the residual is what the dequantised coefficients leave: x = gate * (c @ B) + resid to fp32 rounding
    assert np.abs(gate * (c @ B) + resid.astype(np.float64) - x).max() <= 2.0 ** -23 * np.abs(x).max()
    # and it is bounded by the quantisation step spread over the orthonormal rows, times the gate, plus x's own bf16 rounding
    assert np.abs(resid).max() <= 1.5 * (step / 2 * np.sqrt(r) + 2.0 ** -8 * np.abs(x).max() * np.sqrt(d))


def test_attention_over_int8_coefficients_stays_close_to_bf16_coefficients():
    """Tiny config (BJ:7): quantising the generator's bf16 coefficients to the 8-bit format moves the oracle's attention output by
    well under the 5e-3 rel-L2 parity budget -- the format is usable for the decode path (context for NEXT-1, not a parity claim)."""
    wl = gen.WORKLOADS["tiny"]
    oc, _ = make_oracle(wl)
    oc8, _ = make_oracle(wl)
    inp = workload_inputs(wl, 0)
    nf = int(inp["flag"].sum())
    ranks = np.asarray(wl.tier_ranks)[inp["tier"]]
    cK, cV = f64(inp["cK"]), f64(inp["cV"])
    cK8, cV8 = np.zeros_like(cK), np.zeros_like(cV)
    for rk in set(ranks.tolist()):
        sel = ranks == rk
        for src, dst in ((cK, cK8), (cV, cV8)):
            codes, exps = c8.quantize_coef_i8(src[sel].astype(np.float32), rank=rk)
            dst[sel] = c8.dequant_coef_i8(codes, exps)
    kw = dict(residK=inp["rK"].numpy() if nf else None, residV=inp["rV"].numpy() if nf else None)
    oc.append_raw(0, inp["tier"], inp["flag"], cK, cV, **kw)
    oc8.append_raw(0, inp["tier"], inp["flag"], cK8, cV8, **kw)
    q = f64(gen.make_q(wl, 0))
    o, o8 = oc.decode_all_layers([0], q), oc8.decode_all_layers([0], q)
    assert rel_l2(o8, o) < 2e-2
