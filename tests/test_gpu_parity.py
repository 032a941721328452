"""GPU parity: the CUDA path (through the C ABI / ctypes binding) against the CPU oracle on the same seeded inputs.

Bars (BASELINE.json north_star): tier routing and int4 dequantisation bit-exact; attention outputs within
max-abs <= 2e-3 * max|V-hat| and relative L2 <= 5e-3 per (layer, sequence) block.
"""
import dataclasses

import numpy as np
import pytest
import torch

import gen
from oracle import dwkv_oracle as orc
from helpers import f64, oracle_slice_from_kept, check_output, rel_l2, make_oracle, workload_inputs, oracle_load

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mod():
    from paper_2607_06523_b200 import binding, harness
    return binding, harness


def all_lh(wl):
    return [(l, h) for l in range(wl.L) for h in range(wl.H_kv)]


def load(harness, wl, routings, keep=None, chunk=1024, softmax_scale=0.0):
    cache, consts = harness.make_cache(wl, n_seqs=len(routings), max_tokens=max(len(t) for t, _ in routings) + 256,
                                       arena_bytes=harness.arena_bytes_for(wl, routings, 2), softmax_scale=softmax_scale)
    keep = all_lh(wl) if keep is None else keep
    kept = [harness.fill_sequence(cache, wl, s, s, t, f, chunk=chunk, keep=keep) for s, (t, f) in enumerate(routings)]
    return cache, consts, kept


def compare(wl, cache, consts, kept, routings, q, out, lhs=None, scale=None, what=""):
    """q, out: [n_seq, L, Hq, d] tensors. Checks every (sequence, layer) block over the kv heads in `lhs`."""
    o = out.double().cpu().numpy()
    qn = f64(q)
    worst = 0.0
    lhs = all_lh(wl) if lhs is None else lhs
    for s, (tier, flag) in enumerate(routings):
        for l in sorted({l for l, _ in lhs}):
            hs = [h for (ll, h) in lhs if ll == l]
            ref = []; got = []; vmax = 0.0
            for h in hs:
                sl = slice(h * wl.G, (h + 1) * wl.G)
                o_ref, V, _ = oracle_slice_from_kept(wl, consts, tier, flag, kept[s][(l, h)], qn[s, l, sl], l, h, scale)
                ref.append(o_ref); got.append(o[s, l, sl]); vmax = max(vmax, float(np.abs(V).max()))
            _, rel = check_output(np.concatenate(got), np.concatenate(ref), vmax, f"{what} seq {s} layer {l}")
            worst = max(worst, rel)
    return worst


# ---------------------------------------------------------------------------------------------------------------
def test_tiny_config_all_layers_and_per_layer(mod):
    """BASELINE.json configs[0], element by element, both launch modes, plus the peaked variants (pin P12)."""
    binding, harness = mod
    wl = gen.WORKLOADS["tiny"]
    routings = [gen.make_routing(wl, 0)]
    cache, consts, kept = load(harness, wl, routings)
    for gain in (1.0, 8.0, 64.0):
        q = gen.make_q(wl, device="cuda", gain=gain)
        out = cache.decode_attention(-1, [0], q)
        compare(wl, cache, consts, kept, routings, q, out, what=f"all-layers gain {gain}")
        out2 = torch.stack([cache.decode_attention(l, [0], q[:, l].contiguous()) for l in range(wl.L)], dim=1)
        compare(wl, cache, consts, kept, routings, q, out2, what=f"per-layer gain {gain}")
        assert rel_l2(out2.cpu().numpy(), out.cpu().numpy()) < 2e-3
    fp = cache.footprint()
    assert fp["used_bytes"] == orc.footprint_bytes(*routings[0], wl.tier_ranks, wl.d, wl.L, wl.H_kv)
    assert fp["dense_equiv_bytes"] == 512 * wl.L * wl.H_kv * 4 * wl.d
    cache.destroy()


def test_routing_and_dequant_bit_exact(mod):
    """Export the stored entries: tier/flag/slot == oracle routing; coefficients, codes, scales and dequantised values
    bit-exact against the oracle quantiser on the same fp32 residuals (reading A15 i, ii)."""
    binding, harness = mod
    wl = gen.WORKLOADS["tiny"]
    tier, flag = gen.make_routing(wl, 0)
    cache, consts, kept = load(harness, wl, [(tier, flag)], chunk=200)     # several appends: slots carry over
    dump = cache.export_tokens(0, 0, len(tier))
    cls, slot, _ = orc.route_slots(tier, flag, len(wl.tier_ranks))
    assert np.array_equal(dump["tier"].cpu().numpy(), tier) and np.array_equal(dump["flag"].cpu().numpy(), flag)
    assert np.array_equal(dump["slot"].cpu().numpy(), slot)
    idx = np.nonzero(flag)[0]
    for (l, h) in all_lh(wl):
        k = kept[0][(l, h)]
        for z in "KV":
            got = dump["coef" + z][:, l, h].cpu().view(torch.int16).numpy()
            want = k["c" + z].view(torch.int16).numpy()
            assert np.array_equal(got, want)
            codes, scales = orc.quantize_int4_g16(k["r" + z].numpy())
            gc = dump["code" + z][:, l, h].cpu().numpy()
            lo = (gc & 15).astype(np.int8); hi = (gc >> 4).astype(np.int8)
            lo = np.where(lo > 7, lo - 16, lo); hi = np.where(hi > 7, hi - 16, hi)
            dec = np.stack([lo, hi], axis=-1).reshape(len(tier), wl.d)
            assert np.array_equal(dec[idx], codes) and not dec[flag == 0].any()
            gs = dump["scale" + z][:, l, h].cpu().numpy()
            assert np.array_equal(gs[idx].view(np.uint16), scales.view(np.uint16)) and not gs[flag == 0].view(np.uint16).any()
            deq = dump["deq" + z][:, l, h].cpu().numpy()
            assert np.array_equal(deq[idx].view(np.uint32), orc.dequant_int4_g16(codes, scales).view(np.uint32))
    # partial export window
    d2 = cache.export_tokens(0, 100, 37, want=("slot", "coefK"))
    assert np.array_equal(d2["slot"].cpu().numpy(), slot[100:137])
    cache.destroy()


def test_raw_mode_b_codes_and_minus_eight(mod):
    """Load codes + scales directly (canonical nibble order), including code -8; compare with the oracle."""
    binding, harness = mod
    wl = dataclasses.replace(gen.WORKLOADS["tiny"], T=(77,))
    rng = np.random.default_rng(5)
    T = 77
    tier = rng.integers(0, 2, T).astype(np.uint8); flag = rng.integers(0, 2, T).astype(np.uint8)
    nf = int(flag.sum())
    cK, cV = gen.make_coef_chunk(wl, 0, 0, tier, device="cuda")
    codes = {z: rng.integers(-8, 8, (nf, wl.L, wl.H_kv, wl.d)).astype(np.int8) for z in "KV"}
    scales = {z: rng.uniform(0.001, 0.05, (nf, wl.L, wl.H_kv, wl.d // 16)).astype(np.float16) for z in "KV"}
    packed = {z: ((codes[z][..., 0::2] & 15) | ((codes[z][..., 1::2] & 15) << 4)).astype(np.uint8) for z in "KV"}
    cache, consts = harness.make_cache(wl, n_seqs=1, max_tokens=128)
    dev = lambda a: torch.as_tensor(a).cuda()
    cache.append_raw(0, tier, flag, cK, cV, codeK=dev(packed["K"]), codeV=dev(packed["V"]), scaleK=dev(scales["K"]), scaleV=dev(scales["V"]))
    BK, BV, gK, gV = consts
    oc = orc.OracleCache(wl.L, wl.w, wl.H_kv, wl.G, wl.d, wl.tier_ranks, f64(BK), f64(BV), f64(gK), f64(gV))
    oc.append_raw(0, tier, flag, f64(cK), f64(cV), codeK=codes["K"], scaleK=scales["K"], codeV=codes["V"], scaleV=scales["V"])
    dump = cache.export_tokens(0, 0, T, want=("codeK", "deqV"))
    assert np.array_equal(dump["codeK"].cpu().numpy()[flag == 1], packed["K"])
    assert np.array_equal(dump["deqV"].cpu().numpy()[flag == 1], orc.dequant_int4_g16(codes["V"], scales["V"]))
    q = gen.make_q(wl, device="cuda")
    out = cache.decode_attention(-1, [0], q).double().cpu().numpy()
    ref = oc.decode_all_layers([0], f64(q))
    for l in range(wl.L):
        check_output(out[0, l], ref[0, l], oc.max_abs_vhat(0, l), f"mode B layer {l}")
    cache.destroy()


def test_split_invariance_p11(mod):
    """Result independent of the work split (pin P11): one block per unit, a single warp slice for the whole step, a few
    slices, class-interleaved order with tiny units, every combine shape and the default plan. The softmax reference of
    every warp is integer-valued (log2 units), so different cuts change p, its hi + lo split and the bf16 rounding of the p * scaleV
    operand by exact powers of two only: the variants agree to fp32 summation order (<= 2e-6 rel-L2; SURVEY.md
    section 8c asks 1e-6; measured 5.8e-7, printed); every variant must also meet the oracle tolerance."""
    binding, harness = mod
    wl = gen.WORKLOADS["tiny"]
    routings = [gen.make_routing(wl, 0)]
    cache, consts, kept = load(harness, wl, routings)
    q = gen.make_q(wl, device="cuda", gain=4.0)
    outs, shapes = [], []
    base = {"max_unit_blocks": 0, "n_slices": 0, "interleave": 0, "unit_kb": 64, "combine_warps": 0}
    for change in ({"max_unit_blocks": 1}, {"n_slices": 1}, {"n_slices": 7}, {"interleave": 1, "unit_kb": 1}, {"interleave": -1},
                   {"n_slices": 296, "combine_warps": 4}, {"combine_warps": 4}, {"combine_warps": 1, "n_slices": 592},
                   {"n_slices": 148, "max_unit_blocks": 1}, {}):
        for k, v in {**base, **change}.items():
            cache.set_option(k, v)
        outs.append(cache.decode_attention(-1, [0], q).double().cpu().numpy())
        # the plan really is the one asked for (a cached plan must not survive an option change)
        shapes.append((int(cache.get_stat("plan_slices")), int(cache.get_stat("plan_slots"))))
        want = change.get("n_slices", 0)
        if want:
            assert shapes[-1][0] == want, (change, shapes[-1])
    assert shapes[1][1] == wl.L * wl.H_kv            # one slice: one partial per segment
    assert len(set(shapes)) >= 5, shapes
    worst = max(rel_l2(o, outs[0]) for o in outs[1:])
    print(f"P11 split invariance: worst rel-L2 between work splits {worst:.2e}")
    assert worst < 2e-6
    for o in outs:
        compare(wl, cache, consts, kept, routings, q, torch.as_tensor(o), what="split variant")
    cache.destroy()


@pytest.mark.parametrize("T", [1, 2, 31, 32, 33, 257])
def test_short_and_ragged_lengths(mod, T):
    """T = 1 gives o = V-hat[0] (pin P6); lengths around the 32-slot block and tile sizes (ragged tails)."""
    binding, harness = mod
    wl = dataclasses.replace(gen.WORKLOADS["tiny"], T=(T,), S0=0)
    rng = np.random.default_rng(T)
    tier = rng.integers(0, 2, T).astype(np.uint8); flag = (rng.random(T) < 0.4).astype(np.uint8)
    cache, consts, kept = load(harness, wl, [(tier, flag)])
    q = gen.make_q(wl, device="cuda", gain=3.0)
    out = cache.decode_attention(-1, [0], q)
    compare(wl, cache, consts, kept, [(tier, flag)], q, out, what=f"T={T}")
    if T == 1:
        o = out.double().cpu().numpy()
        for (l, h) in all_lh(wl):
            _, V, _ = oracle_slice_from_kept(wl, consts, tier, flag, kept[0][(l, h)], f64(q)[0, l, h * wl.G:(h + 1) * wl.G], l, h)
            np.testing.assert_allclose(o[0, l, h * wl.G:(h + 1) * wl.G], np.broadcast_to(V[0], (wl.G, wl.d)), rtol=2e-3, atol=1e-6)
    cache.destroy()


def test_extreme_tier_patterns_multi_sequence(mod):
    """All-lowest/no residual, all-top/all flagged, alternating tiers, and an ordinary mix decoded in ONE call
    (BASELINE.json configs[4] extremes, small shape), also addressed through a permuted seq_ids list."""
    binding, harness = mod
    wl = dataclasses.replace(gen.WORKLOADS["tiny"], T=(300, 45, 131, 512),
                             patterns=("all_low", "all_top_flag", "alternating", ""))
    routings = [gen.make_routing(wl, s) for s in range(4)]
    assert routings[0][0].max() == 0 and routings[1][1].all()
    cache, consts, kept = load(harness, wl, routings)
    q = gen.make_q(wl, device="cuda", gain=2.0)
    out = cache.decode_attention(-1, [0, 1, 2, 3], q)
    compare(wl, cache, consts, kept, routings, q, out, what="extremes")
    perm = [2, 0, 3, 1]
    out_p = cache.decode_attention(-1, perm, q[perm].contiguous())
    assert rel_l2(out_p.cpu().numpy(), out[perm].cpu().numpy()) < 1e-6
    cache.destroy()


def test_llama8b_shape_d128_three_tiers_sampled(mod):
    """Llama-3-8B shape (d=128, G=4, ranks 8/16/32), two ragged sequences spanning several pages of the flagged class and
    a ragged tail; sampled (layer, head) slices against the oracle, per-layer launch included."""
    binding, harness = mod
    wl = dataclasses.replace(gen.WORKLOADS["llama8b_16k_b8"], L=4, T=(3000, 1237))
    routings = [gen.make_routing(wl, s) for s in range(2)]
    keep = [(0, 0), (1, 3), (3, 7), (2, 5)]
    cache, consts, kept = load(harness, wl, routings, keep=keep, chunk=700)
    for gain in (1.0, 8.0):
        q = gen.make_q(wl, device="cuda", gain=gain)
        out = cache.decode_attention(-1, [0, 1], q)
        compare(wl, cache, consts, kept, routings, q, out, lhs=keep, what=f"8b gain {gain}")
    out3 = cache.decode_attention(3, [0, 1], q[:, 3].contiguous())
    # a per-layer call cuts the work into different warp slices: other rescale points and other bf16 roundings of the
    # p * scaleV operand of the residual-V MMA, so equality holds to that rounding level only
    assert rel_l2(out3.cpu().numpy(), out[:, 3].cpu().numpy()) < 2e-3
    cache.destroy()


def test_llama70b_shape_g8_ranks_8_24_48(mod):
    """Llama-3-70B shape (G=8, w=4, ranks 8/24/48: odd numbers of 8-column chunks) with isolated top-tier singles."""
    binding, harness = mod
    wl = dataclasses.replace(gen.WORKLOADS["llama70b_128k_b1"], L=4, T=(2100,))
    routings = [gen.make_routing(wl, 0)]
    keep = [(0, 1), (3, 6)]
    cache, consts, kept = load(harness, wl, routings, keep=keep, chunk=1000)
    q = gen.make_q(wl, device="cuda", gain=2.0)
    out = cache.decode_attention(-1, [0], q)
    compare(wl, cache, consts, kept, routings, q, out, lhs=keep, what="70b")
    cache.destroy()


def _check_reconstruction_within_one_step(wl, consts, z, coef_g, coef_w, code_g, code_w, scale_g, scale_w, fl):
    """DESIGN.md reading A15 (iii): where a coefficient differs by its bf16 ulp the residual absorbs the difference, so the two
    reconstructions gate * (c . B) + code * scale of a flagged token agree to within one quantisation step of the group
    (each lies within half a step of x)."""
    BK, BV, gK, gV = consts
    Bz = f64(BK if z == "K" else BV)[np.arange(wl.L) // wl.w]                # [L, H, r, d]
    gz = f64(gK if z == "K" else gV)                                         # [L, H, d]
    sg = np.repeat(scale_g.astype(np.float64), 16, axis=-1); sw = np.repeat(scale_w.astype(np.float64), 16, axis=-1)
    rec_g = gz[None] * np.einsum("tlhr,lhrd->tlhd", coef_g, Bz) + code_g * sg
    rec_w = gz[None] * np.einsum("tlhr,lhrd->tlhd", coef_w, Bz) + code_w * sw
    assert np.all(np.abs(rec_g - rec_w)[fl] <= np.maximum(sg, sw)[fl] * (1 + 1e-6))


def test_append_compress_against_oracle(mod):
    """dwkv_append_compress from dense K/V (reading A15 iii): coefficients within 1 bf16 ulp of the fp64 oracle on a tiny
    fraction, codes within +-1 on <= 0.1 % of entries (and reconstruction within one scale there), attention within
    tolerance; routing bit-exact; a second append continues the slots."""
    binding, harness = mod
    wl = dataclasses.replace(gen.WORKLOADS["tiny"], T=(96,))
    cache, consts = harness.make_cache(wl, n_seqs=2, max_tokens=512)
    BK, BV, gK, gV = consts
    oc = orc.OracleCache(wl.L, wl.w, wl.H_kv, wl.G, wl.d, wl.tier_ranks, f64(BK), f64(BV), f64(gK), f64(gV))
    rng = np.random.default_rng(3)
    t0 = {0: 0, 1: 0}
    for step in range(2):
        n_new = [40, 23] if step == 0 else [9, 64]
        tier = rng.integers(0, 2, sum(n_new)).astype(np.uint8); flag = (rng.random(sum(n_new)) < 0.5).astype(np.uint8)
        ks, vs = [], []
        for s, n in enumerate(n_new):
            k, v = gen.make_dense_kv_chunk(wl, s, t0[s], n, BK, BV, gK, gV, device="cuda")
            ks.append(k); vs.append(v); t0[s] += n
        k_new, v_new = torch.cat(ks), torch.cat(vs)
        cache.append_compress([0, 1], n_new, k_new, v_new, tier, flag)
        off = 0
        for s, n in enumerate(n_new):
            oc.append_compress(s, f64(k_new[off:off + n]), f64(v_new[off:off + n]), tier[off:off + n], flag[off:off + n])
            off += n
    for s in (0, 1):
        T = oc.seq_len(s)
        assert cache.seq_len(s) == T
        dump = cache.export_tokens(s, 0, T)
        S = oc.seqs[s]
        assert np.array_equal(dump["slot"].cpu().numpy(), S["slot"]) and np.array_equal(dump["tier"].cpu().numpy(), S["tier"])
        for z in "KV":
            got = dump["coef" + z].double().cpu().numpy()
            want = S["c" + z]
            ulp = np.maximum(np.abs(want), 2.0 ** -126) * 2.0 ** -7
            assert np.all(np.abs(got - want) <= ulp)
            assert np.mean(got != want) < 5e-3
            gc = dump["code" + z].cpu().numpy()
            lo = (gc & 15).astype(np.int8); hi = (gc >> 4).astype(np.int8)
            lo = np.where(lo > 7, lo - 16, lo); hi = np.where(hi > 7, hi - 16, hi)
            dec = np.stack([lo, hi], axis=-1).reshape(S["code" + z].shape)
            diff = np.abs(dec.astype(np.int32) - S["code" + z])
            fl = S["flag"].astype(bool)
            assert diff.max() <= 1 and np.mean(diff[fl] != 0) <= 2e-3
            assert not dec[~fl].any()
            # where the coefficients of a (token, layer, head) agree the scales must be identical or adjacent fp16 values;
            # where one differs by its bf16 ulp the residual moves with it, and the reconstructions must agree to within one
            # quantisation step of the group (reading A15 iii)
            same = (got == want).all(-1)                                             # [T, L, H]
            gs16 = dump["scale" + z].cpu().numpy(); ws16 = S["scale" + z]
            gs = gs16.view(np.uint16).astype(np.int32); ws = ws16.view(np.uint16).astype(np.int32)
            assert np.abs(gs - ws)[same].max() <= 1 and np.mean(gs != ws) <= 5e-3
            _check_reconstruction_within_one_step(wl, consts, z, got, want, dec, S["code" + z], gs16, ws16, fl)
    q = gen.make_q(wl, device="cuda", n_seq=2)
    out = cache.decode_attention(-1, [0, 1], q).double().cpu().numpy()
    ref = oc.decode_all_layers([0, 1], f64(q))
    for s in (0, 1):
        for l in range(wl.L):
            check_output(out[s, l], ref[s, l], oc.max_abs_vhat(s, l), f"append seq {s} layer {l}")
    cache.destroy()


@pytest.mark.parametrize("d,G,ranks", [(64, 1, (8,)), (64, 3, (16, 24)), (64, 8, (8, 16)), (64, 5, (24, 48, 64)), (128, 2, (8, 64)),
                                        (128, 6, (16, 32)), (128, 7, (8, 24, 48)), (128, 8, (32, 64)), (128, 4, (8, 16, 24, 32))])
def test_kernel_instances_small_shapes(mod, d, G, ranks):
    """Every instance family of the fused decode kernel (PAIR for G <= 4, FULL for G <= 8; head dim 64 / 128; basis ranks 8 .. 64,
    odd and even numbers of 8-column chunks; 1 .. 4 tiers) against the oracle on a small ragged two-sequence cache, all-layer
    and per-layer calls, with a peaked-softmax variant."""
    binding, harness = mod
    nt = len(ranks)
    frac = tuple([1.0 / nt] * nt)
    wl = dataclasses.replace(gen.WORKLOADS["tiny"], d=d, G=G, tier_ranks=ranks, tier_frac=frac, resid_frac=0.2, L=2, w=1, H_kv=2,
                             T=(333, 70), S0=8)
    rng = np.random.default_rng(d + 7 * G + len(ranks))
    routings = []
    for T in wl.T:
        tier = rng.integers(0, nt, T).astype(np.uint8); flag = (rng.random(T) < 0.3).astype(np.uint8)
        routings.append((tier, flag))
    cache, consts, kept = load(harness, wl, routings, chunk=100)
    for gain in (1.0, 16.0):
        q = gen.make_q(wl, device="cuda", gain=gain)
        out = cache.decode_attention(-1, [0, 1], q)
        compare(wl, cache, consts, kept, routings, q, out, what=f"d={d} G={G} ranks={ranks} gain={gain}")
    out1 = cache.decode_attention(1, [0, 1], q[:, 1].contiguous())
    assert rel_l2(out1.cpu().numpy(), out[:, 1].cpu().numpy()) < 2e-3
    cache.destroy()


@pytest.mark.parametrize("shape", ["8b", "70b", "odd", "8b_all_layers", "r64"])
def test_append_compress_tensor_core_tiles(mod, shape):
    """dwkv_append_compress on the shapes of the big configs: d = 128 with three tiers (8B: r = 32, 70B: r = 48, G = 8) and a basis of
    rank 24 (odd number of 8-column chunks, d = 64); token counts that are not multiples of the 16-token tile, several
    sequences per call, a second call that continues the slots. Same bars as the tiny append test (reading A15 iii)."""
    binding, harness = mod
    if shape == "8b":
        wl = dataclasses.replace(gen.WORKLOADS["llama8b_16k_b8"], L=2, T=(64, 64, 64))
    elif shape == "70b":
        wl = dataclasses.replace(gen.WORKLOADS["llama70b_128k_b1"], L=4, T=(64, 64, 64))
    elif shape == "8b_all_layers":   # 256 (layer, head) segments > CTAs of the persistent grid, dozens of tiles per segment:
        wl = dataclasses.replace(gen.WORKLOADS["llama8b_16k_b8"], T=(64, 64, 64))     # CTAs cross segments, warps refill their rings
    elif shape == "r64":             # basis rank 64 at d = 128: the 8-warp / 2-stage launch configuration
        wl = dataclasses.replace(gen.WORKLOADS["llama8b_16k_b8"], L=2, tier_ranks=(16, 64), tier_frac=(0.5, 0.5), T=(64, 64, 64))
    else:
        wl = dataclasses.replace(gen.WORKLOADS["tiny"], tier_ranks=(8, 24), T=(64, 64, 64))
    calls = ([700, 333, 64], [1, 30, 0]) if shape == "8b_all_layers" else ([37, 5, 64], [1, 30, 0])
    cache, consts = harness.make_cache(wl, n_seqs=3, max_tokens=1024)
    BK, BV, gK, gV = consts
    oc = orc.OracleCache(wl.L, wl.w, wl.H_kv, wl.G, wl.d, wl.tier_ranks, f64(BK), f64(BV), f64(gK), f64(gV))
    rng = np.random.default_rng(11)
    nt = len(wl.tier_ranks)
    t0 = {0: 0, 1: 0, 2: 0}
    for n_new in calls:
        tier = rng.integers(0, nt, sum(n_new)).astype(np.uint8); flag = (rng.random(sum(n_new)) < 0.3).astype(np.uint8)
        ks, vs = [], []
        for s_, n in enumerate(n_new):
            k, v = gen.make_dense_kv_chunk(wl, s_, t0[s_], n, BK, BV, gK, gV, device="cuda")
            ks.append(k); vs.append(v); t0[s_] += n
        k_new, v_new = torch.cat(ks), torch.cat(vs)
        cache.append_compress([0, 1, 2], n_new, k_new, v_new, tier, flag)
        off = 0
        for s_, n in enumerate(n_new):
            oc.append_compress(s_, f64(k_new[off:off + n]), f64(v_new[off:off + n]), tier[off:off + n], flag[off:off + n])
            off += n
    for s_ in (0, 1, 2):
        T = oc.seq_len(s_)
        assert cache.seq_len(s_) == T
        dump = cache.export_tokens(s_, 0, T)
        S = oc.seqs[s_]
        assert np.array_equal(dump["slot"].cpu().numpy(), S["slot"]) and np.array_equal(dump["tier"].cpu().numpy(), S["tier"])
        fl = S["flag"].astype(bool)
        for z in "KV":
            got = dump["coef" + z].double().cpu().numpy(); want = S["c" + z]
            # reading A15 (iii): one bf16 ulp of the oracle's value, or -- for dot products that cancel to almost nothing --
            # the fp32 accumulation error of a d-term dot product, 2^-20 of the token's largest coefficient
            ulp = np.maximum(np.abs(want) * 2.0 ** -7, np.abs(want).max(axis=-1, keepdims=True) * 2.0 ** -20)
            assert np.all(np.abs(got - want) <= ulp) and np.mean(got != want) < 1e-3      # measured: <= 3.3e-4 (typically 1e-4)
            gc = dump["code" + z].cpu().numpy()
            lo = (gc & 15).astype(np.int8); hi = (gc >> 4).astype(np.int8)
            lo = np.where(lo > 7, lo - 16, lo); hi = np.where(hi > 7, hi - 16, hi)
            dec = np.stack([lo, hi], axis=-1).reshape(S["code" + z].shape)
            diff = np.abs(dec.astype(np.int32) - S["code" + z])
            assert not dec[~fl].any()
            # a coefficient that differs by one bf16 ulp moves the whole residual of that (token, layer, head): there the two
            # reconstructions must agree to within one quantisation step; everywhere else the scales are identical or adjacent fp16 values
            same = np.all(got == want, axis=-1)                                   # [T, L, H]
            rows = same & fl[:, None, None]                                       # flagged rows with identical coefficients
            assert diff[rows].max(initial=0) <= 1 and (not rows.any() or np.mean(diff[rows] != 0) <= 1e-3)      # S:§8c A15 (iii): 0.1 %; measured <= 3e-6
            print(f"A15(iii) {shape} seq {s_} {z}: coefficients differing from the fp64 oracle {np.mean(got != want):.2e}, "
                  f"codes differing (rows with equal coefficients) {np.mean(diff[rows] != 0) if rows.any() else 0.0:.2e}")
            gsf = dump["scale" + z].cpu().numpy(); wsf = S["scale" + z]
            gs = gsf.view(np.uint16).astype(np.int32); ws = wsf.view(np.uint16).astype(np.int32)
            assert np.abs(gs - ws)[same].max() <= 1 and np.mean((gs != ws)[same]) <= 5e-3
            _check_reconstruction_within_one_step(wl, consts, z, got, want, dec, S["code" + z], gsf, wsf, fl)
    q = gen.make_q(wl, device="cuda", n_seq=3)
    out = cache.decode_attention(-1, [0, 1, 2], q).double().cpu().numpy()
    ref = oc.decode_all_layers([0, 1, 2], f64(q))
    for s_ in (0, 1, 2):
        for l in range(wl.L):
            check_output(out[s_, l], ref[s_, l], oc.max_abs_vhat(s_, l), f"append {shape} seq {s_} layer {l}")
    cache.destroy()


def test_errors_and_reset(mod):
    binding, harness = mod
    wl = dataclasses.replace(gen.WORKLOADS["tiny"], T=(64,))
    cache, consts = harness.make_cache(wl, n_seqs=2, max_tokens=100)
    q = gen.make_q(wl, device="cuda", n_seq=1)
    with pytest.raises(binding.DwkvError) as e:
        cache.decode_attention(-1, [0], q)
    assert e.value.code == binding.DWKV_E_EMPTY
    tier, flag = gen.make_routing(wl, 0)
    cK, cV = gen.make_coef_chunk(wl, 0, 0, tier, device="cuda")
    rK, rV = gen.make_resid_chunk(wl, 0, 0, int(flag.sum()), device="cuda")
    cache.append_raw(0, tier, flag, cK, cV, residK=rK, residV=rV)
    with pytest.raises(binding.DwkvError) as e:      # capacity: 64 + 64 > 100, state unchanged
        cache.append_raw(0, tier, flag, cK, cV, residK=rK, residV=rV)
    assert e.value.code == binding.DWKV_E_CAPACITY and cache.seq_len(0) == 64
    with pytest.raises(binding.DwkvError) as e:
        cache.append_raw(0, np.full(1, 7, np.uint8), np.zeros(1, np.uint8), cK[:1].contiguous(), cV[:1].contiguous())
    assert e.value.code == binding.DWKV_E_INVALID
    with pytest.raises(binding.DwkvError) as e:      # basis frozen once tokens exist (reading A19)
        cache.set_basis(consts[0], consts[1])
    assert e.value.code == binding.DWKV_E_STATE
    with pytest.raises(binding.DwkvError) as e:
        cache.decode_attention(5, [0], q[:, 0].contiguous())
    assert e.value.code == binding.DWKV_E_INVALID
    out1 = cache.decode_attention(-1, [0], q).clone()
    cache.reset_seq(0)
    assert cache.seq_len(0) == 0 and cache.footprint()["reserved_bytes"] == 0
    cache.append_raw(1, tier, flag, cK, cV, residK=rK, residV=rV)       # reuses the freed pages (zeroed on allocation)
    out2 = cache.decode_attention(-1, [1], q)
    assert torch.equal(out1, out2)
    bad = consts[2].clone(); bad[0, 0, 0] = 0
    c2 = binding.DwkvCache(wl.L, wl.w, wl.H_kv, wl.H_q, wl.d, list(wl.tier_ranks), 1, 64)
    with pytest.raises(binding.DwkvError) as e:
        c2.set_gates(bad, consts[3])
    assert e.value.code == binding.DWKV_E_STATE
    c2.destroy()
    with pytest.raises(binding.DwkvError):
        binding.DwkvCache(3, 2, 2, 4, 64, [8, 16], 1, 64)
    # basis construction and probe: argument and state errors
    c3 = binding.DwkvCache(wl.L, wl.w, wl.H_kv, wl.H_q, wl.d, list(wl.tier_ranks), 1, 64)
    kd = torch.zeros(16, wl.L, wl.H_kv, wl.d, dtype=torch.bfloat16, device="cuda")
    om = torch.zeros(wl.w, 32, 16, dtype=torch.bfloat16, device="cuda")
    with pytest.raises(binding.DwkvError) as e:      # gates first: the sketch is taken in gate-normalised space
        c3.build_basis(kd, kd, om)
    assert e.value.code == binding.DWKV_E_STATE
    c3.set_gates(consts[2], consts[3])
    with pytest.raises(binding.DwkvError) as e:      # n must be a multiple of 8
        c3.build_basis(kd[:12].contiguous(), kd[:12].contiguous(), om[:, :, :12].contiguous())
    assert e.value.code == binding.DWKV_E_INVALID
    with pytest.raises(binding.DwkvError) as e:      # sketch rows: multiple of 16, >= r
        c3.build_basis(kd, kd, om[:, :8].contiguous())
    assert e.value.code == binding.DWKV_E_INVALID
    c3.build_basis(kd, kd, om)                       # all-zero input: rows of norm zero are written as zeros, no NaN
    Bk, Bv = c3.export_basis(wl.M, wl.H_kv, wl.r, wl.d)
    assert torch.isfinite(Bk.float()).all() and torch.isfinite(Bv.float()).all()
    with pytest.raises(binding.DwkvError) as e:      # probe on an empty sequence
        c3.probe_error(0, 0, q[:, 0].contiguous(), kd[:, 0].permute(1, 0, 2).contiguous(), kd[:, 0].permute(1, 0, 2).contiguous())
    assert e.value.code == binding.DWKV_E_EMPTY
    c3.destroy()
    cache.destroy()


def test_dense_bf16_kernel_against_oracle_softmax(mod):
    """The comparison kernel: plain attention over a dense bf16 cache vs the oracle's softmax_attention."""
    binding, harness = mod
    torch.manual_seed(0)
    for (n_seq, L, H, G, d, T) in [(2, 2, 2, 4, 128, 1000), (1, 1, 2, 8, 128, 77), (1, 2, 2, 2, 64, 515)]:
        K = (torch.randn(n_seq, L, H, T, d, device="cuda") * 0.3).to(torch.bfloat16)
        V = (torch.randn(n_seq, L, H, T, d, device="cuda") * 0.3).to(torch.bfloat16)
        q = (torch.randn(n_seq, L, H * G, d, device="cuda") * 2).to(torch.bfloat16)
        out = binding.dense_decode_attention(K, V, q, H).double().cpu().numpy()
        Kn, Vn, qn = f64(K), f64(V), f64(q)
        for s in range(n_seq):
            for l in range(L):
                ref = np.concatenate([orc.softmax_attention(qn[s, l, h * G:(h + 1) * G], Kn[s, l, h], Vn[s, l, h], 1 / np.sqrt(d))
                                      for h in range(H)])
                check_output(out[s, l], ref, float(np.abs(Vn[s, l]).max()), f"dense {(n_seq, L, H, G, d, T)}")


def test_reset_returns_cleared_pages(mod):
    """Free pages are always all zero (dwkv_api.cu, zero_pages): a sequence of fat records (every token top tier + flagged, two
    pages) is dropped and a shorter sequence of another class mix is appended; the free list is a stack, so it gets the same two
    pages first, and its ragged page tails would hold the old bytes if they had not been cleared. Decode against the oracle."""
    binding, harness = mod
    wl_a = dataclasses.replace(gen.WORKLOADS["tiny"], T=(600,), patterns=("all_top_flag",))      # 448 tokens of that class per page
    tier_a, flag_a = gen.make_routing(wl_a, 0)
    page = wl_a.L * wl_a.H_kv * harness.PAGE_LH_BYTES
    cache, consts = harness.make_cache(wl_a, n_seqs=1, max_tokens=1024, arena_bytes=2 * len(wl_a.tier_ranks) * page)   # one page per class
    for rep, T in enumerate((77, 33)):
        harness.fill_sequence(cache, wl_a, 0, 0, tier_a, flag_a, chunk=128)
        assert cache.footprint()["reserved_bytes"] == 2 * page
        cache.reset_seq(0)
        assert cache.seq_len(0) == 0 and cache.footprint()["reserved_bytes"] == 0
        wl_b = dataclasses.replace(gen.WORKLOADS["tiny"], T=(T,), patterns=("",))
        rt_b = [gen.make_routing(wl_b, 0)]
        kept = [harness.fill_sequence(cache, wl_b, 0, 0, *rt_b[0], chunk=64, keep=all_lh(wl_b))]
        assert cache.footprint()["reserved_bytes"] >= 2 * page            # the two returned pages are in use again
        q = gen.make_q(wl_b, step=rep, device="cuda")
        out = cache.decode_attention(-1, [0], q)
        compare(wl_b, cache, consts, kept, rt_b, q, out, what=f"after reset, T = {T}")
        cache.reset_seq(0)
    cache.destroy()


@pytest.mark.parametrize("name", ["tiny", "8b"])
def test_probe_error_eq3(mod, name):
    """dwkv_probe_error (Eq. 3, reading A25): the compressed cache against a higher-fidelity dense cache of the same tokens
    (here: the oracle's reconstruction plus noise, rounded to bf16), per kv head over n_q query positions, vs the oracle's number
    computed from fp64 attention on both caches. A reference equal to the reconstruction itself gives e at the bf16 rounding level."""
    binding, harness = mod
    if name == "tiny":
        wl = gen.WORKLOADS["tiny"]
    else:
        wl = dataclasses.replace(gen.WORKLOADS["llama8b_16k_b8"], L=2, T=(777,))
    T = wl.T[0]
    oc, _ = make_oracle(wl)
    inp = workload_inputs(wl, 0, T, device="cuda")
    oracle_load(oc, 0, inp)
    cache, consts = harness.make_cache(wl, n_seqs=1, max_tokens=T + 64)
    nf = int(inp["flag"].sum())
    cache.append_raw(0, inp["tier"], inp["flag"], inp["cK"], inp["cV"], residK=inp["rK"] if nf else None, residV=inp["rV"] if nf else None)
    n_q, layer, eps = 3, wl.L - 1, 1e-6
    rng = np.random.default_rng(5)
    q = torch.stack([gen.make_q(wl, step=i, device="cuda", n_seq=1)[0, layer] for i in range(n_q)]).contiguous()      # [n_q, Hq, d]
    Kh = np.stack([oc.khat_vhat(0, layer, h)[0] for h in range(wl.H_kv)]); Vh = np.stack([oc.khat_vhat(0, layer, h)[1] for h in range(wl.H_kv)])
    for noise in (0.0, 0.05):
        K_ref = torch.from_numpy(Kh + noise * rng.standard_normal(Kh.shape)).to(torch.bfloat16).cuda().contiguous()      # [H, T, d]
        V_ref = torch.from_numpy(Vh + noise * rng.standard_normal(Vh.shape)).to(torch.bfloat16).cuda().contiguous()
        e = cache.probe_error(layer, 0, q, K_ref, V_ref, eps).double().cpu().numpy()
        a_ref = np.zeros((n_q, wl.H_q, wl.d)); a_cmp = np.zeros_like(a_ref)
        qn = f64(q)
        for i in range(n_q):
            for h in range(wl.H_kv):
                sl = slice(h * wl.G, (h + 1) * wl.G)
                a_ref[i, sl] = orc.softmax_attention(qn[i, sl], f64(K_ref[h]), f64(V_ref[h]), oc.scale)
                a_cmp[i, sl] = orc.softmax_attention(qn[i, sl], Kh[h], Vh[h], oc.scale)
        want = orc.probe_error(a_ref, a_cmp, wl.G, eps)
        # the GPU attention outputs carry their own error (<= 5e-3 rel-L2 each, typically 3e-4), which adds to the numerator
        assert np.all(np.abs(e - want) <= 0.02 * want + 2e-3), (name, noise, e, want)
        if noise == 0.0:
            assert np.all(e < 1e-2)
        else:
            assert np.all(e > 5e-2)
    cache.destroy()


@pytest.mark.parametrize("name", ["llama8b_64k_b1", "llama8b_64k_b8", "llama8b_16k_b8", "llama70b_128k_b1", "ragged32"])
def test_full_size_sampled_slices(mod, name):
    """BASELINE.json's full sizes in the launch configuration bench.py times (all layers in one call, persistent grid): sampled
    (sequence, layer, kv head) slices against the oracle, element by element, plus the peaked variant (pin P12) and, at full
    size too, q = 0 => the output is the mean of V-hat over the tokens (pin P5) on the sampled slices."""
    binding, harness = mod
    wl = gen.WORKLOADS[name]
    routings = [gen.make_routing(wl, s) for s in range(wl.n_seq)]
    cache, consts = harness.make_cache(wl, arena_bytes=harness.arena_bytes_for(wl, routings, 1))
    keep = [(0, 0), (wl.L // 2, 3), (wl.L - 1, wl.H_kv - 1)]
    # ragged32: T = 1, T = 12347, all-lowest, all-top-flagged, alternating tiers, and the last of the mixed sequences
    sampled = [0, 1, 2, 3, 4, wl.n_seq - 1] if name == "ragged32" else sorted({0, wl.n_seq - 1})
    kept = {}
    for s, (tier, flag) in enumerate(routings):
        kept[s] = harness.fill_sequence(cache, wl, s, s, tier, flag, chunk=8192, keep=keep if s in sampled else [])
    ids = list(range(wl.n_seq))
    for gain in (1.0, 8.0, 0.0):
        q = gen.make_q(wl, device="cuda", gain=gain)
        o = cache.decode_attention(-1, ids, q).double().cpu().numpy()
        qn = f64(q)
        for s in sampled:
            tier, flag = routings[s]
            for (l, h) in keep:
                sl = slice(h * wl.G, (h + 1) * wl.G)
                o_ref, V, _ = oracle_slice_from_kept(wl, consts, tier, flag, kept[s][(l, h)], qn[s, l, sl], l, h)
                check_output(o[s, l, sl], o_ref, float(np.abs(V).max()), f"{name} gain {gain} seq {s} (l,h)=({l},{h})")
                if gain == 0.0:
                    assert np.allclose(o_ref, V.mean(axis=0)[None], atol=1e-12)
        if gain == 8.0:
            # per-layer calls, the launch shape of a real decoder (and, for one long sequence, the planner's small-call slicing
            # with fewer slices than warps): the sampled layers against the oracle, for all sequences and for sequence 0 alone
            for (l, h) in keep:
                sl = slice(h * wl.G, (h + 1) * wl.G)
                o_l = cache.decode_attention(l, ids, q[:, l].contiguous()).double().cpu().numpy()
                s0 = sampled[-1]
                o_1 = cache.decode_attention(l, [s0], q[s0:s0 + 1, l].contiguous()).double().cpu().numpy()
                for s in sampled:
                    tier, flag = routings[s]
                    o_ref, V, _ = oracle_slice_from_kept(wl, consts, tier, flag, kept[s][(l, h)], qn[s, l, sl], l, h)
                    check_output(o_l[s, sl], o_ref, float(np.abs(V).max()), f"{name} per-layer seq {s} (l,h)=({l},{h})")
                    if s == s0:
                        check_output(o_1[0, sl], o_ref, float(np.abs(V).max()), f"{name} per-layer single seq {s} (l,h)=({l},{h})")
    fp = cache.footprint()
    assert fp["used_bytes"] == sum(orc.footprint_bytes(t, f, wl.tier_ranks, wl.d, wl.L, wl.H_kv) for t, f in routings)
    cache.destroy()


def test_append_compress_chunked_call(mod):
    """A call larger than the library's internal chunk (16384 rows): the chunk boundary falls inside the second sequence. Routing
    bit-exact, coefficients within one bf16 ulp of the oracle, attention within tolerance."""
    binding, harness = mod
    n_new = [10000, 9000]
    wl = dataclasses.replace(gen.WORKLOADS["tiny"], T=(n_new[0], n_new[1]))
    cache, consts = harness.make_cache(wl, n_seqs=2, max_tokens=max(n_new) + 64)
    BK, BV, gK, gV = consts
    oc = orc.OracleCache(wl.L, wl.w, wl.H_kv, wl.G, wl.d, wl.tier_ranks, f64(BK), f64(BV), f64(gK), f64(gV))
    routings = [gen.make_routing(wl, s) for s in range(2)]
    ks, vs = [], []
    for s, n in enumerate(n_new):
        k, v = gen.make_dense_kv_chunk(wl, s, 0, n, BK, BV, gK, gV, device="cuda")
        ks.append(k.contiguous()); vs.append(v.contiguous())
    k_new, v_new = torch.cat(ks), torch.cat(vs)
    tier = np.concatenate([r[0] for r in routings]); flag = np.concatenate([r[1] for r in routings])
    cache.append_compress([0, 1], n_new, k_new, v_new, tier, flag)
    off = 0
    for s, n in enumerate(n_new):
        oc.append_compress(s, f64(k_new[off:off + n]), f64(v_new[off:off + n]), tier[off:off + n], flag[off:off + n])
        off += n
    for s in (0, 1):
        dump = cache.export_tokens(s, 0, n_new[s])
        S = oc.seqs[s]
        assert np.array_equal(dump["slot"].cpu().numpy(), S["slot"]) and np.array_equal(dump["tier"].cpu().numpy(), S["tier"])
        assert np.array_equal(dump["flag"].cpu().numpy(), S["flag"])
        for z in "KV":
            got = dump["coef" + z].double().cpu().numpy(); want = S["c" + z]
            ulp = np.maximum(np.abs(want) * 2.0 ** -7, np.abs(want).max(axis=-1, keepdims=True) * 2.0 ** -20)
            assert np.all(np.abs(got - want) <= ulp) and np.mean(got != want) < 5e-3
    q = gen.make_q(wl, device="cuda", n_seq=2)
    out = cache.decode_attention(-1, [0, 1], q).double().cpu().numpy()
    ref = oc.decode_all_layers([0, 1], f64(q))
    for s in (0, 1):
        for l in range(wl.L):
            check_output(out[s, l], ref[s, l], oc.max_abs_vhat(s, l), f"chunked append seq {s} layer {l}")
    cache.destroy()


@pytest.mark.parametrize("tier_k,flag_k", [(0, 0), (0, 1), (1, 0), (1, 1)])
def test_page_boundaries_single_class(mod, tier_k, flag_k):
    """Sequences of ONE class whose length sits just below, at, just above one page stripe and past two (the planner's units end at
    page ends; a page holds 64 KB / block bytes * 32 tokens per (layer, head)), all decoded in one call and one by one."""
    binding, harness = mod
    base = gen.WORKLOADS["tiny"]
    rank = base.tier_ranks[tier_k]
    tpp = (65536 // (2 * (rank // 8) * 512 + flag_k * 40 * base.d)) * 32
    Ts = (tpp - 1, tpp, tpp + 1, 2 * tpp + 5)
    wl = dataclasses.replace(base, T=Ts, S0=0)
    routings = [(np.full(T, tier_k, np.uint8), np.full(T, flag_k, np.uint8)) for T in Ts]
    cache, consts, kept = load(harness, wl, routings, chunk=700)
    q = gen.make_q(wl, device="cuda", gain=2.0)
    out = cache.decode_attention(-1, [0, 1, 2, 3], q)
    compare(wl, cache, consts, kept, routings, q, out, what=f"class ({tier_k},{flag_k}) page boundary")
    for s in range(4):
        o1 = cache.decode_attention(-1, [s], q[s:s + 1].contiguous())
        assert rel_l2(o1.cpu().numpy(), out[s:s + 1].cpu().numpy()) < 2e-3
    fp = cache.footprint()
    page = wl.L * wl.H_kv * 65536
    assert fp["reserved_bytes"] == page * sum((T + tpp - 1) // tpp for T in Ts)
    cache.destroy()


def test_decode_loop_appends_one_token_per_step(mod):
    """The decode loop of a server: append one token per sequence, decode, repeat. Most steps open no new sub-block, so the planner
    only patches the token counts of its cached plan (fast path); some do and rebuild it. Every step is checked against the oracle,
    all-layer and per-layer."""
    binding, harness = mod
    wl = dataclasses.replace(gen.WORKLOADS["tiny"], T=(200, 77))
    oc, consts = make_oracle(wl)
    BK, BV, gK, gV = consts
    cache, _ = harness.make_cache(wl, n_seqs=2, max_tokens=512)
    for s in range(2):
        inp = workload_inputs(wl, s, wl.T[s], device="cuda")
        oracle_load(oc, s, inp)
        nf = int(inp["flag"].sum())
        cache.append_raw(s, inp["tier"], inp["flag"], inp["cK"], inp["cV"], residK=inp["rK"] if nf else None, residV=inp["rV"] if nf else None)
    rng = np.random.default_rng(9)
    q = gen.make_q(wl, device="cuda", n_seq=2)
    for step in range(40):
        tier = rng.integers(0, 2, 2).astype(np.uint8); flag = (rng.random(2) < 0.3).astype(np.uint8)
        ks, vs = [], []
        for s in range(2):
            k, v = gen.make_dense_kv_chunk(wl, s, 1000 + step, 1, BK.cuda(), BV.cuda(), gK.cuda(), gV.cuda(), device="cuda")
            ks.append(k); vs.append(v)
        k_new, v_new = torch.cat(ks).contiguous(), torch.cat(vs).contiguous()
        cache.append_compress([0, 1], [1, 1], k_new, v_new, tier, flag)
        for s in range(2):
            oc.append_compress(s, f64(k_new[s:s + 1]), f64(v_new[s:s + 1]), tier[s:s + 1], flag[s:s + 1])
        out = cache.decode_attention(-1, [0, 1], q).double().cpu().numpy()
        if step % 4 == 3 or step < 3:
            ref = oc.decode_all_layers([0, 1], f64(q))
            for s in range(2):
                for l in range(wl.L):
                    check_output(out[s, l], ref[s, l], oc.max_abs_vhat(s, l), f"loop step {step} seq {s} layer {l}")
            o1 = cache.decode_attention(1, [0, 1], q[:, 1].contiguous()).double().cpu().numpy()
            assert rel_l2(o1, out[:, 1]) < 2e-3
    assert cache.seq_len(0) == 240 and cache.seq_len(1) == 117
    cache.destroy()


def test_time_scan_sample_ring(mod):
    """Measurement aid of dwkv.h (option "time_scan", dwkv_get_stat): the library brackets the decode kernel of every call and
    keeps the last 64 brackets, so bench.py can run steps back to back and read every sample afterwards."""
    binding, harness = mod
    wl = gen.WORKLOADS["tiny"]
    tier, flag = gen.make_routing(wl, 0)
    cache, _ = harness.make_cache(wl)
    harness.fill_sequence(cache, wl, 0, 0, tier, flag, chunk=512)
    q = gen.make_q(wl, device="cuda")
    ref = cache.decode_attention(-1, [0], q).clone()
    assert cache.get_stat("scan_ms") < 0 and cache.get_stat("scan_samples") == 0      # nothing timed yet
    cache.set_option("time_scan", 1)
    for _ in range(5):
        out = cache.decode_attention(-1, [0], q)
    assert torch.equal(out, ref)                                                      # timing does not change the result
    assert cache.get_stat("scan_samples") == 5
    samples = [cache.get_stat(f"scan_ms@{i}") for i in range(5)]
    assert all(0.0 < s < 50.0 for s in samples)
    assert cache.get_stat("scan_ms") == samples[-1]
    assert cache.get_stat("scan_ms_min") == min(samples)
    assert abs(cache.get_stat("scan_ms_mean") - sum(samples) / 5) < 1e-6
    assert cache.get_stat("scan_ms@5") < 0 and cache.get_stat("scan_ms@-1") < 0
    for _ in range(70):                                                               # the ring keeps the last 64
        cache.decode_attention(-1, [0], q)
    assert cache.get_stat("scan_samples") == 64 and cache.get_stat("scan_ms@63") > 0 and cache.get_stat("scan_ms@64") < 0
    cache.set_option("time_scan", 1)                                                  # setting the option restarts the count
    assert cache.get_stat("scan_samples") == 0
    cache.set_option("time_scan", 0)
    cache.decode_attention(-1, [0], q)
    assert cache.get_stat("scan_samples") == 0
    cache.destroy()
