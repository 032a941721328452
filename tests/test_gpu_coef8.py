"""GPU parity of the 8-bit blockwise coefficient mode (dwkv.h option "coef_int8"; PAPER.md:56;
DESIGN.md reading A27) against the oracle, through the C ABI: the quantiser on load (bit-exact), the decode path over the byte
planes (BASELINE.json tolerance), append/compress from dense K/V, footprint closed form, error paths."""
import dataclasses

import numpy as np
import pytest
import torch

import gen
from oracle import dwkv_coef8_oracle as c8
from oracle import dwkv_oracle as orc
from helpers import f64, check_output, rel_l2, oracle_slice_from_kept
from test_gpu_parity import all_lh, compare

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mod():
    from paper_2607_06523_b200 import binding, harness
    return binding, harness


def load8(harness, wl, routings, keep=None, chunk=1024):
    cache, consts = harness.make_cache(wl, n_seqs=len(routings), max_tokens=max(len(t) for t, _ in routings) + 256,
                                       arena_bytes=harness.arena_bytes_for(wl, routings, 2), coef_int8=True)
    keep = all_lh(wl) if keep is None else keep
    kept = [harness.fill_sequence(cache, wl, s, s, t, f, chunk=chunk, keep=keep) for s, (t, f) in enumerate(routings)]
    return cache, consts, kept


def quantised(wl, tier, c):
    """What the oracle quantiser makes of the generator's coefficients c [T, r] (torch bf16): dequantised float64 [T, r]."""
    ranks = np.asarray(wl.tier_ranks)[tier]
    src = f64(c)
    out = np.zeros_like(src)
    for rk in set(ranks.tolist()):
        sel = ranks == rk
        codes, exps = c8.quantize_coef_i8(src[sel].astype(np.float32), rank=rk)
        out[sel] = c8.dequant_coef_i8(codes, exps)
    return out


def kept_quantised(wl, routings, kept):
    """The kept generator outputs with the coefficients replaced by their 8-bit quantisation: what the GPU cache holds."""
    out = []
    for (tier, _), ks in zip(routings, kept):
        o = {}
        for lh, k in ks.items():
            o[lh] = dict(k)
            for z in "KV":
                o[lh]["c" + z] = torch.tensor(quantised(wl, tier, k["c" + z]), dtype=torch.float64)
        out.append(o)
    return out


def test_load_quantises_bit_exact_and_footprint(mod):
    binding, harness = mod
    wl = gen.WORKLOADS["tiny"]
    tier, flag = gen.make_routing(wl, 0)
    cache, consts, kept = load8(harness, wl, [(tier, flag)], chunk=200)
    dump = cache.export_tokens(0, 0, len(tier))
    _, slot, _ = orc.route_slots(tier, flag, len(wl.tier_ranks))
    assert np.array_equal(dump["slot"].cpu().numpy(), slot)
    idx = np.nonzero(flag)[0]
    for (l, h) in all_lh(wl):
        k = kept[0][(l, h)]
        for z in "KV":
            got = dump["coef" + z][:, l, h].double().cpu().numpy()
            assert np.array_equal(got, quantised(wl, tier, k["c" + z]))              # bit-exact quantiser, exact bf16 export
            codes, scales = orc.quantize_int4_g16(k["r" + z].numpy())                # residual planes are untouched by the mode
            deq = dump["deq" + z][:, l, h].cpu().numpy()
            assert np.array_equal(deq[idx].view(np.uint32), orc.dequant_int4_g16(codes, scales).view(np.uint32))
            assert not deq[flag == 0].any()
    fp = cache.footprint()
    assert fp["used_bytes"] == c8.footprint_bytes_i8(tier, flag, wl.tier_ranks, wl.d, wl.L, wl.H_kv)
    # loading values that already lie on the grid is lossless: export -> reload into a second cache -> same bytes
    cache2, _ = harness.make_cache(wl, n_seqs=1, max_tokens=len(tier) + 8, coef_int8=True)
    nf = int(flag.sum())
    cache2.append_raw(0, tier, flag, dump["coefK"], dump["coefV"], codeK=dump["codeK"][torch.tensor(idx)].contiguous(),
                      codeV=dump["codeV"][torch.tensor(idx)].contiguous(), scaleK=dump["scaleK"][torch.tensor(idx)].contiguous(),
                      scaleV=dump["scaleV"][torch.tensor(idx)].contiguous())
    d2 = cache2.export_tokens(0, 0, len(tier), want=("coefK", "coefV"))
    assert torch.equal(d2["coefK"], dump["coefK"]) and torch.equal(d2["coefV"], dump["coefV"]) and nf > 0
    cache.destroy(); cache2.destroy()


def test_decode_tiny_all_layers_and_per_layer(mod):
    binding, harness = mod
    wl = gen.WORKLOADS["tiny"]
    routings = [gen.make_routing(wl, 0)]
    cache, consts, kept = load8(harness, wl, routings)
    kq = kept_quantised(wl, routings, kept)
    for gain in (1.0, 8.0, 64.0):
        q = gen.make_q(wl, device="cuda", gain=gain)
        out = cache.decode_attention(-1, [0], q)
        compare(wl, cache, consts, kq, routings, q, out, what=f"i8 all-layers gain {gain}")
        out2 = torch.stack([cache.decode_attention(l, [0], q[:, l].contiguous()) for l in range(wl.L)], dim=1)
        compare(wl, cache, consts, kq, routings, q, out2, what=f"i8 per-layer gain {gain}")
    cache.destroy()


@pytest.mark.parametrize("T", [1, 2, 31, 33, 257])
def test_short_and_ragged_lengths(mod, T):
    binding, harness = mod
    wl = dataclasses.replace(gen.WORKLOADS["tiny"], T=(T,), S0=min(32, T))
    rng = np.random.default_rng(T)
    tier = rng.integers(0, 2, T).astype(np.uint8); flag = (rng.random(T) < 0.4).astype(np.uint8)
    routings = [(tier, flag)]
    cache, consts, kept = load8(harness, wl, routings)
    q = gen.make_q(wl, device="cuda", gain=4.0)
    out = cache.decode_attention(-1, [0], q)
    compare(wl, cache, consts, kept_quantised(wl, routings, kept), routings, q, out, what=f"i8 T={T}")
    cache.destroy()


def test_llama8b_shape_pair_mode_sampled(mod):
    """d = 128, G = 4 (PAIR mode), ranks 8/16/32, two ragged sequences over several pages, sampled (layer, head) slices."""
    binding, harness = mod
    wl = dataclasses.replace(gen.WORKLOADS["llama8b_16k_b8"], L=4, T=(3000, 1237))
    routings = [gen.make_routing(wl, s) for s in range(2)]
    keep = [(0, 0), (1, 3), (3, 7), (2, 5)]
    cache, consts, kept = load8(harness, wl, routings, keep=keep, chunk=700)
    kq = kept_quantised(wl, routings, kept)
    for gain in (1.0, 8.0):
        q = gen.make_q(wl, device="cuda", gain=gain)
        out = cache.decode_attention(-1, [0, 1], q)
        compare(wl, cache, consts, kq, routings, q, out, lhs=keep, what=f"i8 8b gain {gain}")
    out3 = cache.decode_attention(3, [0, 1], q[:, 3].contiguous())
    assert rel_l2(out3.cpu().numpy(), out[:, 3].cpu().numpy()) < 2e-3
    cache.destroy()


@pytest.mark.parametrize("d,G,ranks", [(64, 1, (8,)), (64, 8, (8, 16)), (128, 8, (8, 24)), (128, 2, (16, 32)), (64, 3, (24, 32)),
                                        (128, 8, (8, 24, 48)), (128, 2, (16, 64)), (64, 4, (8, 48)), (64, 6, (32, 64))])
def test_kernel_instances(mod, d, G, ranks):
    """FULL mode (G > 4), odd chunk counts (rank 24), both head dims; ranks 48 and 64: two 32-column blocks per token vector
    (two exponent bytes per slot; BASELINE.json configs[3], the 70B shape, has r = 48)."""
    binding, harness = mod
    wl = dataclasses.replace(gen.WORKLOADS["tiny"], d=d, G=G, tier_ranks=ranks, tier_frac=tuple([1.0 / len(ranks)] * len(ranks)), T=(700,))
    routings = [gen.make_routing(wl, 0)]
    cache, consts, kept = load8(harness, wl, routings)
    q = gen.make_q(wl, device="cuda", gain=3.0)
    out = cache.decode_attention(-1, [0], q)
    compare(wl, cache, consts, kept_quantised(wl, routings, kept), routings, q, out, what=f"i8 d={d} G={G} ranks={ranks}")
    cache.destroy()


@pytest.mark.parametrize("shape", ["tiny", "8b", "r24", "70b", "r64"])
def test_append_compress_against_oracle(mod, shape):
    """dwkv_append_compress in 8-bit mode from dense K/V: the fp32 projection differs from the oracle's fp64 one in the last bits,
    which can move a code across a rounding boundary (reading A15 iii carried over): coefficients equal on >= 99.5 % of entries and
    within one quantisation step elsewhere; attention of the GPU path within tolerance of the oracle on ITS OWN compressed cache."""
    binding, harness = mod
    # tiny: d = 64, ranks 8 / 16; 8b: d = 128, G = 4, ranks 8 / 16 / 32 (1, 2 and 4 lane groups per vector in the warp kernel)
    # and calls of more than 64 tokens (several token chunks per (layer, head)); r24: a rank that is not a power of two
    wl = {"tiny": dataclasses.replace(gen.WORKLOADS["tiny"], T=(96,)),
          "8b": dataclasses.replace(gen.WORKLOADS["llama8b_16k_b8"], L=2, w=2, H_kv=2, T=(96, 96)),
          "r24": dataclasses.replace(gen.WORKLOADS["llama8b_16k_b8"], L=2, w=2, H_kv=1, tier_ranks=(8, 24),
                                     tier_frac=(0.5, 0.5), T=(96, 96)),
          # two 32-column blocks per token vector: the 70B shape (ranks 8 / 24 / 48, G = 8, w = 4) and a rank-64 basis
          "70b": dataclasses.replace(gen.WORKLOADS["llama70b_128k_b1"], L=4, H_kv=2, T=(96, 96)),
          "r64": dataclasses.replace(gen.WORKLOADS["llama8b_16k_b8"], L=2, w=2, H_kv=1, tier_ranks=(16, 64),
                                     tier_frac=(0.5, 0.5), T=(96, 96))}[shape]
    n_t = len(wl.tier_ranks)
    cache, consts = harness.make_cache(wl, n_seqs=2, max_tokens=512, coef_int8=True)
    BK, BV, gK, gV = consts
    oc = orc.OracleCache(wl.L, wl.w, wl.H_kv, wl.G, wl.d, wl.tier_ranks, f64(BK), f64(BV), f64(gK), f64(gV))
    rng = np.random.default_rng(5)
    t0 = {0: 0, 1: 0}
    for step in range(2):
        n_new = ([40, 23] if step == 0 else [9, 64]) if shape == "tiny" else ([140, 23] if step == 0 else [9, 75])
        tier = rng.integers(0, n_t, sum(n_new)).astype(np.uint8); flag = (rng.random(sum(n_new)) < 0.5).astype(np.uint8)
        ks, vs = [], []
        for s, n in enumerate(n_new):
            k, v = gen.make_dense_kv_chunk(wl, s, t0[s], n, BK, BV, gK, gV, device="cuda")
            ks.append(k); vs.append(v); t0[s] += n
        k_new, v_new = torch.cat(ks), torch.cat(vs)
        cache.append_compress([0, 1], n_new, k_new, v_new, tier, flag)
        off = 0
        for s, n in enumerate(n_new):
            c8.append_compress_i8(oc, s, f64(k_new[off:off + n]), f64(v_new[off:off + n]), tier[off:off + n], flag[off:off + n])
            off += n
    for s in (0, 1):
        T = oc.seq_len(s)
        assert cache.seq_len(s) == T
        dump = cache.export_tokens(s, 0, T)
        S = oc.seqs[s]
        assert np.array_equal(dump["slot"].cpu().numpy(), S["slot"]) and np.array_equal(dump["tier"].cpu().numpy(), S["tier"])
        fl = S["flag"].astype(bool)
        for z in "KV":
            got = dump["coef" + z].double().cpu().numpy(); want = S["c" + z]
            step_ = np.abs(want).max(axis=-1, keepdims=True) / 63.0                   # >= the block's 2^e (amax / 127 <= 2^e < 2 amax / 127)
            assert np.all(np.abs(got - want) <= step_ + 1e-300)
            assert np.mean(got != want) < 5e-3
            gc = dump["code" + z].cpu().numpy()
            lo = (gc & 15).astype(np.int8); hi = (gc >> 4).astype(np.int8)
            lo = np.where(lo > 7, lo - 16, lo); hi = np.where(hi > 7, hi - 16, hi)
            dec = np.stack([lo, hi], axis=-1).reshape(S["code" + z].shape)
            same = (got == want).all(-1)
            diff = np.abs(dec.astype(np.int32) - S["code" + z])
            assert diff[same].max() <= 1 and np.mean(diff[same] != 0) <= 2e-3 and not dec[~fl].any()
    q = gen.make_q(wl, device="cuda", n_seq=2)
    out = cache.decode_attention(-1, [0, 1], q).double().cpu().numpy()
    ref = oc.decode_all_layers([0, 1], f64(q))
    for s in (0, 1):
        for l in range(wl.L):
            check_output(out[s, l], ref[s, l], oc.max_abs_vhat(s, l), f"i8 append seq {s} layer {l}")
    cache.destroy()


@pytest.mark.parametrize("name", ["llama8b_16k_b8", "llama8b_64k_b1", "llama8b_64k_b8", "llama70b_128k_b1", "ragged32"])
def test_full_size_sampled_slices_i8(mod, name):
    """Every BASELINE.json config at full size in the paper's own coefficient format ("8-bit blockwise quantized";
    the 70B shape has rank 48 = two blocks per token vector): sampled (layer, head) slices of sampled sequences against the oracle
    fed with the oracle-quantised coefficients, all-layer call and one per-layer call."""
    binding, harness = mod
    wl = gen.WORKLOADS[name]
    routings = [gen.make_routing(wl, s) for s in range(wl.n_seq)]
    cache, consts = harness.make_cache(wl, arena_bytes=harness.arena_bytes_for(wl, routings, 1), coef_int8=True)
    keep = [(0, 0), (wl.L - 1, wl.H_kv - 1)]
    sampled = [0, 1, 3, 4, wl.n_seq - 1] if name == "ragged32" else sorted({0, wl.n_seq - 1})
    kept = {}
    for s, (tier, flag) in enumerate(routings):
        kept[s] = harness.fill_sequence(cache, wl, s, s, tier, flag, chunk=8192, keep=keep if s in sampled else [])
    keptq = dict(zip(sampled, kept_quantised(wl, [routings[s] for s in sampled], [kept[s] for s in sampled])))
    ids = list(range(wl.n_seq))
    q = gen.make_q(wl, device="cuda", gain=2.0)
    o = cache.decode_attention(-1, ids, q).double().cpu().numpy()
    l1 = wl.L - 1
    o_l = cache.decode_attention(l1, ids, q[:, l1].contiguous()).double().cpu().numpy()
    qn = f64(q)
    for s in sampled:
        tier, flag = routings[s]
        for (l, h) in keep:
            sl = slice(h * wl.G, (h + 1) * wl.G)
            o_ref, V, _ = oracle_slice_from_kept(wl, consts, tier, flag, keptq[s][(l, h)], qn[s, l, sl], l, h)
            check_output(o[s, l, sl], o_ref, float(np.abs(V).max()), f"i8 {name} seq {s} (l,h)=({l},{h})")
            if l == l1:
                check_output(o_l[s, sl], o_ref, float(np.abs(V).max()), f"i8 {name} per-layer seq {s} (l,h)=({l},{h})")
    assert cache.footprint()["used_bytes"] == sum(c8.footprint_bytes_i8(t, f, wl.tier_ranks, wl.d, wl.L, wl.H_kv) for t, f in routings)
    cache.destroy()


def test_option_errors(mod):
    binding, harness = mod
    wl = gen.WORKLOADS["tiny"]
    cache, _ = harness.make_cache(wl, n_seqs=1, max_tokens=64)
    tier = np.zeros(4, np.uint8); flag = np.zeros(4, np.uint8)
    cK, cV = gen.make_coef_chunk(wl, 0, 0, tier, device="cuda")
    cache.append_raw(0, tier, flag, cK, cV)
    with pytest.raises(binding.DwkvError) as e:
        cache.set_option("coef_int8", 1)                      # the format is fixed once tokens exist
    assert e.value.code == binding.DWKV_E_STATE
    cache.reset_seq(0)
    cache.set_option("coef_int8", 1)
    with pytest.raises(binding.DwkvError):
        cache.set_option("coef_int8", 2)
    cache.destroy()
    wl70 = dataclasses.replace(gen.WORKLOADS["llama70b_128k_b1"], L=4, T=(64,))
    cache, _ = harness.make_cache(wl70, n_seqs=1, max_tokens=64)
    cache.set_option("coef_int8", 1)                          # basis rank 48: two 32-column blocks per token vector
    tier = np.full(5, 2, np.uint8); flag = np.zeros(5, np.uint8)
    cK, cV = gen.make_coef_chunk(wl70, 0, 0, tier, device="cuda")
    cache.append_raw(0, tier, flag, cK, cV)
    assert cache.footprint()["used_bytes"] == 5 * 2 * (48 + 2) * wl70.L * wl70.H_kv
    cache.destroy()
