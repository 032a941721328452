"""GPU parity of the opt-in variants of the per-layer call path (option "fuse_combine"): 1 = the split-combine (SURVEY.md section 8a
step a3) fused into the decode kernel as a last-arrival epilogue (one launch per `dwkv_decode_attention(layer = l)`
"during decoding, the fused kernel ..." is a per-layer operation), 2 = CTA-level merge of the partials + the combine kernel.
Compared with the oracle, with the default separate-combine path, and with itself across repeated calls. Both variants measured
slower than the default, so they stay options."""
import dataclasses

import numpy as np
import pytest
import torch

import gen
from helpers import rel_l2
from test_gpu_parity import load, compare, all_lh

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mod():
    from paper_2607_06523_b200 import binding, harness
    return binding, harness


def per_layer(cache, wl, ids, q):
    return torch.stack([cache.decode_attention(l, ids, q[:, l].contiguous()) for l in range(wl.L)], dim=1)


@pytest.mark.parametrize("name", ["tiny", "extremes", "8b_ragged", "70b_full_mode", "d64_g3"])
def test_fused_per_layer_against_oracle_and_unfused(mod, name):
    binding, harness = mod
    keep = None
    if name == "tiny":
        wl = gen.WORKLOADS["tiny"]
    elif name == "extremes":      # T = 1 and tiny sequences: segments with a single contributor, many segments per slice
        wl = dataclasses.replace(gen.WORKLOADS["tiny"], T=(1, 300, 45, 2, 131, 512, 17), patterns=("", "all_low", "all_top_flag", "", "alternating", "", ""))
    elif name == "8b_ragged":     # segments of several hundred KB: the CTAs of the persistent grid straddle segment boundaries
        wl = dataclasses.replace(gen.WORKLOADS["llama8b_16k_b8"], L=2, T=(9000, 1237, 4100))
        keep = [(0, 0), (1, 3), (1, 7), (0, 5)]
    elif name == "70b_full_mode":
        wl = dataclasses.replace(gen.WORKLOADS["llama70b_128k_b1"], L=4, T=(5000,))
        keep = [(0, 1), (3, 6), (2, 0)]
    else:
        wl = dataclasses.replace(gen.WORKLOADS["tiny"], G=3, tier_ranks=(16, 24), T=(700, 70))
    routings = [gen.make_routing(wl, s) for s in range(wl.n_seq)]
    cache, consts, kept = load(harness, wl, routings, keep=keep, chunk=1500)
    ids = list(range(wl.n_seq))
    for gain in (1.0, 16.0):
        q = gen.make_q(wl, device="cuda", gain=gain)
        cache.set_option("fuse_combine", 1)
        out_f = per_layer(cache, wl, ids, q)
        assert cache.get_stat("plan_fused") == 1.0
        compare(wl, cache, consts, kept, routings, q, out_f, lhs=keep, what=f"{name} fused per-layer gain {gain}")
        out_f2 = per_layer(cache, wl, ids, q)                      # counters were reset by the finishing CTAs; merge order is fixed
        assert torch.equal(out_f, out_f2)
        cache.set_option("fuse_combine", 0)
        out_u = per_layer(cache, wl, ids, q)
        assert cache.get_stat("plan_fused") == 0.0
        assert rel_l2(out_f.cpu().numpy(), out_u.cpu().numpy()) < 2e-3
        cache.set_option("fuse_combine", 2)                        # CTA-level merge of the partials + the separate combine kernel
        out_c = per_layer(cache, wl, ids, q)
        compare(wl, cache, consts, kept, routings, q, out_c, lhs=keep, what=f"{name} CTA-merge per-layer gain {gain}")
        cache.set_option("fuse_combine", 1)                        # fused epilogue on an all-layer call
        out_a = cache.decode_attention(-1, ids, q)
        compare(wl, cache, consts, kept, routings, q, out_a, lhs=keep, what=f"{name} fused all-layers gain {gain}")
    cache.set_option("fuse_combine", 0)
    cache.destroy()


def test_fused_per_layer_coef_int8(mod):
    binding, harness = mod
    from test_gpu_coef8 import load8, kept_quantised
    wl = dataclasses.replace(gen.WORKLOADS["tiny"], T=(700, 33))
    routings = [gen.make_routing(wl, s) for s in range(2)]
    cache, consts, kept = load8(harness, wl, routings)
    q = gen.make_q(wl, device="cuda", gain=3.0)
    cache.set_option("fuse_combine", 1)
    out = per_layer(cache, wl, [0, 1], q)
    assert cache.get_stat("plan_fused") == 1.0
    compare(wl, cache, consts, kept_quantised(wl, routings, kept), routings, q, out, what="i8 fused per-layer")
    cache.destroy()


def test_fused_slice_counts(mod):
    """Fewer slices per CTA (n_slices = 148 * k) and a single CTA's worth of slices give the same result to rounding level."""
    binding, harness = mod
    wl = dataclasses.replace(gen.WORKLOADS["llama8b_16k_b8"], L=2, T=(6000, 800))
    routings = [gen.make_routing(wl, s) for s in range(2)]
    keep = [(1, 2), (0, 6)]
    cache, consts, kept = load(harness, wl, routings, keep=keep, chunk=1500)
    q = gen.make_q(wl, device="cuda", gain=2.0)
    cache.set_option("fuse_combine", 1)
    outs = []
    for ns in (0, 148, 444, 1184):
        cache.set_option("n_slices", ns)
        outs.append(per_layer(cache, wl, [0, 1], q))
        if ns:
            assert cache.get_stat("plan_slices") == ns
        compare(wl, cache, consts, kept, routings, q, outs[-1], lhs=keep, what=f"fused n_slices {ns}")
    for o in outs[1:]:
        assert rel_l2(o.cpu().numpy(), outs[0].cpu().numpy()) < 1e-3
    cache.destroy()


def test_two_handles_two_streams_interleaved(mod):
    """Two caches on one device, their calls interleaved on two streams (per-device kernel attributes, per-handle scratch)."""
    binding, harness = mod
    wl = dataclasses.replace(gen.WORKLOADS["tiny"], T=(400,))
    routings = [gen.make_routing(wl, 0)]
    c1, consts, kept = load(harness, wl, routings)
    c2, _, _ = load(harness, wl, routings)
    q = gen.make_q(wl, device="cuda", gain=2.0)
    ref = c1.decode_attention(-1, [0], q)
    torch.cuda.synchronize()
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    outs1, outs2 = [], []
    for it in range(6):
        with torch.cuda.stream(s1):
            outs1.append(c1.decode_attention(-1 if it % 2 else it % wl.L, [0], q if it % 2 else q[:, it % wl.L].contiguous()))
        with torch.cuda.stream(s2):
            outs2.append(c2.decode_attention(it % wl.L if it % 2 else -1, [0], q[:, it % wl.L].contiguous() if it % 2 else q))
    torch.cuda.synchronize()
    for it in range(6):
        a, b = (outs1[it], outs2[it]) if it % 2 else (outs2[it], outs1[it])          # a: all-layer call, b: per-layer call
        assert torch.equal(a, ref)
        assert rel_l2(b.cpu().numpy(), ref[:, it % wl.L].cpu().numpy()) < 2e-3
    compare(wl, c2, consts, kept, routings, q, outs2[0], what="second handle")
    c1.destroy(); c2.destroy()
