"""Two handles on one device, their calls interleaved on two streams: per-device kernel attributes, per-handle scratch and plans
(round-1 review, hardening)."""
import dataclasses

import pytest
import torch

import gen
from helpers import rel_l2
from test_gpu_parity import load, compare

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mod():
    from paper_2607_06523_b200 import binding, harness
    return binding, harness


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
