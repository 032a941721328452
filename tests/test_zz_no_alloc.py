"""dwkv_dense_decode_attention_static (include/dwkv.h): the allocation-free variant of the dense comparison kernel, its split-T
partial records in a file-scope device array of DWKV_DENSE_STATIC_SCRATCH_BYTES instead of a caller workspace. Checked against the
existing path (dwkv_dense_decode_attention with a torch-allocated workspace) on calls in a row that share the array, within the
tolerance of the other GPU tests (helpers.check_output; the two paths launch the same kernels with the same split, so the
outputs are in fact expected to be bit-identical, which is asserted too). This file is collected last on purpose (pytest -x)."""
import numpy as np
import pytest
import torch

from helpers import check_output

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def binding():
    from paper_2607_06523_b200 import binding as b
    return b


def _inputs(shape, seed):
    n_seq, L, H, G, d, T = shape
    g = torch.Generator(device="cuda").manual_seed(seed)
    K = (torch.randn(n_seq, L, H, T, d, device="cuda", generator=g) * 0.3).to(torch.bfloat16)
    V = (torch.randn(n_seq, L, H, T, d, device="cuda", generator=g) * 0.3).to(torch.bfloat16)
    q = (torch.randn(n_seq, L, H * G, d, device="cuda", generator=g) * 2).to(torch.bfloat16)
    return K, V, q


def test_static_scratch_matches_workspace_path_on_calls_in_a_row(binding):
    # a large call first, then smaller ones of other shapes over the array's stale contents, then the first again
    shapes = [(2, 4, 2, 4, 128, 3000), (1, 1, 2, 8, 128, 77), (1, 2, 2, 2, 64, 515), (2, 4, 2, 4, 128, 3000)]
    cases = []
    for i, shape in enumerate(shapes):
        K, V, q = _inputs(shape, seed=i % 3)
        ref = binding.dense_decode_attention(K, V, q, shape[2])                 # existing path, workspace from torch
        out = torch.full(q.shape, float("nan"), dtype=torch.float32, device="cuda")
        cases.append((shape, K, V, q, ref, out))
    torch.cuda.synchronize()
    K, V, q = cases[0][1:4]
    binding.dense_decode_attention_static(K, V, q, shapes[0][2], cases[0][5])   # first call on this device: resolves the address
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for shape, K, V, q, ref, out in cases:                                      # back to back on one stream, no sync in between
        binding.dense_decode_attention_static(K, V, q, shape[2], out)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0                                # no device memory was taken or returned
    for shape, K, V, q, ref, out in cases:
        check_output(out.double().cpu().numpy(), ref.double().cpu().numpy(), float(V.float().abs().max()), f"static {shape}")
        assert torch.equal(out, ref), shape                                     # same kernels, same split: bit-identical


def test_static_scratch_rejects_calls_beyond_its_size(binding):
    # 1776 (sequence, layer, kv head) rows x 1 split x G = 8 x 130 floats = 7.4 MB fits; 2 x that many rows does not fit in 16 MiB
    # (pointers are never dereferenced: the size check comes first)
    d, G, H = 128, 8, 8
    assert binding.DENSE_STATIC_SCRATCH_BYTES == 16 << 20
    K = torch.empty(1, dtype=torch.bfloat16, device="cuda")
    o = torch.empty(1, dtype=torch.float32, device="cuda")
    lib, vp = binding.lib, lambda t: t.data_ptr()
    n_layers = 5000 // H                                                        # n_lhb = 5000 -> 1 split each, 5000 * 8 * 130 * 4 = 20.8 MB
    rc = lib.dwkv_dense_decode_attention_static(vp(K), vp(K), vp(K), vp(o), 1, n_layers, H, H * G, d, 64, 0.0, None)
    assert rc != 0
    msg = lib.dwkv_last_error().decode()
    assert str(n_layers * H * G * (2 + d) * 4) in msg and str(16 << 20) in msg, msg
    with pytest.raises(binding.DwkvError):
        binding.dense_decode_attention_static(torch.empty(1, 1, 2, 16, 96, dtype=torch.bfloat16, device="cuda"),
                                              torch.empty(1, 1, 2, 16, 96, dtype=torch.bfloat16, device="cuda"),
                                              torch.empty(1, 1, 4, 96, dtype=torch.bfloat16, device="cuda"), 2,
                                              torch.empty(1, 1, 4, 96, dtype=torch.float32, device="cuda"))          # d_head 96
    # the entry point still works after the refused calls
    shape = (1, 1, 2, 4, 64, 300)
    K, V, q = _inputs(shape, seed=5)
    ref = binding.dense_decode_attention(K, V, q, 2)
    out = binding.dense_decode_attention_static(K, V, q, 2, torch.empty_like(ref))
    torch.cuda.synchronize()
    assert torch.equal(out, ref)
