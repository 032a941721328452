"""GPU parity of the basis construction (dwkv_build_basis, reading A24) against oracle/dwkv_basis_oracle.py.

What is unique and compared: the energies the sketch has along the rows (its leading singular values), the subspaces spanned by
the leading r_t rows of every tier, orthonormality, the sign convention, and -- entry by entry -- the bf16 rows themselves
(the rows are unique up to the conditioning of the singular vectors: fp32 accumulation error divided by the relative gap)."""
import dataclasses

import numpy as np
import pytest
import torch

import gen
from oracle import dwkv_basis_oracle as bo
from oracle import dwkv_oracle as orc
from helpers import f64, check_output

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mod():
    from paper_2607_06523_b200 import binding, harness
    return binding, harness


def _dense(wl, n, consts):
    BK, BV, gK, gV = consts
    ks, vs = [], []
    for t0 in range(0, n, 4096):
        k, v = gen.make_dense_kv_chunk(wl, 0, t0, min(4096, n - t0), BK, BV, gK, gV, device="cuda")
        ks.append(k.contiguous()); vs.append(v.contiguous())
    return torch.cat(ks), torch.cat(vs)


SHAPES = {
    # name: (workload, n tokens, sketch rows)
    "tiny": (lambda: dataclasses.replace(gen.WORKLOADS["tiny"], T=(200,)), 200, 32),
    "8b_two_windows": (lambda: dataclasses.replace(gen.WORKLOADS["llama8b_16k_b8"], L=4, T=(1000,)), 1000, 48),   # token splits
    "70b_window4": (lambda: dataclasses.replace(gen.WORKLOADS["llama70b_128k_b1"], L=4, T=(520,)), 520, 64),
}


@pytest.mark.parametrize("umma", [0, 1])
@pytest.mark.parametrize("shape", list(SHAPES))
def test_build_basis_against_oracle(mod, shape, umma):
    """umma = 1: the tcgen05 sketch kernel (d = 128 shapes; the tiny d = 64 shape stays on mma.sync either way)."""
    binding, harness = mod
    mk, n, k = SHAPES[shape]
    wl = mk()
    cache, consts = harness.make_cache(wl, n_seqs=1, max_tokens=n + 64)
    cache.set_option("sketch_umma", umma)
    BK0, BV0, gK, gV = consts
    k_dense, v_dense = _dense(wl, n, consts)
    omega = gen.make_omega(wl, n, k, device="cuda")
    cache.build_basis(k_dense, v_dense, omega)
    BK, BV = cache.export_basis(wl.M, wl.H_kv, wl.r, wl.d)
    torch.cuda.synchronize()
    for z, (x, gate, got_t) in enumerate(((k_dense, gK, BK), (v_dense, gV, BV))):
        S = bo.sketch(f64(x), f64(gate), f64(omega), wl.w)                      # [M, H, k, d]
        want = bo.basis_from_sketch(S, wl.r)                                    # fp64, unrounded
        got = f64(got_t)
        n_off = 0
        for m in range(wl.M):
            for h in range(wl.H_kv):
                g, w_ = got[m, h], want[m, h]
                sig = np.linalg.svd(S[m, h], compute_uv=False)
                # orthonormal to bf16 rounding, energies = the leading singular values of the sketch
                assert np.abs(g @ g.T - np.eye(wl.r)).max() < 2.0 ** -6
                energy = np.linalg.norm(S[m, h] @ g.T, axis=0)
                assert np.allclose(energy, sig[:wl.r], rtol=2e-3), (shape, m, h)
                # the subspace of every tier's leading rows; a close pair of singular values at the cut makes it ill-conditioned
                for rk in wl.tier_ranks:
                    gap = (sig[rk - 1] - sig[rk]) / sig[rk - 1] if rk < len(sig) else 1.0
                    dist = np.linalg.norm(g[:rk].T @ g[:rk] - w_[:rk].T @ w_[:rk], 2)
                    assert dist < 2.0 ** -6 + 1e-4 / max(gap, 1e-6), (shape, m, h, rk, dist, gap)
                # sign convention (applied before the bf16 rounding): same orientation as the oracle's row, unless the two largest
                # magnitudes of that row nearly tie with opposite signs (then either orientation satisfies the rule to fp32 accuracy)
                for i in range(wl.r):
                    top2 = np.argsort(np.abs(w_[i]))[-2:]
                    near_tie = abs(abs(w_[i, top2[0]]) - abs(w_[i, top2[1]])) < 1e-3 * abs(w_[i, top2[1]])
                    if g[i] @ w_[i] < 0:
                        assert near_tie, (shape, m, h, i)
                        g[i] = -g[i]
                # entry by entry: one bf16 ulp of the rounded oracle row, except where neighbouring singular values nearly tie
                wb = orc.round_to_bf16(w_)
                ulp = np.maximum(np.abs(wb), 2.0 ** -10) * 2.0 ** -7
                relgap = np.minimum(np.abs(np.diff(sig[:wl.r + 1], prepend=np.inf)), np.abs(np.diff(sig[:wl.r + 1], append=0.0))[:wl.r + 1])[:wl.r] / sig[:wl.r]
                ok_rows = relgap > 1e-2
                n_off += int((np.abs(g - wb) > ulp)[ok_rows].sum())
        assert n_off <= 0.02 * got.size, (shape, z, n_off, got.size)
    cache.destroy()


def test_built_basis_serves_append_and_decode(mod):
    """The constructed basis is installed like dwkv_set_basis: append/compress and decode on it match the oracle fed with the exact
    bytes the cache holds (dwkv_export_basis); set_basis / build_basis are refused once tokens exist (reading A19)."""
    binding, harness = mod
    n = 256
    wl = dataclasses.replace(gen.WORKLOADS["tiny"], T=(n,))
    cache, consts = harness.make_cache(wl, n_seqs=1, max_tokens=n + 64)
    _, _, gK, gV = consts
    k_dense, v_dense = _dense(wl, n, consts)
    omega = gen.make_omega(wl, n, 32, device="cuda")
    cache.build_basis(k_dense, v_dense, omega)
    BK, BV = cache.export_basis(wl.M, wl.H_kv, wl.r, wl.d)
    tier, flag = gen.make_routing(wl, 0)
    cache.append_compress([0], [n], k_dense, v_dense, tier, flag)
    with pytest.raises(binding.DwkvError):
        cache.build_basis(k_dense, v_dense, omega)
    oc = orc.OracleCache(wl.L, wl.w, wl.H_kv, wl.G, wl.d, wl.tier_ranks, f64(BK), f64(BV), f64(gK), f64(gV))
    oc.append_compress(0, f64(k_dense), f64(v_dense), tier, flag)
    q = gen.make_q(wl, device="cuda", n_seq=1)
    out = cache.decode_attention(-1, [0], q).double().cpu().numpy()
    ref = oc.decode_all_layers([0], f64(q))
    for l in range(wl.L):
        check_output(out[0, l], ref[0, l], oc.max_abs_vhat(0, l), f"built basis layer {l}")
    # the built basis captures the planted low-rank part: the top-tier reconstruction error is the noise floor (0.05 per channel)
    for l in range(wl.L):
        for h in range(wl.H_kv):
            K, _ = oc.khat_vhat(0, l, h)
            top = (tier == len(wl.tier_ranks) - 1) & (flag == 0)
            err = np.abs(K[top] - f64(k_dense[:, l, h])[top]).std()
            assert err < 0.08, (l, h, err)
    cache.destroy()
