"""The int4 quantiser of dwkv_append_compress (step a4; reading A14) bit for bit against the oracle.

The general append tests allow a tiny fraction of codes to differ by one because the fp32 projection may land on the other side of a
bf16 rounding boundary than the oracle's fp64 one (reading A15 iii), which would also hide a rare error of the quantiser itself
(the kernel forms the quotient e / s with an approximate reciprocal and falls back to the IEEE division next to a rounding
boundary). Here the arithmetic in front of the quantiser is EXACT on both sides, so the residual e the quantiser sees is the same
fp32 number in the kernel and in the oracle, with ~18 significant bits and generic quotients: every code and every scale must match.

Construction: basis row j is non-zero on channels 4j .. 4j+3 only (disjoint supports, r * 4 = d), entries (1 + m/128) / 2, gates in
{1, 2}, x = +-(1 + m/128) * 2^k, k in {0, 1}: C_j = sum of four 16-bit products within a 20-bit span (exact in fp32 and fp64),
c = bf16(C) (one rounding, the same on both sides), rec_i = c_j * B_ji (one exact product), e_i = x_i - g_i * rec_i (17 bits)."""
import numpy as np
import pytest
import torch

from oracle import dwkv_oracle as orc
from helpers import f64

pytestmark = pytest.mark.gpu


def _bf16_grid(rng, shape, exps):
    m = rng.integers(0, 128, shape)
    k = rng.choice(exps, shape)
    return (1.0 + m / 128.0) * np.exp2(k)


@pytest.mark.parametrize("d,r,seed", [(128, 32, 0), (64, 16, 1)])
def test_append_quantiser_bit_exact_on_exact_residuals(d, r, seed):
    from paper_2607_06523_b200 import binding
    rng = np.random.default_rng(seed)
    L, w, H, G, T = 2, 1, 2, 1, 8192
    ranks = [8, r]
    B = np.zeros((2, L // w, H, r, d))
    for j in range(r):
        B[..., j, 4 * j:4 * j + 4] = _bf16_grid(rng, (2, L // w, H, 4), [-1]) * rng.choice([-1.0, 1.0], (2, L // w, H, 4))
    g = rng.choice([1.0, 2.0], (2, L, H, d))
    x = _bf16_grid(rng, (2, T, L, H, d), [0, 1]) * rng.choice([-1.0, 1.0], (2, T, L, H, d))
    dev = torch.device("cuda")
    bf = lambda a: torch.tensor(a, dtype=torch.float32).to(torch.bfloat16).to(dev).contiguous()
    BK, BV, gK, gV, k_new, v_new = bf(B[0]), bf(B[1]), bf(g[0]), bf(g[1]), bf(x[0]), bf(x[1])
    assert np.array_equal(f64(BK), B[0]) and np.array_equal(f64(k_new), x[0])           # the inputs are exact in bf16
    tier = rng.integers(0, 2, T).astype(np.uint8)
    flag = np.ones(T, np.uint8)
    cache = binding.DwkvCache(L, w, H, H * G, d, ranks, 1, T + 64)
    cache.set_basis(BK, BV); cache.set_gates(gK, gV)
    cache.append_compress([0], [T], k_new, v_new, tier, flag)
    oc = orc.OracleCache(L, w, H, G, d, tuple(ranks), B[0], B[1], g[0], g[1])
    oc.append_compress(0, x[0], x[1], tier, flag)
    dump = cache.export_tokens(0, 0, T)
    S = oc.seqs[0]
    n_half = 0
    for z in "KV":
        assert np.array_equal(dump["coef" + z].double().cpu().numpy(), S["c" + z])     # the projection is exact: same coefficients
        gc = dump["code" + z].cpu().numpy()
        lo = (gc & 15).astype(np.int8); hi = (gc >> 4).astype(np.int8)
        lo = np.where(lo > 7, lo - 16, lo); hi = np.where(hi > 7, hi - 16, hi)
        dec = np.stack([lo, hi], axis=-1).reshape(S["code" + z].shape)
        assert np.array_equal(dump["scale" + z].cpu().numpy().view(np.uint16), S["scale" + z].view(np.uint16)), z
        bad = np.argwhere(dec != S["code" + z])
        assert bad.size == 0, (z, len(bad), bad[:5])
        n_half += int((np.abs(S["code" + z]) >= 1).sum())
    assert n_half > 0.5 * 2 * T * L * H * d                                             # the case is not degenerate: most codes are non-zero
    cache.destroy()
