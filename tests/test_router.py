"""Router (Eq. 2, reading A26): pins of the oracle and -- the router is host-only code, so this runs without a
GPU -- bit-exact parity of the C-ABI functions dwkv_route_tokens / dwkv_router_thresholds with it."""
import numpy as np
import pytest

from oracle import dwkv_router_oracle as ro


def test_oracle_hand_example():
    """u = (1, 2, 0, -1); phi rows chosen so z = 3, -1, 0.5, 2; thresholds 0 and 2.5 (logit space), flag threshold 1.9."""
    u = [1.0, 2.0, 0.0, -1.0]
    phi = np.array([[1, 1, 9, 0], [0, 0, 9, 1], [0.5, 0, 9, 0], [0, 1.5, 9, 1]], np.float32)
    assert np.array_equal(ro.logits(phi, u), np.array([3.0, -1.0, 0.5, 2.0], np.float32))
    tier, flag = ro.route(phi, u, [0.0, 2.5], 1.9)
    assert tier.tolist() == [2, 0, 1, 1] and flag.tolist() == [1, 0, 0, 1]
    # strict comparison: a token exactly at a threshold stays below it
    tier, _ = ro.route(phi, u, [0.5, 3.0], 0.0)
    assert tier.tolist() == [1, 0, 0, 1]


def test_oracle_thresholds_route_the_requested_fractions():
    rng = np.random.default_rng(0)
    n = 1000
    phi = rng.standard_normal((n, 4)).astype(np.float32); u = np.array([0.7, -1.1, 0.3, 2.0], np.float32)
    tau, tf = ro.thresholds(phi, u, [0.65, 0.25, 0.10], 0.08)
    tier, flag = ro.route(phi, u, tau, tf)
    assert len(np.unique(ro.logits(phi, u))) == n                       # distinct scores: counts are exact
    assert (tier == 2).sum() == int(np.ceil(n * float(np.float32(0.10))))
    assert (tier >= 1).sum() == int(np.ceil(n * (float(np.float32(0.25)) + float(np.float32(0.10)))))
    assert flag.sum() == int(np.ceil(n * float(np.float32(0.08))))
    assert np.all(flag <= (tier == 2))                                   # 8 % flagged lie inside the 10 % top tier
    # monotone in the score: a higher score never gets a lower tier
    z = ro.logits(phi, u); order = np.argsort(z)
    assert np.all(np.diff(tier[order].astype(int)) >= 0)
    # degenerate budgets
    tau0, tf0 = ro.thresholds(phi, u, [1.0, 0.0, 0.0], 0.0)
    assert np.all(np.isposinf(tau0)) and np.isposinf(tf0) and ro.route(phi, u, tau0, tf0)[0].max() == 0
    tau1, tf1 = ro.thresholds(phi, u, [0.0, 0.0, 1.0], 1.0)
    assert np.all(np.isneginf(tau1)) and ro.route(phi, u, tau1, tf1)[1].min() == 1


@pytest.fixture(scope="module")
def binding():
    import __graft_entry__ as entry
    entry.build()
    from paper_2607_06523_b200 import binding as b
    return b


@pytest.mark.parametrize("n,n_tiers", [(1, 3), (17, 2), (4096, 3), (50000, 4), (333, 1)])
def test_library_router_bit_exact(binding, n, n_tiers):
    rng = np.random.default_rng(n)
    phi = (rng.standard_normal((n, 4)) * rng.choice([1e-3, 1.0, 50.0], size=(n, 1))).astype(np.float32)
    phi[:, 2] = rng.integers(0, 2, n)                                     # the boundary indicator is 0 / 1
    u = rng.standard_normal(4).astype(np.float32)
    frac = rng.dirichlet(np.ones(n_tiers)).astype(np.float32)
    flag_frac = float(rng.uniform(0, frac[-1]))
    tau, tf = binding.router_thresholds(phi, u, frac, flag_frac)
    tau_o, tf_o = ro.thresholds(phi, u, frac, flag_frac)
    assert np.array_equal(tau.view(np.uint32), tau_o.view(np.uint32)) and np.float32(tf).view(np.uint32) == np.float32(tf_o).view(np.uint32)
    tier, flag = binding.route_tokens(phi, u, tau, tf, n_tiers)
    tier_o, flag_o = ro.route(phi, u, tau_o, tf_o)
    assert np.array_equal(tier, tier_o) and np.array_equal(flag, flag_o)


def test_library_router_errors(binding):
    phi = np.zeros((4, 4), np.float32); u = np.ones(4, np.float32)
    with pytest.raises(binding.DwkvError):
        binding.route_tokens(phi, u, [1.0, 0.0], 0.0, 3)                  # thresholds must ascend
    with pytest.raises(binding.DwkvError):
        binding.route_tokens(phi, u, [0.0] * 4, 0.0, 5)                   # more tiers than DWKV_MAX_TIERS
    with pytest.raises(binding.DwkvError):
        binding.router_thresholds(phi, u, [0.5, 1.5], 0.0)                # fractions in [0, 1]
