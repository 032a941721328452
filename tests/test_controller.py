"""Probe-driven controller and router attention features (reading A28): pins of the oracle, and -- the
controller is host-only code, so this runs without a GPU -- bit-exact parity of the C-ABI functions dwkv_controller_* with it."""
import numpy as np
import pytest
import torch

from oracle import dwkv_controller_oracle as co


# ---- oracle pins -----------------------------------------------------------------------------------------------------
def test_token_stats_closed_forms():
    rng = np.random.default_rng(0)
    K = rng.standard_normal((37, 16))
    # q = 0: uniform attention -> every token gets 1/T from every head
    p = co.attention_probs(np.zeros((6, 16)), K, 0.25)
    mass, spike = co.token_stats(p)
    np.testing.assert_allclose(mass, 6 / 37, rtol=1e-14); np.testing.assert_allclose(spike, 1 / 37, rtol=1e-14)
    # T = 1: the token takes everything
    mass, spike = co.token_stats(co.attention_probs(rng.standard_normal((5, 16)), K[:1], 0.25))
    assert mass.tolist() == [5.0] and spike.tolist() == [1.0]
    # probabilities of a head sum to one -> the masses sum to the number of heads; spike <= mass <= H_q * spike
    q = rng.standard_normal((4, 16)) * 3
    p = co.attention_probs(q, K, 0.25)
    mass, spike = co.token_stats(p)
    assert abs(mass.sum() - 4.0) < 1e-12 and np.all(spike <= mass + 1e-15) and np.all(mass <= 4 * spike + 1e-15)
    # against a library routine
    ref = torch.softmax(torch.tensor(q @ K.T * 0.25, dtype=torch.float64), dim=-1).numpy()
    np.testing.assert_allclose(p, ref, rtol=1e-12, atol=1e-15)
    # one dominant token: a key aligned with a large query takes (almost) all of that head's mass
    K2 = K.copy(); K2[11] = 10.0 * q[2] / np.linalg.norm(q[2])
    mass2, spike2 = co.token_stats(co.attention_probs(q * 4, K2, 0.25))
    assert np.argmax(spike2) == 11 and spike2[11] > 0.999
    # token permutation permutes the statistics
    perm = rng.permutation(37)
    m3, s3 = co.token_stats(co.attention_probs(q, K[perm], 0.25))
    np.testing.assert_allclose(m3, mass[perm], rtol=1e-12); np.testing.assert_allclose(s3, spike[perm], rtol=1e-12)


def test_controller_hand_trace():
    """tol 0.03, step_down 0.5, step_up 0.25, patience 3, delta in [-1.25, 0.5]; two windows. Expected states written by hand."""
    c = co.Controller(2, 0.03, 0.5, 0.25, 3, -1.25, 0.5)
    trace = [
        # (windows, errors)                         delta after            quiet after
        (([0, 0, 1], [0.01, 0.05, 0.02]),           [-0.5, 0.0],           [0, 1]),     # window 0: max 0.05 > tol -> down; window 1 quiet
        (([0, 1], [0.031, 0.03]),                   [-1.0, 0.0],           [0, 2]),     # 0.03 is NOT above the tolerance (strict)
        (([0], [0.2]),                              [-1.25, 0.0],          [0, 2]),     # clamped at delta_min; window 1 not probed: untouched
        (([1], [0.0]),                              [-1.25, 0.25],         [0, 0]),     # third quiet interval of window 1 -> up
        (([0, 1], [0.0, 0.0]),                      [-1.25, 0.25],         [1, 1]),
        (([0, 1], [0.0, 0.0]),                      [-1.25, 0.25],         [2, 2]),
        (([0, 1], [0.0, 0.0]),                      [-1.0, 0.5],           [0, 0]),     # both up; window 1 reaches delta_max
        (([1, 1, 1], [0.0, 0.0, 0.0]),              [-1.0, 0.5],           [0, 1]),     # several probes of one interval count once
        (([1], [0.0]),                              [-1.0, 0.5],           [0, 2]),
        (([1], [0.0]),                              [-1.0, 0.5],           [0, 0]),     # clamped at delta_max
        (([1], [1.0]),                              [-1.0, 0.0],           [0, 0]),
    ]
    for (w, e), delta, quiet in trace:
        c.step(w, e)
        assert c.delta.tolist() == delta and c.quiet.tolist() == quiet, (w, e, c.delta, c.quiet)
    tau, tf = c.thresholds([0.5, 2.0], 1.5)            # min_m delta_m = -1.0
    assert tau.tolist() == [-0.5, 1.0] and float(tf) == 0.5


def test_controller_window_specific_tolerance_and_rounding():
    c = co.Controller(3, [0.01, 0.1, 1.0], 0.1, 0.1, 1, -10.0, 10.0)
    c.step([0, 1, 2], [0.05, 0.05, 0.05])
    f = np.float32
    assert c.delta.tolist() == [f(0) - f(0.1), f(0.1), f(0.1)]
    d = f(0) - f(0.1)
    for _ in range(9):
        c.step([0], [1.0])
        d = f(d - f(0.1))                               # fp32, one rounding per step
    assert c.delta[0] == d and c.delta[0] != f(-1.0)    # ten fp32 steps of 0.1 do not land on -1 exactly


# ---- the library's controller against the oracle (host-only: no GPU needed) ------------------------------------------
@pytest.fixture(scope="module")
def binding():
    import __graft_entry__ as entry
    entry.build()
    from paper_2607_06523_b200 import binding as b
    return b


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_library_controller_bit_exact(binding, seed):
    rng = np.random.default_rng(seed)
    M = int(rng.integers(1, 20))
    tol = rng.uniform(0.01, 0.06, M).astype(np.float32) if seed else 0.03
    args = (float(np.float32(rng.uniform(0.05, 0.7))), float(np.float32(rng.uniform(0.05, 0.4))), int(rng.integers(1, 5)),
            float(np.float32(-rng.uniform(0.5, 3))), float(np.float32(rng.uniform(0.2, 2))))
    ref = co.Controller(M, tol, *args)
    lib = binding.Controller(M, tol, *args)
    for it in range(200):
        n = int(rng.integers(0, 3 * M))
        w = rng.integers(0, M, n).astype(np.int32)
        e = (rng.uniform(0, 0.08, n) * rng.choice([0.2, 1.0, 3.0], n)).astype(np.float32)
        ref.step(w, e); lib.step(w, e)
        d, q = lib.state()
        assert np.array_equal(d.view(np.uint32), ref.delta.view(np.uint32)) and np.array_equal(q, ref.quiet), it
        base = np.sort(rng.standard_normal(2)).astype(np.float32); bf = float(np.float32(rng.standard_normal()))
        tau, tf = lib.thresholds(base, bf)
        tau_o, tf_o = ref.thresholds(base, bf)
        assert np.array_equal(tau.view(np.uint32), tau_o.view(np.uint32)) and np.float32(tf).view(np.uint32) == np.float32(tf_o).view(np.uint32)
    lib.destroy()


def test_library_controller_errors(binding):
    with pytest.raises(binding.DwkvError):
        binding.Controller(0, 0.03, 0.5, 0.25, 3, -1.0, 1.0)
    with pytest.raises(binding.DwkvError):
        binding.Controller(2, 0.03, -0.5, 0.25, 3, -1.0, 1.0)            # negative step
    with pytest.raises(binding.DwkvError):
        binding.Controller(2, 0.03, 0.5, 0.25, 3, 1.0, 2.0)              # delta_min > 0
    c = binding.Controller(2, 0.03, 0.5, 0.25, 3, -1.0, 1.0)
    with pytest.raises(binding.DwkvError):
        c.step([2], [0.1])                                               # window out of range
    with pytest.raises(binding.DwkvError):
        c.step([0], [float("nan")])
    d, q = c.state()
    assert d.tolist() == [0.0, 0.0] and q.tolist() == [0, 0]             # state untouched by the failed calls
    c.destroy()
