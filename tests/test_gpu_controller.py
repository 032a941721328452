"""GPU parity of the router's attention features (dwkv_probe_token_stats) and the closed control loop of PAPER.md:58-72
(SURVEY.md section 8f NEXT-3 -> NEXT-4): append -> probe statistics + Eq. (3) probe error on the GPU -> controller -> thresholds ->
router -> the next append, with the routing decisions bit-exact against the oracles and the floating-point quantities within the
stated tolerances."""
import dataclasses

import numpy as np
import pytest
import torch

import gen
from oracle import dwkv_controller_oracle as co
from oracle import dwkv_oracle as orc
from oracle import dwkv_router_oracle as ro
from helpers import f64
from test_gpu_parity import load

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mod():
    from paper_2607_06523_b200 import binding, harness
    return binding, harness


def oracle_from_kept(wl, consts, routings, kept):
    """Oracle cache holding exactly what the GPU cache was loaded with (the generator outputs kept on the host)."""
    BK, BV, gK, gV = consts
    oc = orc.OracleCache(wl.L, wl.w, wl.H_kv, wl.G, wl.d, wl.tier_ranks, f64(BK), f64(BV), f64(gK), f64(gV))
    for s, (tier, flag) in enumerate(routings):
        T, nf = len(tier), int(flag.sum())
        c = {z: np.zeros((T, wl.L, wl.H_kv, wl.r)) for z in "KV"}
        r = {z: np.zeros((nf, wl.L, wl.H_kv, wl.d), np.float32) for z in "KV"}
        for (l, h), k in kept[s].items():
            for z in "KV":
                c[z][:, l, h] = f64(k["c" + z])
                if nf:
                    r[z][:, l, h] = k["r" + z].numpy()
        oc.append_raw(s, tier, flag, c["K"], c["V"], residK=r["K"] if nf else None, residV=r["V"] if nf else None)
    return oc


def oracle_stats(oc, wl, seq, layer, q_l):
    """mass, spike of all tokens of `seq` for the query vector q_l [H_q, d] of one layer, from the oracle's K-hat."""
    p = np.zeros((wl.H_q, oc.seq_len(seq)))
    for h in range(wl.H_kv):
        K, _ = oc.khat_vhat(seq, layer, h)
        p[h * wl.G:(h + 1) * wl.G] = co.attention_probs(q_l[h * wl.G:(h + 1) * wl.G], K, oc.scale)
    return co.token_stats(p)


@pytest.mark.parametrize("name", ["tiny", "extremes", "g8_d128", "tiny_i8"])
def test_token_stats_against_oracle(mod, name):
    binding, harness = mod
    i8 = name.endswith("_i8")
    if name.startswith("tiny"):
        wl = gen.WORKLOADS["tiny"]
    elif name == "extremes":
        wl = dataclasses.replace(gen.WORKLOADS["tiny"], T=(1, 300, 77), patterns=("", "all_top_flag", "alternating"))
    else:
        wl = dataclasses.replace(gen.WORKLOADS["llama70b_128k_b1"], L=4, T=(700,))
    routings = [gen.make_routing(wl, s) for s in range(wl.n_seq)]
    if i8:
        from test_gpu_coef8 import load8, kept_quantised
        cache, consts, kept = load8(harness, wl, routings)
        kept = kept_quantised(wl, routings, kept)          # the cache holds the 8-bit quantisation of the generator's coefficients (A27)
    else:
        cache, consts, kept = load(harness, wl, routings, chunk=4096)
    oc = oracle_from_kept(wl, consts, routings, kept)
    for s in range(wl.n_seq):
        T = wl.T[s]
        mass = torch.zeros(T, dtype=torch.float32, device="cuda"); spike = torch.zeros_like(mass)
        ref_mass = np.zeros(T); ref_spike = np.zeros(T)
        for step, (layer, gain) in enumerate([(0, 1.0), (wl.L - 1, 8.0), (0, 1.0)]):
            q = gen.make_q(wl, step=step, device="cuda", gain=gain)[s, layer].contiguous()
            cache.probe_token_stats(layer, s, q, mass, spike)
            m, sp = oracle_stats(oc, wl, s, layer, f64(q))
            ref_mass += m; ref_spike = np.maximum(ref_spike, sp)
        torch.cuda.synchronize()
        gm, gs = mass.double().cpu().numpy(), spike.double().cpu().numpy()
        assert abs(gm.sum() - 3 * wl.H_q) < 1e-3 * wl.H_q                  # every head's probabilities sum to one, three probes
        assert np.all(gs <= gm + 1e-6) and np.all(gs <= 1 + 1e-5)
        np.testing.assert_allclose(gm, ref_mass, rtol=3e-3, atol=1e-7)
        np.testing.assert_allclose(gs, ref_spike, rtol=3e-3, atol=1e-7)
    cache.destroy()


def test_closed_loop_append_probe_controller_route(mod):
    """Four probe intervals on a cache with two depth windows: the router's thresholds move with the measured probe error and the
    routed (tier, flag) of every new token equals the oracles' decision bit for bit."""
    binding, harness = mod
    wl = dataclasses.replace(gen.WORKLOADS["tiny"], L=4, w=2, T=(0,))
    cache, consts = harness.make_cache(wl, n_seqs=1, max_tokens=512)
    BK, BV, gK, gV = consts
    oc = orc.OracleCache(wl.L, wl.w, wl.H_kv, wl.G, wl.d, wl.tier_ranks, f64(BK), f64(BV), f64(gK), f64(gV))
    M = wl.L // wl.w
    ctl_args = (0.05, 1.0, 0.5, 2, -3.0, 1.0)                      # tolerance, step_down, step_up, patience, delta bounds
    ctl = binding.Controller(M, *ctl_args)
    ctl_o = co.Controller(M, *ctl_args)
    u = np.array([40.0, 25.0, 1.5, 20.0], np.float32)             # synthetic router parameter (the learned one needs training data)
    base_tau, base_flag = np.array([1.2], np.float32), 2.0         # two tiers: one tier threshold + the flag threshold (logit space)
    n_new, Tmax = 24, 24 * 5
    mass = torch.zeros(Tmax, dtype=torch.float32, device="cuda"); spike = torch.zeros_like(mass)
    mass_o = np.zeros(Tmax); spike_o = np.zeros(Tmax)
    k_all, v_all = [], []
    e_prev = 0.0
    deltas = []
    for it in range(5):
        T0 = cache.seq_len(0)
        # features of the new tokens (the caller's business: the router takes phi as an input): local attention mass / spike of the
        # most recent cached tokens, a synthetic boundary indicator, the previous interval's probe error
        mh, sh = mass[:max(T0, 1)].cpu().numpy(), spike[:max(T0, 1)].cpu().numpy()
        phi = np.zeros((n_new, 4), np.float32)
        phi[:, 0] = mh[-8:].mean() if T0 else 0.0
        phi[:, 1] = sh[-8:].max() if T0 else 0.0
        phi[:, 2] = (np.arange(T0, T0 + n_new) % 6 == 0)
        phi[:, 3] = e_prev
        phi[:, 0] += np.linspace(0, 0.02, n_new, dtype=np.float32)           # distinct scores
        tau, tf = ctl.thresholds(base_tau, base_flag)
        tau_o, tf_o = ctl_o.thresholds(base_tau, base_flag)
        assert np.array_equal(tau, tau_o) and np.float32(tf) == np.float32(tf_o)
        tier, flag = binding.route_tokens(phi, u, tau, tf, 2)
        tier_o, flag_o = ro.route(phi, u, tau_o, tf_o)
        assert np.array_equal(tier, tier_o) and np.array_equal(flag, flag_o)          # routing bit-exact
        k_new, v_new = gen.make_dense_kv_chunk(wl, 0, T0, n_new, BK, BV, gK, gV, device="cuda")
        k_new, v_new = k_new.contiguous(), v_new.contiguous()
        cache.append_compress([0], [n_new], k_new, v_new, tier, flag)
        oc.append_compress(0, f64(k_new), f64(v_new), tier_o, flag_o)
        k_all.append(k_new); v_all.append(v_new)
        T = T0 + n_new
        exp = cache.export_tokens(0, 0, T, want=("tier", "flag", "slot"))
        assert np.array_equal(exp["tier"].cpu().numpy(), oc.seqs[0]["tier"]) and np.array_equal(exp["slot"].cpu().numpy(), oc.seqs[0]["slot"])
        # probe interval: statistics of every layer, Eq. (3) error of one layer per window against the dense originals
        q = gen.make_q(wl, step=it, device="cuda", gain=4.0)
        for l in range(wl.L):
            cache.probe_token_stats(l, 0, q[0, l].contiguous(), mass, spike)
            m, sp = oracle_stats(oc, wl, 0, l, f64(q[0, l]))
            mass_o[:T] += m; spike_o[:T] = np.maximum(spike_o[:T], sp)
        # (the GPU's append rounds a few coefficients to the neighbouring bf16 value, reading A15 iii: a per-token score difference of
        #  that size, not of the statistics kernel -- its own parity, on identical bytes, is the 3e-3 of the test above)
        np.testing.assert_allclose(mass[:T].double().cpu().numpy(), mass_o[:T], rtol=3e-2, atol=1e-6)
        np.testing.assert_allclose(spike[:T].double().cpu().numpy(), spike_o[:T], rtol=3e-2, atol=1e-6)
        K_all, V_all = torch.cat(k_all), torch.cat(v_all)                    # [T, L, H, d] bf16: the "higher-fidelity cache"
        windows, errs, errs_o = [], [], []
        for l in (0, 3):
            qp = q[:, l].contiguous()                                         # one probed query position [1, H_q, d]
            e = cache.probe_error(l, 0, qp, K_all[:, l].permute(1, 0, 2).contiguous(), V_all[:, l].permute(1, 0, 2).contiguous(), eps=1e-6)
            ref = np.zeros((1, wl.H_q, wl.d)); cmp_ = np.zeros_like(ref)
            for h in range(wl.H_kv):
                sl = slice(h * wl.G, (h + 1) * wl.G)
                ref[0, sl] = orc.softmax_attention(f64(qp)[0, sl], f64(K_all[:, l, h]), f64(V_all[:, l, h]), oc.scale)
                Kh, Vh = oc.khat_vhat(0, l, h)
                cmp_[0, sl] = orc.softmax_attention(f64(qp)[0, sl], Kh, Vh, oc.scale)
            e_o = orc.probe_error(ref, cmp_, wl.G, 1e-6)
            e = e.cpu().numpy()
            np.testing.assert_allclose(e, e_o, rtol=5e-2, atol=1e-4)
            windows += [l // wl.w] * wl.H_kv; errs += e.tolist(); errs_o += e_o.tolist()
        # the controller's input is the measured error: both controllers see the GPU's numbers -> bit-exact state
        ctl.step(windows, errs); ctl_o.step(windows, errs)
        d, qt = ctl.state()
        assert np.array_equal(d, ctl_o.delta) and np.array_equal(qt, ctl_o.quiet)
        # and every measured error lies on the same side of the tolerance as the oracle's own value (unless that sits within 10 % of it)
        assert all((x > 0.05) == (y > 0.05) for x, y in zip(errs, errs_o) if abs(y - 0.05) > 0.005)
        deltas.append(d.copy())
        e_prev = float(max(errs))
    # the loop really moved the thresholds (compression error of rank-8/16 coefficients without residuals is far above 5 %)
    assert deltas[0].min() < 0.0 and not np.array_equal(deltas[0], deltas[-1])
    flags_total = int(oc.seqs[0]["flag"].sum())
    assert flags_total > 0
    ctl.destroy(); cache.destroy()
