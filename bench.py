#!/usr/bin/env python
"""bench.py -- decode-attention throughput of the DepthWeave-KV hot path on B200 (BASELINE.json metric).

A "step" is one pass of the whole hot path (q pre-projection, split-T scan, combine: all layers) over one batch of
synthetic cached sequences. Default workload: BASELINE.json configs[2] at batch 8 (Llama-3-8B shape, T = 65536).
    python bench.py [--gpus N --steps K --warmup W] [--workload NAME] [--impl reference]
Prints ONE JSON line (rank 0). N > 1 (torchrun): independent replicas, one per GPU, no data-path collective.
"""
import argparse
import json
import os
import sys
import threading
import time

import numpy as np
import torch

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import gen  # noqa: E402

METRIC = "decode-attn cached tokens scanned/s (all layers; ms_per_step = ms/step) at 64K ctx"
UNIT = "tokens/s"


def config_of(wl, world, footprint_gb=None, coef_int8=False):
    """The `config` object of the JSON line: the same for our arm and the reference arm."""
    c = {"workload": wl.name, "shape": f"L={wl.L} w={wl.w} H_kv={wl.H_kv} G={wl.G} d={wl.d} r={wl.r}",
         "batch": wl.n_seq, "T": wl.T[0] if len(set(wl.T)) == 1 else [min(wl.T), max(wl.T)], "tiers": list(wl.tier_ranks),
         "tier_frac": list(wl.tier_frac), "resid_frac": wl.resid_frac, "launch_mode": "all layers in one call (layer = -1)",
         "l2_policy": "inputs larger than L2 (compressed cache of the workload >> 126 MB; every step streams all of it): no flush",
         "parallelism": "replicas only (no sharding, no collective)" if world > 1 else "single GPU"}
    c["coefficients"] = "int8 codes + one power-of-two exponent byte per 32-column block (PAPER.md:56, A27)" if coef_int8 else "bf16 (BASELINE.json north_star)"
    return c


def traffic_of(workload):
    """dram__bytes_read + dram__bytes_write of the fused decode kernel per launch, from the committed ncu capture (or None)."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    try:
        return json.load(open(p)).get(workload)
    except Exception:
        return None


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """Samples SM clocks and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index):
        self.samples, self.reasons, self.max_mhz, self.power_w = [], set(), None, []
        self._stop = threading.Event()
        self._t = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def _run(self):
        nv = self.nv
        names = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "sw_thermal_slowdown": 0x20, "hw_thermal_slowdown": 0x40,
                 "hw_power_brake": 0x80, "sync_boost": 0x10, "applications_clocks": 0x2}
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                self.power_w.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
                r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(0.02)

    def __enter__(self):
        if self.nv:
            self._t = threading.Thread(target=self._run, daemon=True)
            self._t.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._t:
            self._t.join()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["unavailable"]}
        out = {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons)}
        if self.power_w:
            out["power_w_median"] = float(np.median(self.power_w)); out["power_w_max"] = float(np.max(self.power_w))
        return out


def time_steps(fn, steps, warmup):
    """CUDA-event timing on the current stream, sync on both sides; returns ms per step."""
    for _ in range(warmup):
        fn()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for i in range(steps):
        fn()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / steps


def prefill_compress(wl, harness, local, reps=3):
    """Batched (prefill-sized) dwkv_append_compress: all tokens of one sequence of the workload's length (capped at 64K) in ONE
    call on a cache of its own -- the TTFT side of the method (PAPER.md:74 'during prefill ... projects keys and values into
    shared coefficient space, stores quantized residuals'). Returns ms per call (host routing + kernel, the
    GPU idle at the start) and the dense bytes read."""
    import dataclasses
    n = min(max(wl.T), 65536)
    wl1 = dataclasses.replace(wl, T=(n,), patterns=())
    tier, flag = gen.make_routing(wl1, 0)
    cache, (BK, BV, gK, gV) = harness.make_cache(wl1, arena_bytes=harness.arena_bytes_for(wl1, [(tier, flag)], 1), device=local)
    dev = torch.device("cuda", local)
    ks, vs = [], []
    for t0 in range(0, n, 8192):              # generator intermediates are fp32: build the dense input chunk-wise
        k, v = gen.make_dense_kv_chunk(wl1, 0, t0, min(8192, n - t0), BK, BV, gK, gV, device=dev)
        ks.append(k.contiguous()); vs.append(v.contiguous())
    k_new, v_new = torch.cat(ks), torch.cat(vs)
    del ks, vs
    # basis construction from the same dense K/V (dwkv_build_basis: sketch GEMM + one-sided Jacobi), before any token exists
    n_sketch = min(wl.d, 80, (wl.r + 16 + 15) // 16 * 16)
    n8 = n // 8 * 8
    omega = gen.make_omega(wl1, n8, n_sketch, device=dev)
    bms = []
    for _ in range(reps + 1):
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); cache.build_basis(k_new[:n8], v_new[:n8], omega); e1.record()
        torch.cuda.synchronize()
        bms.append(e0.elapsed_time(e1))
    cache.set_basis(BK, BV)                   # the timed compress call below uses the workload's own basis
    del omega
    ms = []
    for _ in range(reps + 1):
        cache.reset_seq(0)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); cache.append_compress([0], [n], k_new, v_new, tier, flag); e1.record()
        torch.cuda.synchronize()
        ms.append(e0.elapsed_time(e1))
    cache.destroy()
    dense_bytes = 2 * k_new.numel() * 2
    best = min(ms[1:])
    return {"tokens": n, "ms_per_call": best, "dense_bytes_read": dense_bytes, "dense_GBps": dense_bytes / best / 1e6,
            "tokens_per_s": n / best * 1e3, "build_basis_ms": min(bms[1:]), "build_basis_sketch_rows": n_sketch,
            "build_basis_dense_GBps": 2 * k_new[:n8].numel() * 2 / min(bms[1:]) / 1e6, "note": "one dwkv_append_compress call, timed from an idle GPU: host routing + table upload + kernels (free pages are kept cleared: nothing is zeroed in the call)"}


def reconstruct_dense(cache, wl, consts, seq, K_out, V_out, chunk=2048):
    """Dense comparison cache of one sequence FROM THE COMPRESSED CACHE: K_out, V_out [L, H_kv, T, d] bf16 =
    bf16(K-hat), bf16(V-hat) with X-hat = gate * (c . B[window]) + code * scale (Eq. 1), built from dwkv_export_tokens (token-ordered
    coefficients, zero beyond r_t, and the dequantised residuals) with torch ops. Harness code: the dense kernel then attends to the
    same keys and values as the compressed path, so the two outputs cross-check each other."""
    BK, BV, gK, gV = consts
    grp = torch.arange(wl.L, device=K_out.device) // wl.w
    Bl = {"K": BK.float()[grp], "V": BV.float()[grp]}            # [L, H, r, d]
    gl = {"K": gK.float(), "V": gV.float()}
    T = K_out.shape[2]
    for t0 in range(0, T, chunk):
        n = min(chunk, T - t0)
        dump = cache.export_tokens(seq, t0, n, want=("coefK", "coefV", "deqK", "deqV"))
        for z, dst in (("K", K_out), ("V", V_out)):
            x = torch.einsum("tlhr,lhrd->tlhd", dump["coef" + z].float(), Bl[z]) * gl[z][None] + dump["deq" + z]
            dst[:, :, t0:t0 + n] = x.to(torch.bfloat16).permute(1, 2, 0, 3)
        del dump


def oracle_sample(wl, consts, tier, flag, kept, q_host, layers, budget_s=25.0, coef_int8=False):
    """Time the CPU oracle as it stands on (layer, kv head) slices of sequence 0; returns (token-layers/s, sample text,
    threads, worst rel-L2 vs `gpu_out` if given)."""
    from oracle import dwkv_oracle as orc
    try:
        from threadpoolctl import threadpool_info
        threads = max([p.get("num_threads", 1) for p in threadpool_info()] + [1])
    except Exception:
        threads = os.cpu_count() or 1
    f64 = lambda t: t.detach().double().cpu().numpy()
    BK, BV, gK, gV = [f64(x) for x in consts]
    T = len(tier)
    ranks = np.asarray(wl.tier_ranks)[tier]
    idx = np.nonzero(flag)[0]
    outs = {}

    def coef(c):        # the stored coefficients as float64: the generator's bf16 values, or their 8-bit quantisation (A27)
        c = f64(c)
        if not coef_int8:
            return c
        from oracle import dwkv_coef8_oracle as c8
        q8 = np.zeros_like(c)
        for rk in set(ranks.tolist()):
            sel = ranks == rk
            codes, exps = c8.quantize_coef_i8(c[sel].astype(np.float32), rank=rk)
            q8[sel] = c8.dequant_coef_i8(codes, exps)
        return q8
    t0 = time.perf_counter()
    done_layers = 0
    for l in layers:
        for h in range(wl.H_kv):
            k = kept[(l, h)]
            cK_ = np.zeros((T, wl.d), np.int8); cV_ = np.zeros((T, wl.d), np.int8)
            sK_ = np.zeros((T, wl.d // 16), np.float16); sV_ = np.zeros((T, wl.d // 16), np.float16)
            if len(idx):
                cK_[idx], sK_[idx] = orc.quantize_int4_g16(k["rK"].numpy())
                cV_[idx], sV_[idx] = orc.quantize_int4_g16(k["rV"].numpy())
            o, _, V = orc.attention_slice(coef(k["cK"]), coef(k["cV"]), ranks, flag, cK_, sK_, cV_, sV_, BK[l // wl.w, h],
                                          BV[l // wl.w, h], gK[l, h], gV[l, h], q_host[l, h * wl.G:(h + 1) * wl.G],
                                          1.0 / np.sqrt(wl.d))
            outs[(l, h)] = (o, float(np.abs(V).max()))
        done_layers += 1
        if time.perf_counter() - t0 > budget_s:
            break
    dt = time.perf_counter() - t0
    return done_layers * T / dt, done_layers, dt, threads, outs


def other_workload(name, harness, local, peak, steps, warmup, with_append=False, n_sustained=100):
    """One of the other BASELINE.json configs inside the default run (so that the driver's line carries every config): burst and
    sustained time of the all-layer decode step, roofline fractions, and the oracle's rel-L2 on one sampled (layer, head) slice of the
    longest sequence. with_append: configs[4]'s dwkv_append_compress of wl.n_append tokens per sequence before every decode step."""
    from oracle import dwkv_oracle as orc
    wl = gen.WORKLOADS[name]
    dev = torch.device("cuda", local)
    routings = [gen.make_routing(wl, s) for s in range(wl.n_seq)]
    n_app = wl.n_append if with_append else 0
    n_calls = 2 * (steps + warmup) + n_sustained + 8
    cache, consts = harness.make_cache(wl, max_tokens=max(wl.T) + 4096 + n_app * n_calls,
                                       arena_bytes=harness.arena_bytes_for(wl, routings, 1, slack_tokens=n_app * n_calls), device=local)
    s_samp = int(np.argmax(wl.T))
    lh = (wl.L // 2, wl.H_kv - 1)
    kept = None
    for s, (tier, flag) in enumerate(routings):
        k = harness.fill_sequence(cache, wl, s, s, tier, flag, device=local, chunk=4096, keep=[lh] if s == s_samp else [])
        if s == s_samp:
            kept = k
    torch.cuda.synchronize()
    ids = list(range(wl.n_seq))
    q = gen.make_q(wl, device=dev)
    out = torch.empty(wl.n_seq, wl.L, wl.H_q, wl.d, dtype=torch.float32, device=dev)
    fp = cache.footprint()
    rec = {"workload": name, "used_bytes": fp["used_bytes"], "compression_ratio": fp["dense_equiv_bytes"] / fp["used_bytes"]}
    # parity of one sampled slice at full size (before any append changes the cache)
    cache.decode_attention(-1, ids, q, out)
    torch.cuda.synchronize()
    tier, flag = routings[s_samp]
    f64 = lambda t: t.detach().double().cpu().numpy()
    BK, BV, gK, gV = [f64(x) for x in consts]
    l, h = lh
    T = len(tier)
    cK_ = np.zeros((T, wl.d), np.int8); cV_ = np.zeros((T, wl.d), np.int8)
    sK_ = np.zeros((T, wl.d // 16), np.float16); sV_ = np.zeros((T, wl.d // 16), np.float16)
    idx = np.nonzero(flag)[0]
    if len(idx):
        cK_[idx], sK_[idx] = orc.quantize_int4_g16(kept[lh]["rK"].numpy())
        cV_[idx], sV_[idx] = orc.quantize_int4_g16(kept[lh]["rV"].numpy())
    o_ref, _, _ = orc.attention_slice(f64(kept[lh]["cK"]), f64(kept[lh]["cV"]), np.asarray(wl.tier_ranks)[tier], flag, cK_, sK_, cV_, sV_,
                                      BK[l // wl.w, h], BV[l // wl.w, h], gK[l, h], gV[l, h], f64(q)[s_samp, l, h * wl.G:(h + 1) * wl.G],
                                      1.0 / np.sqrt(wl.d))
    got = out[s_samp, l, h * wl.G:(h + 1) * wl.G].double().cpu().numpy()
    rec["sampled_slice"] = f"sequence {s_samp} (T = {T}), layer {l}, kv head {h}"
    rec["sampled_parity_rel_l2"] = float(np.linalg.norm(got - o_ref) / np.linalg.norm(o_ref))
    if n_app:
        BKt, BVt, gKt, gVt = consts
        rng = np.random.Generator(np.random.PCG64([gen.BASE_SEED, wl.index, 98]))
        kd, vd = [], []
        for s_ in range(wl.n_seq):
            k_, v_ = gen.make_dense_kv_chunk(wl, s_, 10 ** 6, n_app, BKt, BVt, gKt, gVt, device=dev)
            kd.append(k_); vd.append(v_)
        k_new, v_new = torch.cat(kd), torch.cat(vd)
        a_tier = rng.choice(len(wl.tier_ranks), size=n_app * wl.n_seq, p=list(wl.tier_frac)).astype(np.uint8)
        a_flag = ((a_tier == len(wl.tier_ranks) - 1) & (rng.random(n_app * wl.n_seq) < 0.8)).astype(np.uint8)
        n_new = [n_app] * wl.n_seq

        def step():
            cache.append_compress(ids, n_new, k_new, v_new, a_tier, a_flag)
            cache.decode_attention(-1, ids, q, out)
    else:
        def step():
            cache.decode_attention(-1, ids, q, out)
    torch.cuda.synchronize(); time.sleep(1.0)
    b0 = cache.footprint()["used_bytes"]
    ms = time_steps(step, steps, warmup)
    b1 = cache.footprint()["used_bytes"]
    alg = (b0 + b1) // 2
    rec.update({"us_per_step": ms * 1e3, "GBps": alg / ms / 1e6, "frac_of_peak": alg / ms / 1e6 / peak, "frac_of_8TBps_nominal": alg / ms / 1e6 / 8000.0})
    b0 = cache.footprint()["used_bytes"]
    with ClockSampler(local) as cl:
        ms_l = time_steps(step, n_sustained, 3)
    alg = (b0 + cache.footprint()["used_bytes"]) // 2
    rec["sustained"] = {"steps": n_sustained, "us_per_step": ms_l * 1e3, "frac_of_peak": alg / ms_l / 1e6 / peak,
                        "frac_of_8TBps_nominal": alg / ms_l / 1e6 / 8000.0, "clocks": cl.summary()}
    if n_app:
        cache.set_option("time_scan", 1)
        step(); torch.cuda.synchronize()
        rec["append_tokens_per_seq_per_step"] = n_app
        rec["compress_kernel_us"] = cache.get_stat("compress_ms") * 1e3
        rec["decode_kernel_us"] = cache.get_stat("scan_ms") * 1e3
    cache.destroy()
    del cache, out
    torch.cuda.empty_cache()
    return rec


def run_reference(args, wl):
    """--impl reference: the CPU oracle on the host cores, on a bounded sample of the same workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    tier, flag = gen.make_routing(wl, 0)
    consts = gen.make_basis(wl) + gen.make_gates(wl)
    n_layers = 1
    keep = [(l, h) for l in range(n_layers) for h in range(wl.H_kv)]
    kept = {lh: dict(cK=[], cV=[], rK=[], rV=[]) for lh in keep}
    chunk = 8192
    for t0 in range(0, len(tier), chunk):      # generate only the sampled slices' worth of data, chunk by chunk
        tr, fl = tier[t0:t0 + chunk], flag[t0:t0 + chunk]
        wl1 = wl
        cK, cV = gen.make_coef_chunk(wl1, 0, t0, tr, device="cpu")
        nf = int(fl.sum())
        rK, rV = gen.make_resid_chunk(wl1, 0, t0, nf, device="cpu") if nf else (None, None)
        for (l, h) in keep:
            kept[(l, h)]["cK"].append(cK[:, l, h].clone()); kept[(l, h)]["cV"].append(cV[:, l, h].clone())
            if nf:
                kept[(l, h)]["rK"].append(rK[:, l, h].clone()); kept[(l, h)]["rV"].append(rV[:, l, h].clone())
    kept = {lh: {k: (torch.cat(v) if v else None) for k, v in d.items()} for lh, d in kept.items()}
    q = gen.make_q(wl, n_seq=1).double().numpy()[0]
    vals = []
    for i in range(args.warmup + args.steps):
        tps, nl, dt, threads, _ = oracle_sample(wl, consts, tier, flag, kept, q, range(n_layers), budget_s=1e9)
        if i >= args.warmup:
            vals.append((tps, dt))
    tps = float(np.mean([v[0] for v in vals]))
    ms = float(np.mean([v[1] for v in vals])) * 1e3
    sample = f"{n_layers} layer x {wl.H_kv} kv heads x T={len(tier)} of sequence 0 per step (1/{wl.L * wl.n_seq} of the workload step)"
    line = {"impl": "reference", "metric": METRIC, "value": tps, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": config_of(wl, args.gpus),
            "cpu_baseline": {"value": tps, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
            "e2e": {"value": tps, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="llama8b_64k_b8")
    ap.add_argument("--opt", action="append", default=[], help="library option key=value (experiments), repeatable")
    ap.add_argument("--append", action="store_true",
                    help="BASELINE.json configs[4]: dwkv_append_compress of wl.n_append new tokens per sequence before every decode step")
    ap.add_argument("--coef-int8", action="store_true",
                    help="store the coefficients in 8-bit blockwise form (PAPER.md:56; dwkv.h option coef_int8; DESIGN.md A27; rank <= 32)")
    ap.add_argument("--no-dense", action="store_true", help="skip the dense-bf16 comparison kernel")
    ap.add_argument("--no-extra", action="store_true", help="skip batch 1/4, per-layer mode and the CPU baseline")
    args = ap.parse_args()
    wl = gen.WORKLOADS[args.workload]
    if args.impl == "reference":
        return run_reference(args, wl)

    from paper_2607_06523_b200 import harness, binding, replicas
    rank, world, local = replicas.env_rank()
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    replicas.init("nccl", dev)          # replicas only: the group serves the barrier and the max over ranks of the time

    # ---- build the cache (every rank: its own replica of the batch, different seeds would not change the timing) ----
    routings = [gen.make_routing(wl, s) for s in range(wl.n_seq)]
    n_app = wl.n_append if args.append else 0
    app_steps = 2 * (args.steps + args.warmup) + 4
    slack = 1 + (n_app * app_steps + 127) // 128        # pages per (sequence, class) for the appended tokens (>= 227 tokens per page)
    cache, consts = harness.make_cache(wl, max_tokens=max(wl.T) + 4096 + n_app * app_steps,
                                       arena_bytes=harness.arena_bytes_for(wl, routings, slack), device=local)
    if args.coef_int8:
        cache.set_option("coef_int8", 1)
    for kv in args.opt:
        k, v = kv.split("=")
        cache.set_option(k, int(v))
    # layers of sequence 0 the CPU oracle is timed on (and the GPU output is compared with): ~1.5 s of host time per layer at T = 64K
    sample_layers = sorted(set(int(x) for x in np.linspace(0, wl.L - 1, min(wl.L, 8 if max(wl.T) <= 65536 else 4))))
    keep = [(l, h) for l in sample_layers for h in range(wl.H_kv)] if (rank == 0 and not args.no_extra) else []
    kept0 = None
    s_samp = int(np.argmax(wl.T))       # the sequence the CPU oracle is timed on and compared with: the longest
    t_fill = time.perf_counter()
    for s, (tier, flag) in enumerate(routings):
        k = harness.fill_sequence(cache, wl, s, s, tier, flag, device=local, chunk=4096, keep=keep if s == s_samp else [])
        if s == s_samp:
            kept0 = k
    torch.cuda.synchronize()
    t_fill = time.perf_counter() - t_fill
    fp = cache.footprint()
    n_seq, L = wl.n_seq, wl.L
    seq_ids = list(range(n_seq))
    tokens_per_step = sum(wl.T) * L
    nq = 4
    qs = [gen.make_q(wl, step=i, device=dev) for i in range(nq)]
    out = torch.empty(n_seq, L, wl.H_q, wl.d, dtype=torch.float32, device=dev)
    it = [0]

    def step():
        cache.decode_attention(-1, seq_ids, qs[it[0] % nq], out)
        it[0] += 1

    append_ms = []
    if n_app:
        # dense K/V of the new tokens (x = gate * (c . B) + e, gen.make_dense_kv_chunk) and their tiers / flags, generated once
        BK, BV, gK, gV = consts
        rng = np.random.Generator(np.random.PCG64([gen.BASE_SEED, wl.index, 99]))
        n_new = [n_app] * n_seq
        kd, vd = [], []
        for s_ in range(n_seq):
            k_, v_ = gen.make_dense_kv_chunk(wl, s_, 10 ** 6, n_app, BK, BV, gK, gV, device=dev)
            kd.append(k_); vd.append(v_)
        k_new, v_new = torch.cat(kd), torch.cat(vd)
        a_tier = rng.choice(len(wl.tier_ranks), size=n_app * n_seq, p=list(wl.tier_frac)).astype(np.uint8)
        a_flag = ((a_tier == len(wl.tier_ranks) - 1) & (rng.random(n_app * n_seq) < 0.8)).astype(np.uint8)
        decode_only = step

        def step():
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            cache.append_compress(seq_ids, n_new, k_new, v_new, a_tier, a_flag)
            e1.record()
            decode_only()
            append_ms.append((e0, e1))

    # ---- timed region: K steps, inputs resident in HBM ------------------------------------------------------------
    step(); torch.cuda.synchronize()
    replicas.barrier()
    l0 = cache.launch_count()
    with ClockSampler(local) as cs:
        ms = time_steps(step, args.steps, args.warmup)
    launches = (cache.launch_count() - l0) * args.steps // (args.steps + args.warmup)
    ms = replicas.max_over_ranks(ms, dev)
    value = replicas.aggregate_throughput(tokens_per_step, ms, world)

    # ---- e2e: host q -> device, decode, result -> host, every step ------------------------------------------------
    # Double-buffered: every step still copies ITS q from pinned host memory and ITS fp32 output back (both inside the timed
    # region), but the copies run on a second stream: q of step i + 1 goes up and the output of step i - 1 comes down while the
    # kernels of step i run; the host waits for the output of step i - 1 before it enqueues step i + 1 (results are consumed in order).
    q_host = [q.cpu().pin_memory() for q in qs]
    q_dev2 = [torch.empty_like(qs[0]) for _ in range(2)]
    out2 = [torch.empty_like(out) for _ in range(2)]
    out_host2 = [torch.empty(out.shape, dtype=out.dtype).pin_memory() for _ in range(2)]
    main_s, copy_s = torch.cuda.current_stream(), torch.cuda.Stream()
    ev_q = [torch.cuda.Event() for _ in range(2)]; ev_dec = [torch.cuda.Event() for _ in range(2)]; ev_out = [torch.cuda.Event() for _ in range(2)]

    def run_e2e(n_steps):
        def upload(i):
            with torch.cuda.stream(copy_s):
                copy_s.wait_event(ev_dec[i % 2])              # the decode that last read this q buffer has finished
                q_dev2[i % 2].copy_(q_host[i % nq], non_blocking=True)
                ev_q[i % 2].record(copy_s)
        for b in range(2):
            ev_dec[b].record(main_s); ev_out[b].record(copy_s)
        upload(0)
        for i in range(n_steps):
            if i + 1 < n_steps:
                upload(i + 1)
            main_s.wait_event(ev_q[i % 2])
            main_s.wait_event(ev_out[i % 2])                 # the previous download of this output buffer has finished
            cache.decode_attention(-1, seq_ids, q_dev2[i % 2], out2[i % 2])
            ev_dec[i % 2].record(main_s)
            with torch.cuda.stream(copy_s):
                copy_s.wait_event(ev_dec[i % 2])
                out_host2[i % 2].copy_(out2[i % 2], non_blocking=True)
                ev_out[i % 2].record(copy_s)
            if i >= 1:
                ev_out[(i - 1) % 2].synchronize()            # the host consumes the result of step i - 1
        ev_out[(n_steps - 1) % 2].synchronize()

    run_e2e(args.warmup)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    run_e2e(args.steps)
    torch.cuda.synchronize()
    e2e_ms = (time.perf_counter() - t0) * 1e3 / args.steps
    e2e_ms = replicas.max_over_ranks(e2e_ms, dev)
    e2e = {"value": replicas.aggregate_throughput(tokens_per_step, e2e_ms, world), "unit": UNIT, "ms_per_step": e2e_ms,
           "h2d_bytes_per_step": q_dev2[0].numel() * 2, "d2h_bytes_per_step": out.numel() * 4,
           "note": "pinned host q -> device, decode, fp32 output -> pinned host, every step; copies double-buffered on a second stream"}
    del q_dev2, out2

    # ---- roofline of the dominant kernel group (split-T scan), CUDA events inside the library on the launch stream --
    cache.set_option("time_scan", 1)
    scan_ms, compress_ms = [], []
    fp_before = cache.footprint()
    if not n_app:         # the kernel as it runs in the timed region: steps back to back, no synchronise between the samples
        torch.cuda.synchronize()
        time.sleep(1.0)       # same start as the timed region: an idle board (power-limit averaging window empty), W warm-up steps, K steps
        n_samp, n_trail = min(args.steps, 56), 6              # (the library keeps the event brackets of the last 64 calls)
        for i in range(args.warmup + n_samp + n_trail):       # trailing steps keep the queue full behind the last sample: the
            if i == args.warmup:                              # last kernels before the stream drains measure 3-10 % slower
                cache.set_option("time_scan", 1)              # restarts the sample count after the warm-up steps
            step()
        torch.cuda.synchronize()
        scan_ms = [cache.get_stat(f"scan_ms@{i}") for i in range(n_samp)]
        scan_trail = [round(cache.get_stat(f"scan_ms@{i}"), 4) for i in range(n_samp, n_samp + n_trail)]
        scan_min = float(np.min(scan_ms))
    else:
        for i in range(args.steps):
            step()
            scan_ms.append(cache.get_stat("scan_ms"))
            compress_ms.append(cache.get_stat("compress_ms"))
        scan_min = float(np.min(scan_ms))
        scan_trail = []
    cache.set_option("time_scan", 0)
    scan_samples = [round(float(x), 4) for x in scan_ms]
    scan_median = float(np.median(scan_ms))
    scan_ms = float(np.mean(scan_ms))
    peak, peak_src = peaks()
    # calibration of the denominator: MEASURED_PEAKS.json is a read + WRITE copy; the decode kernel is a read-only stream. The same
    # protocol (idle start, 3 warm-up + 20 timed launches) on a read-only library reduction over a buffer of the cache's size:
    read_only = None
    if rank == 0 and not args.no_extra:
        try:
            probe = torch.empty(min(fp["used_bytes"], 8 << 30) // 2, dtype=torch.bfloat16, device=dev)
            probe.zero_()
            torch.cuda.synchronize(); time.sleep(1.0)
            ro_ms = time_steps(lambda: torch.sum(probe, dtype=torch.float32), 20, 3)
            read_only = probe.numel() * 2 / (ro_ms * 1e-3) / 1e9
            del probe
        except Exception:  # pragma: no cover
            read_only = None
    # compressed records: 4 r_t + f_t*2*(d/2+d/8) per (l, h, token); with --append the cache grows while the kernel is timed
    alg_bytes = (fp_before["used_bytes"] + cache.footprint()["used_bytes"]) // 2 if n_app else fp["used_bytes"]
    achieved = alg_bytes / (scan_ms * 1e-3) / 1e9
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": traffic_of(wl.name + ("_i8" if args.coef_int8 else "")), "kernel": "scan3_kernel<NKB,D,PAIR> (fused q pre-projection + split-T scan, one persistent launch per step)",
                "scan_ms": scan_ms, "scan_ms_min": scan_min, "scan_ms_median": scan_median, "scan_ms_samples": scan_samples, "scan_ms_trailing_unused": scan_trail, "algorithmic_bytes": alg_bytes, "peak_source": peak_src,
                "frac_of_8TBps_nominal": achieved / 8000.0, "step_frac_of_peak": alg_bytes / (ms * 1e-3) / 1e9 / peak,
                "read_only_stream_GBps": read_only, "frac_of_read_only_stream": (achieved / read_only) if read_only else None,
                "read_only_stream_note": "torch.sum over a bf16 buffer of the cache's size, same idle-start protocol: a read-only ceiling "
                                         "beside the driver's read + write copy figure (`peak`)"}

    extra_append = None
    if n_app:
        torch.cuda.synchronize()
        am = [a.elapsed_time(b) for a, b in append_ms[-args.steps:]]
        extra_append = {"tokens_per_seq_per_step": n_app, "append_us_per_step": float(np.mean(am)) * 1e3,
                        "decode_us_per_step": (ms - float(np.mean(am))) * 1e3,
                        "compress_kernel_us": float(np.mean(compress_ms)) * 1e3 if compress_ms else None,
                        "new_vectors_per_step": 2 * n_app * n_seq * L * wl.H_kv,
                        "dense_bytes_read_per_step": 2 * n_app * n_seq * L * wl.H_kv * wl.d * 2,
                        "note": "ms_per_step = append + plan rebuild + decode; the cache grows by n_append tokens per sequence every step; "
                                "append_us / decode_us split the step at the event after dwkv_append_compress (host routing and planning "
                                "show up in whichever interval the GPU waits for the host); compress_kernel_us is the a4 kernel alone"}
    extra = {"fill_s": t_fill, "append": extra_append, "footprint": fp, "compression_ratio": fp["dense_equiv_bytes"] / fp["used_bytes"],
             "us_per_step": ms * 1e3}
    cpu_baseline = None
    if rank == 0 and not args.no_extra:
        # batch 1 and 4 on the same cache; per-layer launch mode
        for nb in (1, 4):
            if nb < n_seq:
                ids = seq_ids[:nb]
                qb = [q[:nb].contiguous() for q in qs]
                ob = torch.empty(nb, L, wl.H_q, wl.d, dtype=torch.float32, device=dev)
                msb = time_steps(lambda: cache.decode_attention(-1, ids, qb[0], ob), args.steps, args.warmup)
                extra[f"batch{nb}_us_per_step"] = msb * 1e3
                extra[f"batch{nb}_frac_of_peak"] = alg_bytes * nb / n_seq / (msb * 1e-3) / 1e9 / peak
        # per-layer calls: the launch mode a real decoder issues (layer l + 1's q depends on layer l's output): L calls
        # per step, plain and captured once in a CUDA graph (no host work between the layers), at batch 1 / 4 / full
        per_layer = {}
        for nb in sorted({1, min(4, n_seq), n_seq}):
            ids = seq_ids[:nb]
            ql = [qs[0][:nb, l].contiguous() for l in range(L)]
            ol = [torch.empty(nb, wl.H_q, wl.d, dtype=torch.float32, device=dev) for l in range(L)]

            def per_layer_calls():
                for l in range(L):
                    cache.decode_attention(l, ids, ql[l], ol[l])
            rec = {"plain_us_per_step": time_steps(per_layer_calls, max(3, args.steps // 2), args.warmup) * 1e3}
            try:
                side = torch.cuda.Stream()
                side.wait_stream(torch.cuda.current_stream())
                with torch.cuda.stream(side):
                    per_layer_calls()
                    graph = torch.cuda.CUDAGraph()
                    with torch.cuda.graph(graph, stream=side):
                        per_layer_calls()
                torch.cuda.current_stream().wait_stream(side)
                torch.cuda.synchronize(); time.sleep(0.5)
                g_us = time_steps(graph.replay, args.steps, args.warmup) * 1e3
                got = torch.stack(ol, dim=1)
                ob = torch.empty(nb, L, wl.H_q, wl.d, dtype=torch.float32, device=dev)
                cache.decode_attention(-1, ids, qs[0][:nb].contiguous(), ob)
                b_alg = alg_bytes * sum(wl.T[:nb]) / sum(wl.T)
                rec.update({"graph_us_per_step": g_us, "graph_GBps": b_alg / g_us / 1e3, "graph_frac_of_peak": b_alg / g_us / 1e3 / peak,
                            "graph_frac_of_8TBps_nominal": b_alg / g_us / 1e3 / 8000.0,
                            "vs_all_layers_rel_l2": float((got - ob).norm() / ob.norm())})
                del graph
            except Exception as ex:  # pragma: no cover
                rec["graph_error"] = repr(ex)[:200]
            per_layer[f"batch{nb}"] = rec
        extra["per_layer"] = per_layer
        full = per_layer.get(f"batch{n_seq}", {})
        extra["per_layer_mode_us_per_step"] = full.get("plain_us_per_step")
        extra["per_layer_graph_us_per_step"] = full.get("graph_us_per_step")
        extra["per_layer_graph_vs_all_layers_rel_l2"] = full.get("vs_all_layers_rel_l2")
        roofline["frac_all_layers"] = roofline["step_frac_of_peak"]
        roofline["frac_per_layer"] = full.get("graph_frac_of_peak")
        roofline["frac_per_layer_batch1"] = per_layer.get("batch1", {}).get("graph_frac_of_peak")
        try:
            extra["prefill_compress"] = prefill_compress(wl, harness, local)
        except Exception as ex:
            extra["prefill_compress"] = {"error": repr(ex)[:200]}
        # CPU oracle on the host cores: bounded sample, and parity of the sampled slices at full size
        tier, flag = routings[s_samp]
        o_gpu = out.clone()
        cache.decode_attention(-1, seq_ids, qs[0], o_gpu)
        torch.cuda.synchronize()
        tps, nl, dt, threads, outs = oracle_sample(wl, consts, tier, flag, kept0, qs[0][s_samp].double().cpu().numpy(),
                                                   sample_layers, budget_s=25.0, coef_int8=args.coef_int8)
        og = o_gpu[s_samp].double().cpu().numpy()
        rels = []
        for (l, h), (o_ref, vmax) in outs.items():
            got = og[l, h * wl.G:(h + 1) * wl.G]
            rels.append(float(np.linalg.norm(got - o_ref) / np.linalg.norm(o_ref)))
        cpu_baseline = {"value": tps, "unit": UNIT, "cores": threads, "kind": "oracle",
                        "sample": f"{nl} layer(s) x {wl.H_kv} kv heads x T={len(tier)} of sequence {s_samp} ({dt:.1f} s)",
                        "sampled_parity_rel_l2_max": max(rels)}

    # ---- the paper's own coefficient format ("8-bit blockwise quantized"; option coef_int8, A27) on the same workload ---
    if rank == 0 and not args.no_extra and not args.coef_int8 and not n_app and wl.r <= 32:
        try:
            c8, _ = harness.make_cache(wl, max_tokens=max(wl.T) + 4096, arena_bytes=harness.arena_bytes_for(wl, routings, 1),
                                       device=local, coef_int8=True)
            for s, (tier, flag) in enumerate(routings):
                harness.fill_sequence(c8, wl, s, s, tier, flag, device=local, chunk=4096)
            o8 = torch.empty_like(o_gpu)
            ms8 = time_steps(lambda: c8.decode_attention(-1, seq_ids, qs[0], o8), args.steps, args.warmup)
            fp8 = c8.footprint()
            extra["coef_int8"] = {"us_per_step": ms8 * 1e3, "used_bytes": fp8["used_bytes"],
                                  "compression_ratio": fp8["dense_equiv_bytes"] / fp8["used_bytes"],
                                  "GBps": fp8["used_bytes"] / (ms8 * 1e-3) / 1e9, "frac_of_peak": fp8["used_bytes"] / (ms8 * 1e-3) / 1e9 / peak,
                                  "rel_l2_vs_bf16_coefficients": float((o8 - o_gpu).norm() / o_gpu.norm()),
                                  "note": "same generator outputs quantised on load (one power-of-two scale per token vector); the decode "
                                          "kernel widens the codes in registers and is ALU-pipe bound in this mode (profiles/r1_v6.md): a "
                                          "footprint option, not a speed-up"}
            c8.destroy()
        except Exception as ex:  # pragma: no cover
            extra["coef_int8"] = {"error": repr(ex)[:200]}

    # ---- dense bf16 comparison kernel on the same shapes ------------------------------------------------------------
    if rank == 0 and not args.no_dense and len(set(wl.T)) > 1:
        extra["dense"] = {"skipped": "the dense comparison kernel takes one length for all sequences; this workload is ragged"}
    elif rank == 0 and not args.no_dense:
        try:
            T = wl.T[0]
            free, _ = torch.cuda.mem_get_info()
            need = 2 * n_seq * L * wl.H_kv * T * wl.d * 2
            nb = n_seq
            while need * nb // n_seq > free - (4 << 30) and nb > 1:
                nb //= 2
            K = torch.empty(nb, L, wl.H_kv, T, wl.d, dtype=torch.bfloat16, device=dev)
            V = torch.empty_like(K)
            # sequences 0 and 1 are reconstructed from the compressed cache (cross-check below); the others repeat them (timing only)
            n_rec = min(nb, 2)
            for s in range(n_rec):
                reconstruct_dense(cache, wl, consts, s, K[s], V[s])
            for s in range(n_rec, nb):
                K[s].copy_(K[s % n_rec]); V[s].copy_(V[s % n_rec])
            qd = qs[0][:nb].contiguous()
            od = torch.empty(nb, L, wl.H_q, wl.d, dtype=torch.float32, device=dev)
            ws = torch.empty(binding.lib.dwkv_dense_workspace_bytes(nb, L, wl.H_q, wl.d, T), dtype=torch.uint8, device=dev)
            with ClockSampler(local) as cd:
                dms = time_steps(lambda: binding.dense_decode_attention(K, V, qd, wl.H_kv, workspace=ws, out=od),
                                 max(3, args.steps // 2), args.warmup)
            cache.decode_attention(-1, seq_ids[:n_rec], qs[0][:n_rec].contiguous(), out[:n_rec])
            dense_rel = float((od[:n_rec] - out[:n_rec]).norm() / out[:n_rec].norm())
            dense_bytes = 2 * K.numel() * 2
            comp_ms_same_batch = ms if nb == n_seq else extra.get(f"batch{nb}_us_per_step", ms * 1e3 * nb / n_seq) / 1e3
            extra["dense"] = {"batch": nb, "us_per_step": dms * 1e3, "GBps": dense_bytes / (dms * 1e-3) / 1e9,
                              "frac_of_peak": dense_bytes / (dms * 1e-3) / 1e9 / peak, "clocks": cd.summary(),
                              "speedup_compressed_vs_dense": dms / comp_ms_same_batch,
                              "rel_l2_dense_vs_compressed": dense_rel,
                              "cross_check": f"dense cache of sequences 0..{n_rec - 1} = bf16(K-hat), bf16(V-hat) reconstructed from the compressed cache "
                                             "(the other sequences repeat them: timing only); the two kernels' outputs differ by the bf16 rounding of K-hat / V-hat",
                              "required_speedup_0.7x_ratio": 0.7 * extra["compression_ratio"]}
            del K, V
        except Exception as ex:  # pragma: no cover
            extra["dense"] = {"error": repr(ex)}

    # ---- the same step held for ~0.5 s: at ~1 kW the board reaches its power limit and lowers the SM clocks ----------------
    if rank == 0 and not args.no_extra and not n_app:
        n_long = max(300, args.steps)
        with ClockSampler(local) as cl:
            ms_long = time_steps(step, n_long, 10)
        roofline["sustained_frac"] = alg_bytes / (ms_long * 1e-3) / 1e9 / peak
        extra["sustained"] = {"steps": n_long, "us_per_step": ms_long * 1e3, "clocks": cl.summary(),
                              "frac_of_peak": alg_bytes / (ms_long * 1e-3) / 1e9 / peak,
                              "frac_of_8TBps_nominal": alg_bytes / (ms_long * 1e-3) / 1e9 / 8000.0,
                              "note": "the timed region above (K steps, tens of ms) runs at full SM clocks; held for hundreds of steps the board "
                                      "hits its power limit (sw_power_cap) and the partly issue-bound decode kernel slows with the clocks"}

    # ---- the other BASELINE.json configs (configs[1], [3], [4] with and without appends), each on a cache of its own --------------
    if rank == 0 and not args.no_extra and not n_app and not args.coef_int8 and args.workload == "llama8b_64k_b8":
        cache.destroy()
        torch.cuda.empty_cache()
        others = {}
        for nm, app in (("llama8b_16k_b8", False), ("llama70b_128k_b1", False), ("ragged32", False), ("ragged32", True)):
            try:
                others[nm + ("_append" if app else "")] = other_workload(nm, harness, local, peak, args.steps, args.warmup, with_append=app)
            except Exception as ex:  # pragma: no cover
                others[nm + ("_append" if app else "")] = {"error": repr(ex)[:300]}
        extra["workloads"] = others

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16",
                "data": "synthetic",
                "config": config_of(wl, world, fp["used_bytes"] / 1e9, args.coef_int8),
                "clocks": cs.summary(), "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline,
                "cpu_baseline": cpu_baseline, "extra": extra}
        print(json.dumps(line))
    cache.destroy()
    if world > 1:
        torch.distributed.destroy_process_group()


if __name__ == "__main__":
    main()
