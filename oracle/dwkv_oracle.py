"""CPU oracle for DepthWeave-KV decode attention over the compressed cache.  TEST INFRASTRUCTURE ONLY.

Only `tests/`, `__graft_entry__.smoke()` and bench.py's `cpu_baseline` / `--impl reference` legs may import this
module. The product (paper_2607_06523_b200) never does; it shares no code, constants or layout with this file.

What it computes (plain definition, fp64, token-ordered storage, no blocking / fusion / reordering):

  Reconstruction, Eq. (1)  X-hat = A.B + g.R , read as BASELINE.json `north_star` fixes it
  (SURVEY.md §8 box, DESIGN.md §3 readings A1-A21):
      K-hat[t,:] = gK[l,h,:] * ( sum_{j<r_t} cK[l,h,t,j] * BK[m(l),h,j,:] ) + f_t * deq(RK[l,h,t])
      V-hat[t,:] = gV[l,h,:] * ( sum_{j<r_t} cV[l,h,t,j] * BV[m(l),h,j,:] ) + f_t * deq(RV[l,h,t])
      deq(R)[i]  = code[i] * scale[i // 16]          code in {-8..7}, scale fp16           ("4-bit group")
      m(l) = l // w   (disjoint depth windows, reading A1)
  Attention, the `Attn` of PAPER.md:67-70 Eq. (3), standard softmax:
      s[t] = q . K-hat[t] * softmax_scale ;  p = softmax_t(s) ;  o = sum_t p[t] * V-hat[t]
      query head h_q uses KV head h_q // G   (reading A11)
  Append / compress, "projecting the original cache vector onto the current basis" (readings A13, A14):
      c = bf16( B[:r_t] @ (x / g) )  (fp64 dot, one rounding) ;  e = x - g * (c @ B[:r_t])  (fp64, then fp32)
      int4 group-16 quantiser in fp32 IEEE (quantize_int4_g16 below)
  Routing (reading A15): class = 2*tier + flag, slot = number of earlier tokens of the sequence in that class.

Inputs are the stored numbers (bf16 / fp16 / int4 values held exactly in float64 / float16 / int8 arrays).
Pins: tests/test_oracle_pins.py (P1-P10, P12, P13 of SURVEY.md §8c), tests/test_oracle_pins_windows.py (P14 hand-derived
append case with two depth windows, P15 / P16 multi-window decode and append against loop-built references) and tests/test_retier.py
(OracleCache.retier, reading A29: against a fresh append at the lower tier, a closed form of the change of K-hat, brute-force slots). The paper prints no worked numeric example
of this path, so Eq. (3)'s 0.027 and the 72.8 tok/s are *parity unpinned* (out of scope, need real activations).
"""
from __future__ import annotations

import numpy as np

GROUP = 16  # residual quantisation group (BASELINE.json north_star: "int4 residual with group size 16")


# ------------------------------------------------------------------------------------------------------------
# storage-type helpers
# ------------------------------------------------------------------------------------------------------------

def round_to_bf16(x) -> np.ndarray:
    """Round float64 values to the nearest bfloat16 (ties to even), returned as float64.

    Direct fp64 -> bf16 rounding (no intermediate fp32 rounding): pick the nearest of the bf16 neighbours of x."""
    x = np.asarray(x, dtype=np.float64)
    f32 = x.astype(np.float32)
    bits = f32.view(np.uint32).astype(np.int64)
    base = bits & ~np.int64(0xFFFF)                       # truncate the low 16 bits (towards zero in magnitude)
    cands = []
    for k in (-1, 0, 1, 2):
        b = (base + k * 0x10000).astype(np.uint32)
        cands.append(b.view(np.float32).astype(np.float64))
    cands = np.stack(cands, axis=0)
    with np.errstate(invalid="ignore"):
        dist = np.abs(cands - x[None])
    dist = np.where(np.isfinite(dist), dist, np.inf)
    # ties -> even bf16 mantissa (bit 16 of the fp32 pattern clear)
    even = np.stack([(((base + k * 0x10000) >> 16) & 1) == 0 for k in (-1, 0, 1, 2)], axis=0)
    best = np.min(dist, axis=0)
    is_best = dist == best[None]
    pick_even = is_best & even
    idx = np.where(pick_even.any(axis=0), np.argmax(pick_even, axis=0), np.argmax(is_best, axis=0))
    out = np.take_along_axis(cands, idx[None], axis=0)[0]
    return np.where(x == 0.0, 0.0, out)


def quantize_int4_g16(e):
    """Reading A14: symmetric int4, group 16 along the last axis, fp16 scale, all in fp32 IEEE RN-even,
    no FMA, no reciprocal:
        amax = max|e_i| ; s32 = amax / 7.0f ; s32 = min(s32, 65504.0f) ; s = fp16_rn(s32)
        s == 0 -> codes 0 ; else code_i = clamp(rint(e_i / float(s)), -7, 7)
    Returns (codes int8 [..., d], scales float16 [..., d/16])."""
    e = np.asarray(e, dtype=np.float32)
    d = e.shape[-1]
    assert d % GROUP == 0
    g = e.reshape(e.shape[:-1] + (d // GROUP, GROUP))
    amax = np.max(np.abs(g), axis=-1).astype(np.float32)
    s32 = (amax / np.float32(7.0)).astype(np.float32)
    s32 = np.minimum(s32, np.float32(65504.0)).astype(np.float32)
    s16 = s32.astype(np.float16)
    sf = s16.astype(np.float32)
    with np.errstate(divide="ignore", invalid="ignore"):
        ratio = (g / sf[..., None]).astype(np.float32)
    code = np.rint(ratio)
    code = np.clip(code, -7.0, 7.0)
    code = np.where(sf[..., None] == 0, 0.0, code)
    return code.astype(np.int8).reshape(e.shape), s16


def dequant_int4_g16(codes, scales) -> np.ndarray:
    """deq[i] = code[i] * scale[i // 16]; exact in fp32 (4-bit integer times an 11-bit significand)."""
    codes = np.asarray(codes)
    d = codes.shape[-1]
    sf = np.asarray(scales).astype(np.float32)
    out = codes.astype(np.float32).reshape(codes.shape[:-1] + (d // GROUP, GROUP)) * sf[..., None]
    return out.reshape(codes.shape).astype(np.float32)


def route_slots(tier, flag, n_tiers: int, counts=None):
    """class[t] = 2*tier[t] + flag[t]; slot[t] = number of earlier tokens (including `counts` carried over from
    previous appends) in the same class. Returns (cls int32[T], slot int32[T], counts int64[2*n_tiers])."""
    tier = np.asarray(tier).astype(np.int64)
    flag = np.asarray(flag).astype(np.int64)
    counts = np.zeros(2 * n_tiers, dtype=np.int64) if counts is None else np.array(counts, dtype=np.int64)
    cls = 2 * tier + flag
    slot = np.zeros(len(cls), dtype=np.int64)
    for t in range(len(cls)):
        slot[t] = counts[cls[t]]
        counts[cls[t]] += 1
    return cls.astype(np.int32), slot.astype(np.int32), counts


# ------------------------------------------------------------------------------------------------------------
# one (layer, kv head) slice: reconstruction and attention
# ------------------------------------------------------------------------------------------------------------

def reconstruct(coef, ranks, flag, deq, B, gate) -> np.ndarray:
    """X-hat[t,:] = gate * sum_{j<r_t} coef[t,j] B[j,:] + flag[t] * deq[t,:]      (Eq. 1 as read in the header).

    coef [T,r], ranks [T] (r_t), flag [T] in {0,1}, deq [T,d] (ignored where flag==0; may be None), B [r,d], gate [d]."""
    coef = np.asarray(coef, dtype=np.float64)
    B = np.asarray(B, dtype=np.float64)
    gate = np.asarray(gate, dtype=np.float64)
    T, r = coef.shape
    lead = (np.arange(r)[None, :] < np.asarray(ranks)[:, None])          # leading-r_t coefficients only
    X = gate[None, :] * ((coef * lead) @ B)
    if deq is not None:
        f = np.asarray(flag).astype(bool)
        X = X + np.where(f[:, None], np.asarray(deq, dtype=np.float64), 0.0)
    return X


def softmax_attention(q, K, V, scale: float) -> np.ndarray:
    """o[g,:] = sum_t softmax_t(q[g] . K[t] * scale) V[t,:]; q [G,d], K,V [T,d]; fp64, max-subtracted."""
    q = np.asarray(q, dtype=np.float64)
    out = np.zeros((q.shape[0], V.shape[1]), dtype=np.float64)
    for g in range(q.shape[0]):
        s = (K @ q[g]) * scale
        s = s - np.max(s)
        p = np.exp(s)
        p = p / np.sum(p)
        out[g] = p @ V
    return out


# ------------------------------------------------------------------------------------------------------------
# token-ordered cache
# ------------------------------------------------------------------------------------------------------------

class OracleCache:
    """Token-ordered DepthWeave-KV cache for a set of sequences; everything kept as plain numpy arrays."""

    def __init__(self, L, w, H_kv, G, d, tier_ranks, BK, BV, gK, gV, softmax_scale=None):
        assert L % w == 0 and d % GROUP == 0
        self.L, self.w, self.H, self.G, self.d = L, w, H_kv, G, d
        self.tier_ranks = tuple(int(x) for x in tier_ranks)
        self.r = self.tier_ranks[-1]
        self.BK = np.asarray(BK, dtype=np.float64)     # [M,H,r,d]
        self.BV = np.asarray(BV, dtype=np.float64)
        self.gK = np.asarray(gK, dtype=np.float64)     # [L,H,d]
        self.gV = np.asarray(gV, dtype=np.float64)
        assert self.BK.shape == (L // w, H_kv, self.r, d) and self.gK.shape == (L, H_kv, d)
        self.scale = float(softmax_scale) if softmax_scale else 1.0 / np.sqrt(d)      # reading A9
        self.seqs = {}

    def _seq(self, s):
        if s not in self.seqs:
            L, H, r, d = self.L, self.H, self.r, self.d
            self.seqs[s] = dict(
                tier=np.zeros(0, np.uint8), flag=np.zeros(0, np.uint8),
                cls=np.zeros(0, np.int32), slot=np.zeros(0, np.int32), counts=np.zeros(2 * len(self.tier_ranks), np.int64),
                cK=np.zeros((0, L, H, r)), cV=np.zeros((0, L, H, r)),
                codeK=np.zeros((0, L, H, d), np.int8), codeV=np.zeros((0, L, H, d), np.int8),
                scaleK=np.zeros((0, L, H, d // GROUP), np.float16), scaleV=np.zeros((0, L, H, d // GROUP), np.float16))
        return self.seqs[s]

    def seq_len(self, s) -> int:
        return len(self._seq(s)["tier"])

    # -- load path: pre-compressed entries -----------------------------------------------------------------
    def append_raw(self, s, tier, flag, coefK, coefV, residK=None, residV=None,
                   codeK=None, scaleK=None, codeV=None, scaleV=None):
        """coef* [n,L,H,r] (values beyond r_t ignored), residuals for the FLAGGED tokens only, in token order:
        either fp32 resid* [n_flagged,L,H,d] (quantised here, reading A14) or int codes + fp16 scales."""
        S = self._seq(s)
        tier = np.asarray(tier, np.uint8)
        flag = np.asarray(flag, np.uint8)
        n = len(tier)
        L, H, d = self.L, self.H, self.d
        cls, slot, counts = route_slots(tier, flag, len(self.tier_ranks), S["counts"])
        full_code = {z: np.zeros((n, L, H, d), np.int8) for z in "KV"}
        full_scale = {z: np.zeros((n, L, H, d // GROUP), np.float16) for z in "KV"}
        idx = np.nonzero(flag)[0]
        if len(idx):
            for z, resid, code, scale in (("K", residK, codeK, scaleK), ("V", residV, codeV, scaleV)):
                if resid is not None:
                    code, scale = quantize_int4_g16(resid)
                full_code[z][idx] = np.asarray(code, np.int8)
                full_scale[z][idx] = np.asarray(scale, np.float16)
        S["tier"] = np.concatenate([S["tier"], tier]); S["flag"] = np.concatenate([S["flag"], flag])
        S["cls"] = np.concatenate([S["cls"], cls]); S["slot"] = np.concatenate([S["slot"], slot]); S["counts"] = counts
        S["cK"] = np.concatenate([S["cK"], np.asarray(coefK, np.float64)])
        S["cV"] = np.concatenate([S["cV"], np.asarray(coefV, np.float64)])
        for z in "KV":
            S["code" + z] = np.concatenate([S["code" + z], full_code[z]])
            S["scale" + z] = np.concatenate([S["scale" + z], full_scale[z]])

    # -- append / compress from dense K, V (readings A13, A14) ----------------------------------
    def append_compress(self, s, k_new, v_new, tier, flag):
        """k_new, v_new [n,L,H,d] (bf16 values). Returns nothing; entries are appended in token order."""
        tier = np.asarray(tier, np.uint8)
        flag = np.asarray(flag, np.uint8)
        n, L, H, d, r = len(tier), self.L, self.H, self.d, self.r
        coef = {z: np.zeros((n, L, H, r)) for z in "KV"}
        resid = {z: np.zeros((n, L, H, d), np.float32) for z in "KV"}
        for z, x_all, B_all, g_all in (("K", k_new, self.BK, self.gK), ("V", v_new, self.BV, self.gV)):
            x_all = np.asarray(x_all, np.float64)
            for t in range(n):
                rt = self.tier_ranks[tier[t]]
                for l in range(L):
                    for h in range(H):
                        B = B_all[l // self.w, h, :rt, :]                  # leading r_t rows of the shared basis
                        g = g_all[l, h]
                        x = x_all[t, l, h]
                        c = round_to_bf16(B @ (x / g))                     # projection in gate-normalised space
                        coef[z][t, l, h, :rt] = c
                        resid[z][t, l, h] = (x - g * (c @ B)).astype(np.float32)
        fidx = np.nonzero(flag)[0]
        self.append_raw(s, tier, flag, coef["K"], coef["V"],
                        residK=resid["K"][fidx] if len(fidx) else None,
                        residV=resid["V"][fidx] if len(fidx) else None)

    # -- reconstruction and attention ------------------------------------------------------------------------
    # -- re-tiering of stored tokens (reading A29): lowering only ---------------------------
    def retier(self, s, new_tier, new_flag):
        """Every token of sequence s gets the class (new_tier[t], new_flag[t]) <= its stored one. The stored coefficient vector is
        the leading-r_t part of B (x / gate), so the lower tier keeps its leading r' entries; a cleared flag drops the residual.
        Token order is kept and the slots are renumbered per class (route_slots from an empty sequence)."""
        S = self._seq(s)
        new_tier = np.asarray(new_tier, np.uint8)
        new_flag = np.asarray(new_flag, np.uint8)
        assert len(new_tier) == len(S["tier"]) == len(new_flag)
        assert np.all(new_tier <= S["tier"]) and np.all(new_flag <= S["flag"]), "re-tiering only lowers a token"
        ranks = np.asarray(self.tier_ranks)[new_tier]                                    # [n]
        keep = np.arange(self.r)[None, :] < ranks[:, None]                                # [n, r]
        for z in "KV":
            S["c" + z] = np.where(keep[:, None, None, :], S["c" + z], 0.0)
            S["code" + z] = np.where(new_flag[:, None, None, None] != 0, S["code" + z], 0).astype(np.int8)
            S["scale" + z] = np.where(new_flag[:, None, None, None] != 0, S["scale" + z], 0).astype(np.float16)
        S["tier"], S["flag"] = new_tier, new_flag
        S["cls"], S["slot"], S["counts"] = route_slots(new_tier, new_flag, len(self.tier_ranks), None)

    def khat_vhat(self, s, l, h):
        """K-hat, V-hat in R^{T x d} for sequence s, layer l, kv head h (Eq. 1)."""
        S = self._seq(s)
        ranks = np.asarray(self.tier_ranks)[S["tier"]]
        m = l // self.w
        dK = dequant_int4_g16(S["codeK"][:, l, h], S["scaleK"][:, l, h])
        dV = dequant_int4_g16(S["codeV"][:, l, h], S["scaleV"][:, l, h])
        K = reconstruct(S["cK"][:, l, h], ranks, S["flag"], dK, self.BK[m, h], self.gK[l, h])
        V = reconstruct(S["cV"][:, l, h], ranks, S["flag"], dV, self.BV[m, h], self.gV[l, h])
        return K, V

    def decode_attention(self, l, s, q) -> np.ndarray:
        """q [H_q, d] for layer l, sequence s  ->  o [H_q, d] fp64."""
        q = np.asarray(q, np.float64)
        assert self.seq_len(s) > 0, "softmax over an empty sequence is undefined (reading A17)"
        out = np.zeros((self.H * self.G, self.d))
        for h in range(self.H):
            K, V = self.khat_vhat(s, l, h)
            out[h * self.G:(h + 1) * self.G] = softmax_attention(q[h * self.G:(h + 1) * self.G], K, V, self.scale)
        return out

    def decode_all_layers(self, seqs, q) -> np.ndarray:
        """q [n_seq, L, H_q, d] -> o [n_seq, L, H_q, d]."""
        q = np.asarray(q, np.float64)
        out = np.zeros_like(q)
        for i, s in enumerate(seqs):
            for l in range(self.L):
                out[i, l] = self.decode_attention(l, s, q[i, l])
        return out

    def max_abs_vhat(self, s, l) -> float:
        return max(float(np.max(np.abs(self.khat_vhat(s, l, h)[1]))) for h in range(self.H))

    def footprint_bytes(self, s) -> int:
        S = self._seq(s)
        return footprint_bytes(S["tier"], S["flag"], self.tier_ranks, self.d, self.L, self.H)


def footprint_bytes(tier, flag, tier_ranks, d, L, H) -> int:
    """Compressed bytes of one sequence: per (layer, kv head, token) 4*r_t (bf16 cK + cV) plus, if flagged,
    2*(d/2 + d/8) (int4 codes + fp16 group-16 scales for K and V)   (reading A2, pin P13; "8.3x")."""
    ranks = np.asarray(tier_ranks, np.int64)[np.asarray(tier)]
    per = 4 * ranks + np.asarray(flag).astype(np.int64) * 2 * (d // 2 + d // 8)
    return int(per.sum()) * L * H


def attention_slice(coefK, coefV, ranks, flag, codeK, scaleK, codeV, scaleV, BK, BV, gK, gV, q, scale):
    """One (layer, kv head) slice from raw stored arrays; used for sampled full-size parity checks.
    coef* [T,r]; code* [T,d] int8 and scale* [T,d/16] fp16 (rows of unflagged tokens ignored); q [G,d]."""
    dK = dequant_int4_g16(codeK, scaleK) if codeK is not None else None
    dV = dequant_int4_g16(codeV, scaleV) if codeV is not None else None
    K = reconstruct(coefK, ranks, flag, dK, BK, gK)
    V = reconstruct(coefV, ranks, flag, dV, BV, gV)
    return softmax_attention(q, K, V, scale), K, V


def probe_error(attn_ref, attn_cmp, G: int, eps: float) -> np.ndarray:
    """Attention-output probe, Eq. (3):  e[h] = || Attn(Q,K,V) - Attn(Q,K^,V^) ||_2 / ( || Attn(Q,K,V) ||_2 + eps ).

    attn_ref, attn_cmp: [n_q, H_q, d] attention outputs of the n_q probed query positions over the higher-fidelity cache and
    over the compressed reconstruction; the norm of kv head h runs over its G query heads, all positions and all channels
    (reading A25: "a small subset of heads and recent query positions", one number per (layer, kv head))."""
    a = np.asarray(attn_ref, np.float64); b = np.asarray(attn_cmp, np.float64)
    n_q, Hq, d = a.shape
    H = Hq // G
    e = np.zeros(H)
    for h in range(H):
        num = 0.0; den = 0.0
        for i in range(n_q):
            for g in range(G):
                for ch in range(d):
                    x = a[i, h * G + g, ch]; y = b[i, h * G + g, ch]
                    num += (x - y) * (x - y)
                    den += x * x
        e[h] = np.sqrt(num) / (np.sqrt(den) + eps)
    return e
