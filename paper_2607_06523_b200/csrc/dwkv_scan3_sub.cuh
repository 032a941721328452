// dwkv_scan3_sub.cuh -- one sub-block (32 slots, or 16 slots of a flagged class) of the split-T scan, from shared memory.
#pragma once
#include "dwkv_scan3.cuh"

namespace dwkv {
namespace s3 {

template <int D>
__device__ __forceinline__ void lds_scales(uint32_t (&sc)[D / 16], uint32_t base, int tile, int t) {
  if constexpr (D == 128) {
    const uint4 s0 = lds128(base + tile * D + t * 32), s1 = lds128(base + tile * D + t * 32 + 16);
    sc[0] = s0.x; sc[1] = s0.y; sc[2] = s0.z; sc[3] = s0.w; sc[4] = s1.x; sc[5] = s1.y; sc[6] = s1.z; sc[7] = s1.w;
  } else {
    const uint4 s0 = lds128(base + tile * D + t * 16);
    sc[0] = s0.x; sc[1] = s0.y; sc[2] = s0.z; sc[3] = s0.w;
  }
}
template <int D>
__device__ __forceinline__ void lds_kcodes(uint32_t (&w)[D / 32], uint32_t base, int tile, int lane) {
  if constexpr (D == 128) {
    const uint4 c = lds128(base + tile * 4 * D + lane * 16);
    w[0] = c.x; w[1] = c.y; w[2] = c.z; w[3] = c.w;
  } else {
    const uint2 c = lds64(base + tile * 4 * D + lane * 8);
    w[0] = c.x; w[1] = c.y;
  }
}

// NK = rank / 8 of the class, RESID = flagged class, NKB / D / PAIR = kernel instance (see State / QRegs), I8 = 8-bit coefficient
// planes (dwkv_layout.cuh): codes are widened to exact 16-bit floating integers in registers (K: fp16, the score MMA runs in fp16
// with q~ split hi + lo in fp16; V: bf16, because p * 2^e needs the bf16 exponent range), the token's power-of-two scale multiplies its
// score after the MMA and its p before the value MMA -- the contractions themselves are unchanged.
// RAGGED = the sub-block may hold fewer than 8 * TB valid tokens (only the last sub-block of a unit can): the full ones skip the checks
template <int NK, bool RESID, int NKB, int D, bool PAIR, bool I8, bool RAGGED>
__device__ __forceinline__ void process_sub(State<NKB, D>& st, const uint32_t sp, const int nv, const int lane,
                                            const QRegs<NKB, D, PAIR>& q, const float cscale) {
  constexpr int NBK = (NK + 3) / 4;                // 8-bit planes: 32-column blocks of the class rank, one exponent byte per slot and block
  constexpr int TB = RESID ? 2 : 4, NG = D / 16, COEF = I8 ? NK * 64 * TB + NBK * 8 * TB : NK * 128 * TB;
  constexpr int NSC = PAIR ? TB / 2 : TB;          // score pairs held by a lane
  const int g = lane >> 2, t = lane & 3;
  const int jt = PAIR ? (g >> 2) : 0;              // PAIR: token tile parity of this lane's row
  const uint32_t mA = (g < 4) ? 0xffffffffu : 0u;  // PAIR: lane belongs to a tile-A row
  uint32_t kw[NK][TB], vw[NK][TB];
  float ksc[NBK][NSC][2], vsc[NBK][NSC][2];      // I8: 2^e (per block) of the tokens behind s[x][0], s[x][1]
  if constexpr (I8) {
#pragma unroll
    for (int i = 0; i < NK; ++i) {
      if constexpr (TB == 4) {
        const uint2 a = lds64(sp + i * 256 + lane * 8);
        const uint2 b = lds64(sp + COEF + i * 256 + lane * 8);
        kw[i][0] = u8pair_to_f16x2(a.x, 0); kw[i][1] = u8pair_to_f16x2(a.x, 1); kw[i][2] = u8pair_to_f16x2(a.y, 0); kw[i][3] = u8pair_to_f16x2(a.y, 1);
        vw[i][0] = u8pair_to_bf16x2(b.x, 0); vw[i][1] = u8pair_to_bf16x2(b.x, 1); vw[i][2] = u8pair_to_bf16x2(b.y, 0); vw[i][3] = u8pair_to_bf16x2(b.y, 1);
      } else {
        const uint32_t a = lds32(sp + i * 128 + lane * 4);
        const uint32_t b = lds32(sp + COEF + i * 128 + lane * 4);
        kw[i][0] = u8pair_to_f16x2(a, 0); kw[i][1] = u8pair_to_f16x2(a, 1);
        vw[i][0] = u8pair_to_bf16x2(b, 0); vw[i][1] = u8pair_to_bf16x2(b, 1);
      }
    }
#pragma unroll
    for (int bk = 0; bk < NBK; ++bk) {
      uint32_t ek[2], ev[2];             // exponent bytes of lane t: (tile j, hi) at byte 2j + hi
      if constexpr (TB == 4) {
        const uint2 a = lds64(sp + NK * 256 + bk * 32 + t * 8), b = lds64(sp + COEF + NK * 256 + bk * 32 + t * 8);
        ek[0] = a.x; ek[1] = a.y; ev[0] = b.x; ev[1] = b.y;
      } else {
        ek[0] = lds32(sp + NK * 128 + bk * 16 + t * 4); ev[0] = lds32(sp + COEF + NK * 128 + bk * 16 + t * 4);
        ek[1] = 0u; ev[1] = 0u;
      }
#pragma unroll
      for (int x = 0; x < NSC; ++x) {    // PAIR: s[x] is tile 2x + jt; FULL: tile x
        const int wi = PAIR ? x : (x >> 1);
        const int sh = PAIR ? 16 * jt : 16 * (x & 1);
        ksc[bk][x][0] = exp_byte_to_scale(ek[wi], sh); ksc[bk][x][1] = exp_byte_to_scale(ek[wi], sh + 8);
        vsc[bk][x][0] = exp_byte_to_scale(ev[wi], sh); vsc[bk][x][1] = exp_byte_to_scale(ev[wi], sh + 8);
      }
    }
  } else {
#pragma unroll
  for (int i = 0; i < NK; ++i) {
    if constexpr (TB == 4) {
      const uint4 a = lds128(sp + i * 512 + lane * 16);
      const uint4 b = lds128(sp + COEF + i * 512 + lane * 16);
      kw[i][0] = a.x; kw[i][1] = a.y; kw[i][2] = a.z; kw[i][3] = a.w;
      vw[i][0] = b.x; vw[i][1] = b.y; vw[i][2] = b.z; vw[i][3] = b.w;
    } else {
      const uint2 a = lds64(sp + i * 256 + lane * 8);
      const uint2 b = lds64(sp + COEF + i * 256 + lane * 8);
      kw[i][0] = a.x; kw[i][1] = a.y;
      vw[i][0] = b.x; vw[i][1] = b.y;
    }
  }
  }
  // ---- scores relative to the reference: s' = q~ . cK - m_ref, hi and lo parts of q~ on MMA rows r and r + 8 ----------
  const float cinit = st.cq[0];
  float s[NSC][2];
#pragma unroll
  for (int x = 0; x < NSC; ++x) {
    if constexpr (I8) {      // integer-valued code dots per 32-column block, the block's power-of-two scale afterwards
      s[x][0] = cinit; s[x][1] = cinit;
#pragma unroll
      for (int bk = 0; bk < NBK; ++bk) {
        const int i0 = 4 * bk, i1 = (4 * bk + 4 < NK) ? 4 * bk + 4 : NK;
        float c[4] = {0.f, 0.f, 0.f, 0.f};
        if constexpr (PAIR) {
#pragma unroll
          for (int i = 0; i < NK; ++i)
            if (i >= i0 && i < i1) mma16h(c, q.qa[i][0], q.qa[i][1], q.qa[i][2], q.qa[i][3], kw[i][2 * x], kw[i][2 * x + 1]);
        } else {
#pragma unroll
          for (int pi = 0; pi < NK / 2; ++pi)
            if (2 * pi >= i0 && 2 * pi < i1) mma16h(c, q.qa[2 * pi][0], q.qa[2 * pi][1], q.qa[2 * pi + 1][0], q.qa[2 * pi + 1][1], kw[2 * pi][x], kw[2 * pi + 1][x]);
          if constexpr (NK & 1)
            if (NK - 1 >= i0 && NK - 1 < i1) mma8h(c, q.qa[NK - 1][0], q.qa[NK - 1][1], kw[NK - 1][x]);
        }
        s[x][0] = fmaf(ksc[bk][x][0], c[0] + c[2], s[x][0]);
        s[x][1] = fmaf(ksc[bk][x][1], c[1] + c[3], s[x][1]);
      }
    } else {
    float c[4];              // the first MMA of the chain takes C = (-m_ref, -m_ref, 0, 0) from the state's own registers
    if constexpr (PAIR) {    // k = (tile 2x: 8 rank columns | tile 2x+1: 8 rank columns), block-diagonal A
      mma16c(c, q.qa[0][0], q.qa[0][1], q.qa[0][2], q.qa[0][3], kw[0][2 * x], kw[0][2 * x + 1], st.cq);
#pragma unroll
      for (int i = 1; i < NK; ++i) mma16(c, q.qa[i][0], q.qa[i][1], q.qa[i][2], q.qa[i][3], kw[i][2 * x], kw[i][2 * x + 1]);
    } else {                 // k = 16 rank columns of tile x
      if constexpr (NK >= 2) {
        mma16c(c, q.qa[0][0], q.qa[0][1], q.qa[1][0], q.qa[1][1], kw[0][x], kw[1][x], st.cq);
#pragma unroll
        for (int pi = 1; pi < NK / 2; ++pi)
          mma16(c, q.qa[2 * pi][0], q.qa[2 * pi][1], q.qa[2 * pi + 1][0], q.qa[2 * pi + 1][1], kw[2 * pi][x], kw[2 * pi + 1][x]);
        if constexpr (NK & 1) mma8(c, q.qa[NK - 1][0], q.qa[NK - 1][1], kw[NK - 1][x]);
      } else {
        mma8c(c, q.qa[0][0], q.qa[0][1], kw[0][x], st.cq);
      }
    }
    s[x][0] = c[0] + c[2];
    s[x][1] = c[1] + c[3];
    }
  }
  // ---- residual-K term: exact integer-code dot on the tensor cores (biased codes, bias folded into C), fp32 scales ----
  if constexpr (RESID) {
    const uint32_t codeK = sp + 2 * COEF, scaleK = codeK + 8 * D;
    if constexpr (PAIR) {
      uint32_t wA[D / 32], wB[D / 32], sc[NG];
      lds_kcodes<D>(wA, codeK, 0, lane);
      lds_kcodes<D>(wB, codeK, 1, lane);
      lds_scales<D>(sc, scaleK, jt, t);
      float sr0 = 0.f, sr1 = 0.f;
#pragma unroll
      for (int grp = 0; grp < NG; ++grp) {
        const int qq = 2 * grp;
        float c1[4], c2[4];     // one A quad for both products: tile A reads rows g (c1[0..1]), tile B rows g+8 (c2[2..3])
        mma16z(c1, q.qr[grp][0], q.qr[grp][1], q.qr[grp][2], q.qr[grp][3], nib_to_bf16x2_biased(wA[qq >> 2], qq & 3),
               nib_to_bf16x2_biased(wA[qq >> 2], (qq & 3) + 1));
        mma16z(c2, q.qr[grp][0], q.qr[grp][1], q.qr[grp][2], q.qr[grp][3], nib_to_bf16x2_biased(wB[qq >> 2], qq & 3),
               nib_to_bf16x2_biased(wB[qq >> 2], (qq & 3) + 1));
        const float2 f = h2f2(sc[grp]);
        sr0 = fmaf((c1[0] + c2[2]) + q.qbias[grp], f.x, sr0);      // the -136 * sum(q) offset of the biased codes
        sr1 = fmaf((c1[1] + c2[3]) + q.qbias[grp], f.y, sr1);
      }
      s[0][0] = fmaf(cscale, sr0, s[0][0]);
      s[0][1] = fmaf(cscale, sr1, s[0][1]);
    } else {
#pragma unroll
      for (int j = 0; j < TB; ++j) {
        uint32_t w[D / 32], sc[NG];
        lds_kcodes<D>(w, codeK, j, lane);
        lds_scales<D>(sc, scaleK, j, t);
        float sr0 = 0.f, sr1 = 0.f;
#pragma unroll
        for (int grp = 0; grp < NG; ++grp) {
          const int qq = 2 * grp;
          float c[4];             // the quad holds groups 2p (rows g) and 2p + 1 (rows g+8): take the rows of this group
          mma16z(c, q.qr[grp >> 1][0], q.qr[grp >> 1][1], q.qr[grp >> 1][2], q.qr[grp >> 1][3], nib_to_bf16x2_biased(w[qq >> 2], qq & 3),
                 nib_to_bf16x2_biased(w[qq >> 2], (qq & 3) + 1));
          const float2 f = h2f2(sc[grp]);
          sr0 = fmaf(c[2 * (grp & 1)] + q.qbias[grp], f.x, sr0);
          sr1 = fmaf(c[2 * (grp & 1) + 1] + q.qbias[grp], f.y, sr1);
        }
        s[j][0] = fmaf(cscale, sr0, s[j][0]);
        s[j][1] = fmaf(cscale, sr1, s[j][1]);
      }
    }
  }
  if constexpr (RAGGED) {   // ragged tail: slots >= nv do not exist
#pragma unroll
    for (int x = 0; x < NSC; ++x) {
      const int slot = PAIR ? (16 * x + 8 * jt + 2 * t) : (8 * x + 2 * t);
      if (slot >= nv) s[x][0] = -INFINITY;
      if (slot + 1 >= nv) s[x][1] = -INFINITY;
    }
  }
  // ---- lazy online softmax (per MMA row) -----------------------------------------------------------------------------
  float mx = fmaxf(s[0][0], s[0][1]);
#pragma unroll
  for (int x = 1; x < NSC; ++x) mx = fmaxf(mx, fmaxf(s[x][0], s[x][1]));
  if (__any_sync(kFull, mx > st.thr)) {
    mx = fmaxf(mx, __shfl_xor_sync(kFull, mx, 1));
    mx = fmaxf(mx, __shfl_xor_sync(kFull, mx, 2));
    const bool unref = st.thr == -INFINITY, none = mx == -INFINITY;
    // The reference is kept INTEGER-valued (log2 units): references of different work splits then differ by whole powers of two, so
    // p = 2^(s - m), its hi + lo split and the bf16 rounding of the p * scaleV operand scale exactly and the result no longer depends
    // on where the slices were cut beyond fp32 summation order (pin P11)
    mx = ceilf(mx);
    const float up = unref ? (none ? 0.f : mx) : fmaxf(mx, 0.f);   // new reference = old reference + up
    const float corr = unref ? 1.f : ex2(-up);
    st.m = unref ? (none ? -INFINITY : mx) : st.m + up;
    st.thr = (unref && none) ? -INFINITY : kLazy;
    st.cq[0] = st.cq[1] = (st.thr == -INFINITY) ? st.cq[2] : -st.m;
    st.l *= corr;
#pragma unroll
    for (int i = 0; i < NKB; ++i) { st.acc[i][0] *= corr; st.acc[i][1] *= corr; st.acc[i][2] *= corr; st.acc[i][3] *= corr; }
    {   // e is held transposed: this lane's columns 2t, 2t+1 belong to rows 2t, 2t+1 (lanes 8t, 8t+4)
      const float c0 = __shfl_sync(kFull, corr, 8 * t), c1 = __shfl_sync(kFull, corr, 8 * t + 4);
#pragma unroll
      for (int grp = 0; grp < NG; ++grp) {
        st.eacc[grp][0] *= c0; st.eacc[grp][1] *= c1; st.eacc[grp][2] *= c0; st.eacc[grp][3] *= c1;
      }
    }
#pragma unroll
    for (int x = 0; x < NSC; ++x) { s[x][0] -= up; s[x][1] -= up; }
  }
  float pr[NSC][2];
#pragma unroll
  for (int x = 0; x < NSC; ++x) {
    pr[x][0] = ex2(s[x][0]);
    pr[x][1] = ex2(s[x][1]);
    st.l += pr[x][0] + pr[x][1];
  }
  // ---- a += P . cV, p = hi + lo on MMA rows r and r + 8 -------------------------------------------------------------------
  if constexpr (PAIR) {
#pragma unroll
    for (int x = 0; x < NSC; ++x) {
#pragma unroll
      for (int bk = 0; bk < (I8 ? NBK : 1); ++bk) {      // 8-bit planes: p * 2^e of the block that the rank chunks belong to
        uint32_t ph, pl;
        if constexpr (I8) split_bf16x2(pr[x][0] * vsc[bk][x][0], pr[x][1] * vsc[bk][x][1], ph, pl);
        else split_bf16x2(pr[x][0], pr[x][1], ph, pl);
        const uint32_t a0 = ph & mA, a1 = pl & mA, a2 = ph & ~mA, a3 = pl & ~mA;
#pragma unroll
        for (int i = 0; i < NK; ++i)
          if (!I8 || (i >> 2) == bk) mma16(st.acc[i], a0, a1, a2, a3, vw[i][2 * x], vw[i][2 * x + 1]);
      }
    }
  } else {
#pragma unroll
    for (int ks = 0; ks < TB / 2; ++ks) {
#pragma unroll
      for (int bk = 0; bk < (I8 ? NBK : 1); ++bk) {
        uint32_t a0, a1, a2, a3;
        if constexpr (I8) {
          split_bf16x2(pr[2 * ks][0] * vsc[bk][2 * ks][0], pr[2 * ks][1] * vsc[bk][2 * ks][1], a0, a1);
          split_bf16x2(pr[2 * ks + 1][0] * vsc[bk][2 * ks + 1][0], pr[2 * ks + 1][1] * vsc[bk][2 * ks + 1][1], a2, a3);
        } else {
          split_bf16x2(pr[2 * ks][0], pr[2 * ks][1], a0, a1);
          split_bf16x2(pr[2 * ks + 1][0], pr[2 * ks + 1][1], a2, a3);
        }
#pragma unroll
        for (int i = 0; i < NK; ++i)
          if (!I8 || (i >> 2) == bk) mma16(st.acc[i], a0, a1, a2, a3, vw[i][2 * ks], vw[i][2 * ks + 1]);
      }
    }
  }
  // ---- e^T += codeV^T . (P * scaleV): channels on the MMA m dimension, rows/heads on n ----------------------------------
  if constexpr (RESID) {
    const uint32_t codeV = sp + 2 * COEF + 10 * D, scaleV = codeV + 8 * D;
    uint32_t w[NG];
    if constexpr (D == 128) {
      const uint4 c0 = lds128(codeV + lane * 32), c1 = lds128(codeV + lane * 32 + 16);
      w[0] = c0.x; w[1] = c0.y; w[2] = c0.z; w[3] = c0.w; w[4] = c1.x; w[5] = c1.y; w[6] = c1.z; w[7] = c1.w;
    } else {
      const uint4 c0 = lds128(codeV + lane * 16);
      w[0] = c0.x; w[1] = c0.y; w[2] = c0.z; w[3] = c0.w;
    }
    constexpr uint32_t neg136 = 0xC308C308u;   // bf16 pair (-136, -136)
    if constexpr (PAIR) {
      uint32_t sc[NG];
      lds_scales<D>(sc, scaleV, jt, t);
#pragma unroll
      for (int grp = 0; grp < NG; ++grp) {
        const float2 f = h2f2(sc[grp]);
        const uint32_t xb = pack_bf16x2(pr[0][0] * f.x, pr[0][1] * f.y);
        const uint32_t b0 = xb & mA, b1 = xb & ~mA;
        mma16(st.eacc[grp], nib_to_bf16x2_biased(w[grp], 0), nib_to_bf16x2_biased(w[grp], 1),
              nib_to_bf16x2_biased(w[grp], 2), nib_to_bf16x2_biased(w[grp], 3), b0, b1);
        mma16(st.eacc[grp], neg136, neg136, neg136, neg136, b0, b1);   // removes the 136 offset on the tensor pipe
      }
    } else {
      uint32_t sc0[NG], sc1[NG];
      lds_scales<D>(sc0, scaleV, 0, t);
      lds_scales<D>(sc1, scaleV, 1, t);
#pragma unroll
      for (int grp = 0; grp < NG; ++grp) {
        const float2 f0 = h2f2(sc0[grp]), f1 = h2f2(sc1[grp]);
        const uint32_t b0 = pack_bf16x2(pr[0][0] * f0.x, pr[0][1] * f0.y);
        const uint32_t b1 = pack_bf16x2(pr[1][0] * f1.x, pr[1][1] * f1.y);
        mma16(st.eacc[grp], nib_to_bf16x2_biased(w[grp], 0), nib_to_bf16x2_biased(w[grp], 1),
              nib_to_bf16x2_biased(w[grp], 2), nib_to_bf16x2_biased(w[grp], 3), b0, b1);
        mma16(st.eacc[grp], neg136, neg136, neg136, neg136, b0, b1);
      }
    }
  }
}

}  // namespace s3
}  // namespace dwkv
