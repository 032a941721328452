// dwkv_scan.cu -- the decode hot path ("fused kernel"):
//   a1  qprep_kernel    q~ = cscale * BK[m,h] . (gK[l,h] * q)      (q projected into basis space once per step)
//   a2  scan_kernel     split-T online-softmax scan over the class pages, mma.sync bf16 tensor-core contractions
//                       on fragment-native data (dwkv_layout.cuh); K-hat / V-hat are never formed
//   a3  combine_kernel  log-sum-exp merge of the unit partials + back-projection through BV and gV + residual-V term
// Algebra (SURVEY.md section 8 box), log2 domain, cscale = softmax_scale * log2(e):
//   s[hq,t] = sum_{j<r_t} q~[hq,j] cK[t,j] + f_t * cscale * sum_g scaleK[t,g] sum_{i in g} q[hq,i] codeK[t,i]
//   a[hq,j] = sum_t p[t] cV[t,j]      e[hq,i] = sum_{t flagged} p[t] scaleV[t,i/16] codeV[t,i]
//   o[hq,i] = ( gV[l,h,i] * sum_j a[hq,j] BV[m,h,j,i] + e[hq,i] ) / sum_t p[t]
#include "dwkv_internal.h"
#include "dwkv_mma.cuh"

namespace dwkv {

namespace {

using namespace dwkv::dev;

// ---------------------------------------------------------------------------------------------------------------
// a1: q -> basis pre-projection
// ---------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) qprep_kernel(QPrepParams p) {
  __shared__ float qg[8][128];
  const int b = blockIdx.x / p.H, h = blockIdx.x % p.H;
  const int lsel = blockIdx.y, layer = p.layer0 + lsel;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const __nv_bfloat16* gk = p.gK + ((size_t)layer * p.H + h) * p.d;
  const __nv_bfloat16* q = p.q + (((size_t)b * p.Lq + (p.Lq == 1 ? 0 : layer)) * (p.H * p.G) + (size_t)h * p.G) * p.d;
  for (int idx = tid; idx < 8 * p.d; idx += 128) {
    const int g = idx / p.d, i = idx % p.d;
    qg[g][i] = (g < p.G) ? __bfloat162float(q[(size_t)g * p.d + i]) * __bfloat162float(gk[i]) : 0.f;
  }
  __syncthreads();
  const __nv_bfloat16* B = p.BK + ((size_t)(layer / p.w) * p.H + h) * p.r * p.d;
  const size_t ooff = (((size_t)b * p.Lsel + lsel) * p.H + h) * 8 * p.r;
  for (int j = warp; j < p.r; j += 4) {
    float acc[8];
#pragma unroll
    for (int g = 0; g < 8; ++g) acc[g] = 0.f;
    for (int i = lane; i < p.d; i += 32) {
      const float bv = __bfloat162float(B[(size_t)j * p.d + i]);
#pragma unroll
      for (int g = 0; g < 8; ++g) acc[g] = fmaf(bv, qg[g][i], acc[g]);
    }
#pragma unroll
    for (int g = 0; g < 8; ++g) {
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) acc[g] += __shfl_xor_sync(kFull, acc[g], o);
    }
    if (lane < 8) {
      float v = 0.f;
#pragma unroll
      for (int g = 0; g < 8; ++g) v = (lane == g) ? acc[g] : v;
      v *= p.cscale;
      const __nv_bfloat16 hi = __float2bfloat16_rn(v);
      const __nv_bfloat16 lo = __float2bfloat16_rn(v - __bfloat162float(hi));
      p.qt_hi[ooff + (size_t)lane * p.r + j] = hi;
      p.qt_lo[ooff + (size_t)lane * p.r + j] = lo;
    }
  }
}

}  // namespace

// ---------------------------------------------------------------------------------------------------------------
// a2: split-T scan. One CTA (4 warps) per (unit, layer, kv head); warp w takes blocks w, w+4, ... of the unit and
// keeps its own online-softmax state; the four states are merged in shared memory and one partial is written.
// ---------------------------------------------------------------------------------------------------------------
namespace {

template <int NK, bool RESID, int D>
struct ScanState {
  float m, l;
  float acc[NK][2];                    // a[row g][8i + 2t + {0,1}]
  float eacc[RESID ? D / 8 : 1][2];    // e[row g][8c + 2t + {0,1}]
};

template <int NK, bool RESID, int D>
__device__ __forceinline__ void process_block(ScanState<NK, RESID, D>& st, const uint4 (&kc)[NK], const uint4 (&vc)[NK],
                                              const uint8_t* __restrict__ blk, int nv, int lane,
                                              const uint32_t (&qh)[NK], const uint32_t (&ql)[NK],
                                              const uint32_t (&qa)[RESID ? D / 16 : 1][2],
                                              const float (&qbias)[RESID ? D / 16 : 1], float cscale) {
  constexpr int NG = D / 16;
  const int t = lane & 3;
  float s[4][2];
  // ---- scores: S = q~ . cK^T (hi + lo parts of q~), tokens on the MMA n dimension --------------------------------
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    s[j][0] = 0.f;
    s[j][1] = 0.f;
#pragma unroll
    for (int i = 0; i < NK; i += 2) {
      constexpr int kLast = NK - 1;
      const int i1 = (i + 1 < NK) ? i + 1 : kLast;
      const uint32_t k0 = comp(kc[i], j);
      if (i + 1 < NK) {
        const uint32_t k1 = comp(kc[i1], j);
        mma16816(s[j][0], s[j][1], qh[i], qh[i1], k0, k1);
        mma16816(s[j][0], s[j][1], ql[i], ql[i1], k0, k1);
      } else {
        mma1688(s[j][0], s[j][1], qh[i], k0);
        mma1688(s[j][0], s[j][1], ql[i], k0);
      }
    }
  }
  // ---- residual-K term: integer-code dot on the tensor cores, fp32 group scales applied afterwards -----------------
  if constexpr (RESID) {
    constexpr int CB = NK * 1024;
    const uint8_t* codeK = blk + CB;
    const uint8_t* scaleK = blk + CB + 16 * D;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      uint32_t w[D / 32];
      uint32_t sc[NG];
      if constexpr (D == 128) {
        const uint4 c4 = ldg_stream(codeK + j * 4 * D + lane * 16);
        w[0] = c4.x; w[1] = c4.y; w[2] = c4.z; w[3] = c4.w;
        const uint4 s0 = __ldg(reinterpret_cast<const uint4*>(scaleK + j * D + t * 32));
        const uint4 s1 = __ldg(reinterpret_cast<const uint4*>(scaleK + j * D + t * 32 + 16));
        sc[0] = s0.x; sc[1] = s0.y; sc[2] = s0.z; sc[3] = s0.w; sc[4] = s1.x; sc[5] = s1.y; sc[6] = s1.z; sc[7] = s1.w;
      } else {
        const uint2 c2 = __ldg(reinterpret_cast<const uint2*>(codeK + j * 4 * D + lane * 8));
        w[0] = c2.x; w[1] = c2.y;
        const uint4 s0 = __ldg(reinterpret_cast<const uint4*>(scaleK + j * D + t * 16));
        sc[0] = s0.x; sc[1] = s0.y; sc[2] = s0.z; sc[3] = s0.w;
      }
      float sr0 = 0.f, sr1 = 0.f;
#pragma unroll
      for (int grp = 0; grp < NG; ++grp) {
        float c0 = qbias[grp], c1 = qbias[grp];       // -136 * sum_i q_i cancels the offset of the biased codes
        const int q = 2 * grp;
        const uint32_t b0 = nib_to_bf16x2_biased(w[q >> 2], q & 3);
        const uint32_t b1 = nib_to_bf16x2_biased(w[q >> 2], (q & 3) + 1);
        mma16816(c0, c1, qa[grp][0], qa[grp][1], b0, b1);
        const float2 f = h2f2(sc[grp]);
        sr0 = fmaf(c0, f.x, sr0);
        sr1 = fmaf(c1, f.y, sr1);
      }
      s[j][0] = fmaf(cscale, sr0, s[j][0]);
      s[j][1] = fmaf(cscale, sr1, s[j][1]);
    }
  }
  // ---- ragged tail: slots >= nv do not exist ----------------------------------------------------------------------
  if (nv < kBlockTok) {
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      if (8 * j + 2 * t >= nv) s[j][0] = -INFINITY;
      if (8 * j + 2 * t + 1 >= nv) s[j][1] = -INFINITY;
    }
  }
  // ---- online softmax ----------------------------------------------------------------------------------------------
  float mx = fmaxf(fmaxf(fmaxf(s[0][0], s[0][1]), fmaxf(s[1][0], s[1][1])),
                   fmaxf(fmaxf(s[2][0], s[2][1]), fmaxf(s[3][0], s[3][1])));
  mx = fmaxf(mx, __shfl_xor_sync(kFull, mx, 1));
  mx = fmaxf(mx, __shfl_xor_sync(kFull, mx, 2));
  const float m_new = fmaxf(st.m, mx);
  if (__any_sync(kFull, m_new > st.m)) {
    const float corr = ex2(st.m - m_new);      // m = -inf on the first block -> 0
    st.l *= corr;
#pragma unroll
    for (int i = 0; i < NK; ++i) { st.acc[i][0] *= corr; st.acc[i][1] *= corr; }
    if constexpr (RESID) {
#pragma unroll
      for (int c = 0; c < D / 8; ++c) { st.eacc[c][0] *= corr; st.eacc[c][1] *= corr; }
    }
    st.m = m_new;
  }
  float pr[4][2];
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    pr[j][0] = ex2(s[j][0] - st.m);
    pr[j][1] = ex2(s[j][1] - st.m);
    st.l += pr[j][0] + pr[j][1];
  }
  // ---- a += P . cV : tokens on the MMA k dimension ------------------------------------------------------------------
#pragma unroll
  for (int ks = 0; ks < 2; ++ks) {
    const uint32_t a0 = pack_bf16x2(pr[2 * ks][0], pr[2 * ks][1]);
    const uint32_t a2 = pack_bf16x2(pr[2 * ks + 1][0], pr[2 * ks + 1][1]);
#pragma unroll
    for (int i = 0; i < NK; ++i) {
      mma16816(st.acc[i][0], st.acc[i][1], a0, a2, comp(vc[i], 2 * ks), comp(vc[i], 2 * ks + 1));
    }
  }
  // ---- e += (P * scaleV) . codeV -------------------------------------------------------------------------------------
  if constexpr (RESID) {
    constexpr int CB = NK * 1024;
    const uint8_t* codeV = blk + CB + 20 * D;
    const uint8_t* scaleV = blk + CB + 36 * D;
#pragma unroll
    for (int ks = 0; ks < 2; ++ks) {
      uint32_t w[D / 16];
      uint32_t sc0[NG], sc1[NG];
      if constexpr (D == 128) {
        const uint4 c0 = ldg_stream(codeV + ks * 8 * D + lane * 32);
        const uint4 c1 = ldg_stream(codeV + ks * 8 * D + lane * 32 + 16);
        w[0] = c0.x; w[1] = c0.y; w[2] = c0.z; w[3] = c0.w; w[4] = c1.x; w[5] = c1.y; w[6] = c1.z; w[7] = c1.w;
        const uint8_t* sp = scaleV + (2 * ks) * D + t * 32;
        const uint4 x0 = __ldg(reinterpret_cast<const uint4*>(sp));
        const uint4 x1 = __ldg(reinterpret_cast<const uint4*>(sp + 16));
        const uint4 y0 = __ldg(reinterpret_cast<const uint4*>(sp + D));
        const uint4 y1 = __ldg(reinterpret_cast<const uint4*>(sp + D + 16));
        sc0[0] = x0.x; sc0[1] = x0.y; sc0[2] = x0.z; sc0[3] = x0.w; sc0[4] = x1.x; sc0[5] = x1.y; sc0[6] = x1.z; sc0[7] = x1.w;
        sc1[0] = y0.x; sc1[1] = y0.y; sc1[2] = y0.z; sc1[3] = y0.w; sc1[4] = y1.x; sc1[5] = y1.y; sc1[6] = y1.z; sc1[7] = y1.w;
      } else {
        const uint4 c0 = ldg_stream(codeV + ks * 8 * D + lane * 16);
        w[0] = c0.x; w[1] = c0.y; w[2] = c0.z; w[3] = c0.w;
        const uint8_t* sp = scaleV + (2 * ks) * D + t * 16;
        const uint4 x0 = __ldg(reinterpret_cast<const uint4*>(sp));
        const uint4 y0 = __ldg(reinterpret_cast<const uint4*>(sp + D));
        sc0[0] = x0.x; sc0[1] = x0.y; sc0[2] = x0.z; sc0[3] = x0.w;
        sc1[0] = y0.x; sc1[1] = y0.y; sc1[2] = y0.z; sc1[3] = y0.w;
      }
#pragma unroll
      for (int grp = 0; grp < NG; ++grp) {
        const float2 f0 = h2f2(sc0[grp]);
        const float2 f1 = h2f2(sc1[grp]);
        const uint32_t a0 = pack_bf16x2(pr[2 * ks][0] * f0.x, pr[2 * ks][1] * f0.y);
        const uint32_t a2 = pack_bf16x2(pr[2 * ks + 1][0] * f1.x, pr[2 * ks + 1][1] * f1.y);
#pragma unroll
        for (int cc = 0; cc < 2; ++cc) {
          const int c = 2 * grp + cc, q = 2 * c;
          const uint32_t b0 = nib_to_bf16x2(w[q >> 2], q & 3);
          const uint32_t b1 = nib_to_bf16x2(w[q >> 2], (q & 3) + 1);
          mma16816(st.eacc[c][0], st.eacc[c][1], a0, a2, b0, b1);
        }
      }
    }
  }
}

template <int NK, bool RESID, int D, int PF>
__global__ void __launch_bounds__(128) scan_kernel(ScanParams p) {
  constexpr int R = NK * 8;
  constexpr int NG = D / 16;
  constexpr int BB = NK * 1024 + (RESID ? 40 * D : 0);
  const int u = p.unit0 + blockIdx.x;
  const Unit un = p.units[u];
  const int lsel = blockIdx.y / p.H, h = blockIdx.y % p.H;
  const int layer = p.layer0 + lsel;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int g = lane >> 2, t = lane & 3;
  const uint8_t* base = p.arena + un.page_off + (size_t)(layer * p.H + h) * kPageLhBytes + (size_t)un.blk0 * BB;

  // query fragments (A operand: row g = query head g of this kv head, rows >= G are zero)
  uint32_t qh[NK], ql[NK];
  {
    const size_t qoff = (((size_t)un.b * p.Lsel + lsel) * p.H + h) * 8 * p.r + (size_t)g * p.r + 2 * t;
#pragma unroll
    for (int i = 0; i < NK; ++i) {
      qh[i] = *reinterpret_cast<const uint32_t*>(p.qt_hi + qoff + 8 * i);
      ql[i] = *reinterpret_cast<const uint32_t*>(p.qt_lo + qoff + 8 * i);
    }
  }
  uint32_t qa[RESID ? NG : 1][2];
  float qbias[RESID ? NG : 1];
  if constexpr (RESID) {
    const __nv_bfloat16* q = p.q + (((size_t)un.b * p.Lq + (p.Lq == 1 ? 0 : layer)) * (p.H * p.G) + (size_t)h * p.G + g) * D;
#pragma unroll
    for (int grp = 0; grp < NG; ++grp) {
      qa[grp][0] = (g < p.G) ? *reinterpret_cast<const uint32_t*>(q + 16 * grp + 2 * t) : 0u;
      qa[grp][1] = (g < p.G) ? *reinterpret_cast<const uint32_t*>(q + 16 * grp + 8 + 2 * t) : 0u;
      const float2 x = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&qa[grp][0]));
      const float2 y = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&qa[grp][1]));
      float sum = (x.x + x.y) + (y.x + y.y);
      sum += __shfl_xor_sync(kFull, sum, 1);
      sum += __shfl_xor_sync(kFull, sum, 2);
      qbias[grp] = -136.f * sum;
    }
  } else {
    qa[0][0] = qa[0][1] = 0u;
    qbias[0] = 0.f;
  }

  ScanState<NK, RESID, D> st;
  st.m = -INFINITY;
  st.l = 0.f;
#pragma unroll
  for (int i = 0; i < NK; ++i) st.acc[i][0] = st.acc[i][1] = 0.f;
#pragma unroll
  for (int c = 0; c < (RESID ? D / 8 : 1); ++c) st.eacc[c][0] = st.eacc[c][1] = 0.f;

  const int nmy = (un.nblk > warp) ? (un.nblk - warp + 3) / 4 : 0;
  uint4 kb[PF][NK], vb[PF][NK];
  auto load = [&](int k, uint4 (&kk)[NK], uint4 (&vv)[NK]) {
    const uint8_t* bp = base + (size_t)(warp + 4 * k) * BB + lane * 16;
#pragma unroll
    for (int i = 0; i < NK; ++i) {
      kk[i] = ldg_stream(bp + i * 512);
      vv[i] = ldg_stream(bp + NK * 512 + i * 512);
    }
  };
#pragma unroll
  for (int pp = 0; pp < PF; ++pp)
    if (pp < nmy) load(pp, kb[pp], vb[pp]);
  for (int k0 = 0; k0 < nmy; k0 += PF) {
#pragma unroll
    for (int pp = 0; pp < PF; ++pp) {
      const int k = k0 + pp;
      if (k < nmy) {
        uint4 kc[NK], vc[NK];
#pragma unroll
        for (int i = 0; i < NK; ++i) { kc[i] = kb[pp][i]; vc[i] = vb[pp][i]; }
        if (k + PF < nmy) load(k + PF, kb[pp], vb[pp]);
        const int bi = warp + 4 * k;
        const int nv = min(kBlockTok, un.ntok - kBlockTok * bi);
        process_block<NK, RESID, D>(st, kc, vc, base + (size_t)bi * BB, nv, lane, qh, ql, qa, qbias, p.cscale);
      }
    }
  }
  // row sums: every lane of a quad holds a partial of row g
  st.l += __shfl_xor_sync(kFull, st.l, 1);
  st.l += __shfl_xor_sync(kFull, st.l, 2);

  // ---- merge the four warps and write one partial (m, l, a[R], e[D]) per query head ---------------------------------
  __shared__ float sm_m[4][8], sm_l[4][8];
  __shared__ float sm_a[4][8][R];
  __shared__ float sm_e[RESID ? 4 : 1][8][RESID ? D : 1];
  if (t == 0) { sm_m[warp][g] = st.m; sm_l[warp][g] = st.l; }
#pragma unroll
  for (int i = 0; i < NK; ++i) {
    sm_a[warp][g][8 * i + 2 * t] = st.acc[i][0];
    sm_a[warp][g][8 * i + 2 * t + 1] = st.acc[i][1];
  }
  if constexpr (RESID) {
#pragma unroll
    for (int c = 0; c < D / 8; ++c) {
      sm_e[warp][g][8 * c + 2 * t] = st.eacc[c][0];
      sm_e[warp][g][8 * c + 2 * t + 1] = st.eacc[c][1];
    }
  }
  __syncthreads();
  const int G = p.G;
  const int PR = 2 + p.r;
  float* prec = p.part + ((size_t)blockIdx.y * p.n_units_total + u) * (size_t)(G * PR);
  for (int idx = tid; idx < G * (2 + R); idx += 128) {
    const int gq = idx / (2 + R), k = idx % (2 + R);
    const float ms = fmaxf(fmaxf(sm_m[0][gq], sm_m[1][gq]), fmaxf(sm_m[2][gq], sm_m[3][gq]));
    float v = 0.f;
#pragma unroll
    for (int w = 0; w < 4; ++w) {
      const float f = (sm_m[w][gq] == -INFINITY) ? 0.f : ex2(sm_m[w][gq] - ms);
      const float x = (k == 0) ? 0.f : (k == 1) ? sm_l[w][gq] : sm_a[w][gq][k - 2];
      v = fmaf(f, x, v);
    }
    prec[gq * PR + k] = (k == 0) ? ms : v;
  }
  if constexpr (RESID) {
    float* erec = p.epart + ((size_t)blockIdx.y * p.n_eunits_total + un.epart) * (size_t)(G * D);
    for (int idx = tid; idx < G * D; idx += 128) {
      const int gq = idx / D, i = idx % D;
      const float ms = fmaxf(fmaxf(sm_m[0][gq], sm_m[1][gq]), fmaxf(sm_m[2][gq], sm_m[3][gq]));
      float v = 0.f;
#pragma unroll
      for (int w = 0; w < 4; ++w) {
        const float f = (sm_m[w][gq] == -INFINITY) ? 0.f : ex2(sm_m[w][gq] - ms);
        v = fmaf(f, sm_e[w][gq][i], v);
      }
      erec[idx] = v;
    }
  }
}

}  // namespace

// ---------------------------------------------------------------------------------------------------------------
// a3: split-combine + back-projection. One CTA per (sequence, layer, kv head).
// ---------------------------------------------------------------------------------------------------------------
namespace {

constexpr int kCombChunk = 128;

__global__ void __launch_bounds__(128) combine_kernel(CombineParams p) {
  __shared__ float red[16][8];
  __shared__ float mstar[8], lstar[8];
  __shared__ float wbuf[kCombChunk][8];
  __shared__ int u_id[kCombChunk], u_rk[kCombChunk], u_ep[kCombChunk];
  __shared__ float astar[8][64];
  const int b = blockIdx.x, lh = blockIdx.y;
  const int lsel = lh / p.H, h = lh % p.H, layer = p.layer0 + lsel;
  const int tid = threadIdx.x;
  const int G = p.G, r = p.r, d = p.d, PR = 2 + p.r;
  const int u0 = p.ustart[b], n = p.ustart[b + 1] - u0;
  const float* part = p.part + (size_t)lh * p.n_units_total * (size_t)(G * PR);
  const float* epart = p.epart + (size_t)lh * p.n_eunits_total * (size_t)(G * d);

  // m* per query head
  {
    const int gq = tid & 7, sl = tid >> 3;
    float mx = -INFINITY;
    if (gq < G)
      for (int k = sl; k < n; k += 16) mx = fmaxf(mx, part[(size_t)p.ulist[u0 + k] * (G * PR) + gq * PR]);
    red[sl][gq] = mx;
    __syncthreads();
    if (tid < 8) {
      float v = red[0][tid];
      for (int s2 = 1; s2 < 16; ++s2) v = fmaxf(v, red[s2][tid]);
      mstar[tid] = v;
    }
    __syncthreads();
  }
  float lacc = 0.f;          // thread tid < G
  float areg[4] = {0.f, 0.f, 0.f, 0.f};   // elements idx = tid + 128*x of the G x r matrix a*
  float ereg[8];             // thread i < d : e*[gq][i]
#pragma unroll
  for (int gq = 0; gq < 8; ++gq) ereg[gq] = 0.f;

  for (int c0 = 0; c0 < n; c0 += kCombChunk) {
    const int nc = min(kCombChunk, n - c0);
    if (tid < nc) {
      const int uid = p.ulist[u0 + c0 + tid];
      u_id[tid] = uid;
      u_rk[tid] = p.units[uid].rk;
      u_ep[tid] = p.units[uid].epart;
      for (int gq = 0; gq < G; ++gq) wbuf[tid][gq] = ex2(part[(size_t)uid * (G * PR) + gq * PR] - mstar[gq]);
    }
    __syncthreads();
    if (tid < G)
      for (int k = 0; k < nc; ++k) lacc = fmaf(wbuf[k][tid], part[(size_t)u_id[k] * (G * PR) + tid * PR + 1], lacc);
#pragma unroll
    for (int x = 0; x < 4; ++x) {
      const int idx = tid + 128 * x;
      if (idx < G * r) {
        const int gq = idx / r, j = idx % r;
        float a = areg[x];
        for (int k = 0; k < nc; ++k)
          if (j < u_rk[k]) a = fmaf(wbuf[k][gq], part[(size_t)u_id[k] * (G * PR) + gq * PR + 2 + j], a);
        areg[x] = a;
      }
    }
    if (tid < d) {
      for (int k = 0; k < nc; ++k) {
        const int ep = u_ep[k];
        if (ep >= 0) {
          const float* e = epart + (size_t)ep * (G * d) + tid;
#pragma unroll
          for (int gq = 0; gq < 8; ++gq)
            if (gq < G) ereg[gq] = fmaf(wbuf[k][gq], e[gq * d], ereg[gq]);
        }
      }
    }
    __syncthreads();
  }
  if (tid < G) lstar[tid] = lacc;
#pragma unroll
  for (int x = 0; x < 4; ++x) {
    const int idx = tid + 128 * x;
    if (idx < G * r) astar[idx / r][idx % r] = areg[x];
  }
  __syncthreads();
  if (tid < d) {
    const __nv_bfloat16* BV = p.BV + ((size_t)(layer / p.w) * p.H + h) * (size_t)r * d + tid;
    const float gv = __bfloat162float(p.gV[((size_t)layer * p.H + h) * d + tid]);
    float acc[8];
#pragma unroll
    for (int gq = 0; gq < 8; ++gq) acc[gq] = 0.f;
    for (int j = 0; j < r; ++j) {
      const float bv = __bfloat162float(BV[(size_t)j * d]);
#pragma unroll
      for (int gq = 0; gq < 8; ++gq) acc[gq] = fmaf(astar[gq][j], bv, acc[gq]);
    }
    float* out = p.out + (((size_t)b * p.Lq + (p.Lq == 1 ? 0 : layer)) * (p.H * G) + (size_t)h * G) * d + tid;
#pragma unroll
    for (int gq = 0; gq < 8; ++gq)
      if (gq < G) out[(size_t)gq * d] = (gv * acc[gq] + ereg[gq]) / lstar[gq];
  }
}

template <int NK, bool RESID, int D, int PF>
void launch_scan_t(const ScanParams& p, int n_units, cudaStream_t s) {
  dim3 grid(n_units, p.Lsel * p.H);
  scan_kernel<NK, RESID, D, PF><<<grid, 128, 0, s>>>(p);
}

template <bool RESID, int D>
bool launch_scan_nk(const ScanParams& p, int nk, int n_units, cudaStream_t s) {
  switch (nk) {
    case 1: launch_scan_t<1, RESID, D, RESID ? 1 : 4>(p, n_units, s); return true;
    case 2: launch_scan_t<2, RESID, D, RESID ? 1 : 2>(p, n_units, s); return true;
    case 3: launch_scan_t<3, RESID, D, 1>(p, n_units, s); return true;
    case 4: launch_scan_t<4, RESID, D, 1>(p, n_units, s); return true;
    case 5: launch_scan_t<5, RESID, D, 1>(p, n_units, s); return true;
    case 6: launch_scan_t<6, RESID, D, 1>(p, n_units, s); return true;
    case 7: launch_scan_t<7, RESID, D, 1>(p, n_units, s); return true;
    case 8: launch_scan_t<8, RESID, D, 1>(p, n_units, s); return true;
  }
  return false;
}

}  // namespace

int launch_qprep(const QPrepParams& p, cudaStream_t s) {
  dim3 grid(p.n_seqs * p.H, p.Lsel);
  qprep_kernel<<<grid, 128, 0, s>>>(p);
  return 1;
}

int launch_scan(const ScanParams& p, int cls_rank, int resid, int n_units, int /*variant*/, cudaStream_t s) {
  if (n_units <= 0) return 0;
  const int nk = cls_rank / 8;
  bool ok;
  if (resid) return 0;   // v1 (one CTA per unit) serves unflagged classes only; flagged classes use the persistent kernel
  ok = launch_scan_nk<false, 128>(p, nk, n_units, s);   // D is irrelevant without the residual
  return ok ? 1 : 0;
}

int launch_combine(const CombineParams& p, int n_seqs, cudaStream_t s) {
  dim3 grid(n_seqs, p.Lsel * p.H);
  combine_kernel<<<grid, 128, 0, s>>>(p);
  return 1;
}

}  // namespace dwkv
