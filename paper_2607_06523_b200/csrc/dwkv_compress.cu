// dwkv_compress.cu -- a4: append / compress on the tensor cores (PAPER.md:56
// "projecting the original cache vector onto the current basis"; readings A13, A14).
//
// For a tile of 16 new tokens and one (layer, kv head), per Z in {K, V}:
//   C   = X . B'^T             [16 x r]   B'[j][i] = B[j][i] / g[i] (fp32 IEEE division), split hi + mid + lo bf16 (24 bits)
//                                         once per (layer, head) and CTA; x is bf16 already, so the A operand needs no work
//   c   = bf16(C), columns >= r_t of a token dropped (leading-r_t coefficients of its tier)
//   rec = c . B                [16 x d]   exact bf16 products, fp32 accumulate     (only if a token of the tile is flagged)
//   e   = x - g * rec  ->  int4 / group 16 / fp16 scale  (quantiser A14, fp32 IEEE, no reciprocal)
// Persistent grid: the (layer-head, tile) items are cut into equal-cost contiguous ranges, one per CTA (a flagged tile counts
// kCostFlag, an unflagged one kCostPlain); a CTA stages B' of its current (layer, head) in shared memory in the register
// order of the MMA B fragments (one 16-byte + one 8-byte ld.shared per MMA triple) and its 8 warps take tiles round-robin.
// The contraction index of the projection is permuted so that a lane's A fragments are plain 16-byte global loads of its
// token rows; the loads of the next Z / next tile are in flight while the current one is multiplied. Results go straight
// to their fragment-native positions in the class pages (dwkv_layout.cuh): every 32-bit coefficient word, 16-byte K-code row,
// V-code byte and scale is owned by exactly one (token, lane), so no atomics are needed (pages are zeroed when allocated).
#include <algorithm>

#include "dwkv_internal.h"
#include "dwkv_mma.cuh"

namespace dwkv {
namespace {
using namespace dwkv::dev;

constexpr int kCostFlag = 4, kCostPlain = 1;   // relative cost of a tile with / without the reconstruction + quantiser part
constexpr int kCompressWarps = 12;

__device__ __forceinline__ void mma16(float (&d)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t b0, uint32_t b1) {
  asm("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
      : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
      : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
__device__ __forceinline__ void mma8(float (&d)[4], uint32_t a0, uint32_t a1, uint32_t b0) {
  asm("mma.sync.aligned.m16n8k8.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5}, {%6}, {%0,%1,%2,%3};"
      : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
      : "r"(a0), "r"(a1), "r"(b0));
}
__device__ __forceinline__ float2 bf2(uint32_t w) { return make_float2(__uint_as_float(w << 16), __uint_as_float(w & 0xffff0000u)); }
// (x, y) = hi + mid + lo, three bf16 terms = 24 significant bits: the projection keeps fp32 accuracy on the tensor cores
// (a near-cancelling dot product would otherwise miss the correctly rounded bf16 coefficient by more than one ulp)
__device__ __forceinline__ void split3(float x, float y, uint32_t& hi, uint32_t& mid, uint32_t& lo) {
  hi = pack_bf16x2(x, y);
  const float rx = x - __uint_as_float(hi << 16), ry = y - __uint_as_float(hi & 0xffff0000u);
  mid = pack_bf16x2(rx, ry);
  lo = pack_bf16x2(rx - __uint_as_float(mid << 16), ry - __uint_as_float(mid & 0xffff0000u));
}

// Reading A14: fp32 IEEE, round-to-nearest-even, no FMA contraction, no reciprocal.
__device__ __forceinline__ int quant_code(float e, float sf) {
  if (sf == 0.f) return 0;
  float r = rintf(__fdiv_rn(e, sf));
  r = fminf(fmaxf(r, -7.f), 7.f);
  return (int)r;
}
__device__ __forceinline__ __half quant_scale(float amax) {
  float s32 = __fdiv_rn(amax, 7.0f);
  s32 = fminf(s32, 65504.0f);
  return __float2half_rn(s32);
}

struct RowDst {          // destination of one token row of the tile for this (layer, head), packed to 4 registers
  uint8_t* blk;          // sub-block base
  int meta;              // slot inside the sub-block | rank of the token's tier << 8 | valid << 16 | flagged << 17
  int src;               // row of the token in k_new / v_new
  __device__ __forceinline__ int slot() const { return meta & 0xff; }
  __device__ __forceinline__ int rk() const { return (meta >> 8) & 0xff; }
  __device__ __forceinline__ bool valid() const { return (meta >> 16) & 1; }
  __device__ __forceinline__ bool flagged() const { return (meta >> 17) & 1; }
  __device__ __forceinline__ int tb() const { return flagged() ? 2 : 4; }          // tiles per sub-block
  __device__ __forceinline__ int coef_bytes() const { return rk() * 16 * tb(); }    // bytes of [K coef] (= [V coef])
};

// the ClassLayout arithmetic of dwkv_layout.cuh with shifts only (tb is 2 or 4); tier ranks come as 4 bytes of one word
__device__ __forceinline__ RowDst row_dst(const uint8_t* arena, const uint32_t ranks4, const int d, const TokDst* dst, int tok, int n_tok, int lh) {
  RowDst r;
  const bool valid = tok < n_tok;
  const TokDst td = dst[valid ? tok : 0];
  const int resid = td.cls & 1;
  const int rk = (ranks4 >> (8 * (td.cls >> 1))) & 0xff;
  const int tb = resid ? 2 : 4;
  const int coef_bytes = rk * 16 * tb;
  const int sub_bytes = 2 * coef_bytes + (resid ? 2 * 5 * tb * d : 0);
  const int block_bytes = resid ? 2 * sub_bytes : sub_bytes;
  r.src = valid ? td.src : 0;
  r.blk = const_cast<uint8_t*>(arena) + td.page_off + (size_t)lh * kPageLhBytes + (size_t)td.blk * block_bytes +
          ((resid && td.slot >= 16) ? sub_bytes : 0);
  r.meta = (resid ? (td.slot & 15) : td.slot) | (rk << 8) | ((int)valid << 16) | ((int)(valid && resid) << 17);
  return r;
}

// item position in cost space -> (layer-head, tile). Per layer-head: nf flagged tiles first (cost kCostFlag each), then plain ones.
__device__ __forceinline__ void cost_to_item(long long pos, int per_lh, int nf, int nt_lh, int* lh, int* tile) {
  *lh = (int)(pos / per_lh);
  const int rem = (int)(pos - (long long)*lh * per_lh);
  *tile = rem < nf * kCostFlag ? rem / kCostFlag : min(nt_lh, nf + (rem - nf * kCostFlag) / kCostPlain);
}

template <int D>
__device__ __forceinline__ void load_x(const __nv_bfloat16* X, const RowDst& ra, const RowDst& rb, int LH, int lh, int t,
                                       uint4 (&xa)[D / 32], uint4 (&xb)[D / 32]) {
  // lane (g, t) takes channels 32u + 8t .. +7 of rows g and g+8: with the permuted contraction index these are the A registers
  const uint4* pa = reinterpret_cast<const uint4*>(X + ((size_t)ra.src * LH + lh) * D + 8 * t);
  const uint4* pb = reinterpret_cast<const uint4*>(X + ((size_t)rb.src * LH + lh) * D + 8 * t);
#pragma unroll
  for (int u = 0; u < D / 32; ++u) {
    xa[u] = ra.valid() ? __ldg(pa + 4 * u) : make_uint4(0u, 0u, 0u, 0u);
    xb[u] = rb.valid() ? __ldg(pb + 4 * u) : make_uint4(0u, 0u, 0u, 0u);
  }
}

// C = X . B'^T for one Z: 3 MMAs (lo, mid, hi term of B') per (k step, rank chunk); returns the rounded coefficients of rows g
// (ca) and g+8 (cb), columns 8nt + 2t, +1, zero beyond the token's rank
template <int D, int NT>
__device__ __forceinline__ void project(const uint4* P4, const uint2* P2, int lane, const uint4 (&xa)[D / 32], const uint4 (&xb)[D / 32],
                                        const RowDst& ra, const RowDst& rb, uint32_t (&ca)[NT], uint32_t (&cb)[NT]) {
  float c[NT][4];
#pragma unroll
  for (int nt = 0; nt < NT; ++nt) c[nt][0] = c[nt][1] = c[nt][2] = c[nt][3] = 0.f;
#pragma unroll
  for (int kk = 0; kk < D / 16; ++kk) {
    const int u = kk >> 1;
    const uint32_t a0 = (kk & 1) ? xa[u].z : xa[u].x, a2 = (kk & 1) ? xa[u].w : xa[u].y;
    const uint32_t a1 = (kk & 1) ? xb[u].z : xb[u].x, a3 = (kk & 1) ? xb[u].w : xb[u].y;
#pragma unroll
    for (int nt = 0; nt < NT; ++nt) {
      const uint4 hm = P4[(kk * NT + nt) * 32 + lane];
      const uint2 lo = P2[(kk * NT + nt) * 32 + lane];
      mma16(c[nt], a0, a1, a2, a3, lo.x, lo.y);      // small terms first
      mma16(c[nt], a0, a1, a2, a3, hm.z, hm.w);
      mma16(c[nt], a0, a1, a2, a3, hm.x, hm.y);
    }
  }
#pragma unroll
  for (int nt = 0; nt < NT; ++nt) {
    ca[nt] = (8 * nt < ra.rk() && ra.valid()) ? pack_bf16x2(c[nt][0], c[nt][1]) : 0u;
    cb[nt] = (8 * nt < rb.rk() && rb.valid()) ? pack_bf16x2(c[nt][2], c[nt][3]) : 0u;
  }
}

template <int NT>
__device__ __forceinline__ void store_coef(const RowDst& rd, const uint32_t (&cw)[NT], int z, int t) {
  if (!rd.valid()) return;
  uint8_t* base = rd.blk + (z ? rd.coef_bytes() : 0);
#pragma unroll
  for (int nt = 0; nt < NT; ++nt) {
    if (8 * nt < rd.rk()) {
      if (z == 0) {
        *reinterpret_cast<uint32_t*>(base + kcoef_elem_off(rd.slot(), 8 * nt + 2 * t, rd.tb())) = cw[nt];
      } else {
        *reinterpret_cast<uint16_t*>(base + vcoef_elem_off(rd.slot(), 8 * nt + 2 * t, rd.tb())) = (uint16_t)(cw[nt] & 0xffff);
        *reinterpret_cast<uint16_t*>(base + vcoef_elem_off(rd.slot(), 8 * nt + 2 * t + 1, rd.tb())) = (uint16_t)(cw[nt] >> 16);
      }
    }
  }
}

// rec = c . B, e = x - g * rec, int4 quantiser (A14), fragment-native code / scale stores: tiles with a flagged token only.
// x is re-read from global (L1 / L2 hits) in the unpermuted channel order of the reconstruction's n dimension; the loop is
// kept rolled so the kernel stays inside the instruction cache.
template <int D, int NT>
__device__ __forceinline__ void reconstruct_quantise(const int z, const __nv_bfloat16* BTz, const int ldT, const __nv_bfloat16* gt,
                                                     const __nv_bfloat16* xa, const __nv_bfloat16* xb, const RowDst& ra, const RowDst& rb,
                                                     const uint32_t (&ca)[NT], const uint32_t (&cb)[NT], const int gr, const int t) {
#pragma unroll 1
  for (int wx = 0; wx < D / 32; ++wx) {     // K code word wx of a row = groups 2wx, 2wx+1 (registers q = 4wx .. 4wx+3)
    uint32_t kwa = 0u, kwb = 0u;
#pragma unroll
    for (int gg = 0; gg < 2; ++gg) {
      const int grp = 2 * wx + gg;
      float rec[2][4];                      // n-tiles 2grp (channels 16grp + 2t, +1) and 2grp+1 (channels 16grp + 8 + 2t, +1)
#pragma unroll
      for (int hf = 0; hf < 2; ++hf) {
        rec[hf][0] = rec[hf][1] = rec[hf][2] = rec[hf][3] = 0.f;
        const __nv_bfloat16* bt = BTz + (16 * grp + 8 * hf + gr) * ldT + 2 * t;
#pragma unroll
        for (int ks = 0; ks < (NT + 1) / 2; ++ks) {
          if (2 * ks + 1 < NT) {
            const uint32_t b0 = *reinterpret_cast<const uint32_t*>(bt + 16 * ks), b1 = *reinterpret_cast<const uint32_t*>(bt + 16 * ks + 8);
            mma16(rec[hf], ca[2 * ks], cb[2 * ks], ca[2 * ks + 1], cb[2 * ks + 1], b0, b1);
          } else if (2 * ks < NT) {        // odd number of 8-column chunks: last chunk with k = 8
            const uint32_t b0 = *reinterpret_cast<const uint32_t*>(bt + 16 * ks);
            mma8(rec[hf], ca[2 * ks], cb[2 * ks], b0);
          }
        }
      }
      const float2 g0 = bf2(__ldg(reinterpret_cast<const uint32_t*>(gt + 16 * grp))), g2 = bf2(__ldg(reinterpret_cast<const uint32_t*>(gt + 16 * grp + 8)));
#pragma unroll
      for (int row = 0; row < 2; ++row) {
        const RowDst& rd = row ? rb : ra;
        const __nv_bfloat16* xp = row ? xb : xa;
        const float2 x0 = bf2(rd.valid() ? __ldg(reinterpret_cast<const uint32_t*>(xp + 16 * grp)) : 0u);
        const float2 x2 = bf2(rd.valid() ? __ldg(reinterpret_cast<const uint32_t*>(xp + 16 * grp + 8)) : 0u);
        float e[4];
        e[0] = fmaf(-g0.x, rec[0][2 * row], x0.x); e[1] = fmaf(-g0.y, rec[0][2 * row + 1], x0.y);
        e[2] = fmaf(-g2.x, rec[1][2 * row], x2.x); e[3] = fmaf(-g2.y, rec[1][2 * row + 1], x2.y);
        float amax = fmaxf(fmaxf(fabsf(e[0]), fabsf(e[1])), fmaxf(fabsf(e[2]), fabsf(e[3])));
        amax = fmaxf(amax, __shfl_xor_sync(kFull, amax, 1));
        amax = fmaxf(amax, __shfl_xor_sync(kFull, amax, 2));
        if (rd.flagged()) {
          const __half s = quant_scale(amax);
          const float sf = __half2float(s);
          int code[4];
#pragma unroll
          for (int x = 0; x < 4; ++x) code[x] = (quant_code(e[x], sf) + 8) & 15;     // offset binary
          uint8_t* res = rd.blk + 2 * rd.coef_bytes();          // [K code | K scale | V code | V scale], sub-block of 16 slots
          const int j = rd.slot() >> 3, p = rd.slot() & 7;
          if (z == 0) {
            const uint32_t bits = ((uint32_t)code[0] << (8 * gg)) | ((uint32_t)code[1] << (16 + 8 * gg)) |
                                  ((uint32_t)code[2] << (8 * gg + 4)) | ((uint32_t)code[3] << (16 + 8 * gg + 4));
            if (row) kwb |= bits; else kwa |= bits;
            if (t == 0) *reinterpret_cast<__half*>(res + 8 * D + scale_elem_off(rd.slot(), grp, D)) = s;
          } else {
            // V codes: byte (2*hi + tile) of word (4*gch + ts)*(D/4) + 4*grp holds channels gch (low nibble) and gch + 8
            const int ts = p >> 1, hi = p & 1;
            uint8_t* cv = res + 10 * D + 4 * grp + 2 * hi + j;
            cv[(4 * (2 * t) + ts) * (D / 4)] = (uint8_t)(code[0] | (code[2] << 4));
            cv[(4 * (2 * t + 1) + ts) * (D / 4)] = (uint8_t)(code[1] | (code[3] << 4));
            if (t == 0) *reinterpret_cast<__half*>(res + 18 * D + scale_elem_off(rd.slot(), grp, D)) = s;
          }
        }
      }
    }
    if (z == 0) {
      if (ra.flagged()) *reinterpret_cast<uint32_t*>(ra.blk + 2 * ra.coef_bytes() + (ra.slot() >> 3) * 4 * D + (4 * (ra.slot() & 7) + t) * (D / 8) + 4 * wx) = kwa;
      if (rb.flagged()) *reinterpret_cast<uint32_t*>(rb.blk + 2 * rb.coef_bytes() + (rb.slot() >> 3) * 4 * D + (4 * (rb.slot() & 7) + t) * (D / 8) + 4 * wx) = kwb;
    }
  }
}

template <int D, int NT>      // NT = basis rank / 8
__global__ void __launch_bounds__(kCompressWarps * 32, 1)
compress_mma_kernel(const uint8_t* arena, const CacheGeom g, const TokDst* dst, const int n_tok, const int n_flag_tiles,
                    const __nv_bfloat16* k_new, const __nv_bfloat16* v_new, const __nv_bfloat16* BK, const __nv_bfloat16* BV,
                    const __nv_bfloat16* gK, const __nv_bfloat16* gV) {
  constexpr int NKK = D / 16, r = 8 * NT, ldT = r + 8, NFRAG = NKK * NT * 32, NTHR = kCompressWarps * 32;
  extern __shared__ __align__(16) uint8_t smem_raw[];
  uint4* P4 = reinterpret_cast<uint4*>(smem_raw);                        // [2][NFRAG]  (hi.b0, hi.b1, mid.b0, mid.b1) of B'
  uint2* P2 = reinterpret_cast<uint2*>(P4 + 2 * NFRAG);                  // [2][NFRAG]  (lo.b0, lo.b1)
  __nv_bfloat16* BT = reinterpret_cast<__nv_bfloat16*>(P2 + 2 * NFRAG);  // [2][D][ldT] transposed basis (reconstruction B operand)
  const int LH = g.L * g.H;
  const uint32_t ranks4 = (uint32_t)g.tier_rank[0] | ((uint32_t)g.tier_rank[1] << 8) | ((uint32_t)g.tier_rank[2] << 16) | ((uint32_t)g.tier_rank[3] << 24);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, gr = lane >> 2, t = lane & 3;
  const int nt_lh = (n_tok + 15) >> 4, nf = n_flag_tiles;
  const int per_lh = nf * kCostFlag + (nt_lh - nf) * kCostPlain;
  const long long total = (long long)LH * per_lh;
  int lh0, t0, lh1, t1;
  cost_to_item(total * blockIdx.x / gridDim.x, per_lh, nf, nt_lh, &lh0, &t0);
  cost_to_item(total * (blockIdx.x + 1) / gridDim.x, per_lh, nf, nt_lh, &lh1, &t1);
#pragma unroll 1
  for (int lh = lh0; lh <= lh1 && lh < LH; ++lh) {
    const int tb = lh == lh0 ? t0 : 0, te = lh == lh1 ? t1 : nt_lh;
    if (tb >= te) continue;
    const int l = lh / g.H, h = lh - l * g.H;
    __syncthreads();                                                     // the previous segment's readers are done
    // ---- stage B' = B / g (hi + mid + lo) in B-fragment order and the transposed basis --------------------------------------
#pragma unroll 1
    for (int z = 0; z < 2; ++z) {
      const __nv_bfloat16* B = (z ? BV : BK) + ((size_t)(l / g.w) * g.H + h) * (size_t)r * D;
      const __nv_bfloat16* gz = (z ? gV : gK) + (size_t)lh * D;
      for (int idx = tid; idx < NFRAG; idx += NTHR) {
        const int fl = idx & 31, fnt = (idx >> 5) % NT, fkk = (idx >> 5) / NT;
        const int fg = fl >> 2, ft = fl & 3;
        const int ch = 32 * (fkk >> 1) + 8 * ft + 4 * (fkk & 1);           // k slots 2t, 2t+1, 8+2t, 8+2t+1 <-> channels ch .. ch+3
        const uint2 bw = __ldg(reinterpret_cast<const uint2*>(B + (size_t)(8 * fnt + fg) * D + ch));
        const uint2 gw = __ldg(reinterpret_cast<const uint2*>(gz + ch));
        const float2 b01 = bf2(bw.x), b23 = bf2(bw.y), g01 = bf2(gw.x), g23 = bf2(gw.y);
        uint32_t h0, m0, l0, h1, m1, l1;
        split3(__fdiv_rn(b01.x, g01.x), __fdiv_rn(b01.y, g01.y), h0, m0, l0);
        split3(__fdiv_rn(b23.x, g23.x), __fdiv_rn(b23.y, g23.y), h1, m1, l1);
        P4[z * NFRAG + idx] = make_uint4(h0, h1, m0, m1);
        P2[z * NFRAG + idx] = make_uint2(l0, l1);
      }
      for (int idx = tid; idx < r * D / 2; idx += NTHR) {                 // pairs of channels
        const uint32_t w = __ldg(reinterpret_cast<const uint32_t*>(B) + idx);
        const int j = idx / (D / 2), i = (idx - j * (D / 2)) * 2;
        *reinterpret_cast<uint16_t*>(BT + (z * D + i) * ldT + j) = (uint16_t)(w & 0xffff);
        *reinterpret_cast<uint16_t*>(BT + (z * D + i + 1) * ldT + j) = (uint16_t)(w >> 16);
      }
    }
    __syncthreads();
    // ---- this warp's tiles of the segment: tb + warp, + 8, ... ; loads run one Z ahead of the multiplications ---------------
    int tile = tb + warp;
    if (tile >= te) continue;
    RowDst ra = row_dst(arena, ranks4, g.d, dst, 16 * tile + gr, n_tok, lh), rb = row_dst(arena, ranks4, g.d, dst, 16 * tile + gr + 8, n_tok, lh);
    uint4 xka[D / 32], xkb[D / 32], xva[D / 32], xvb[D / 32];
    load_x<D>(k_new, ra, rb, LH, lh, t, xka, xkb);
#pragma unroll 1
    while (true) {
      const bool any_flag = __any_sync(kFull, ra.flagged() || rb.flagged());
      const int next = tile + kCompressWarps;
      RowDst na = ra, nb = rb;
      if (next < te) {                       // destination table rows of the next tile: needed (src) before its K rows can be fetched
        na = row_dst(arena, ranks4, g.d, dst, 16 * next + gr, n_tok, lh);
        nb = row_dst(arena, ranks4, g.d, dst, 16 * next + gr + 8, n_tok, lh);
      }
      load_x<D>(v_new, ra, rb, LH, lh, t, xva, xvb);
      uint32_t ca[NT], cb[NT];
      project<D, NT>(P4, P2, lane, xka, xkb, ra, rb, ca, cb);
      store_coef<NT>(ra, ca, 0, t);
      store_coef<NT>(rb, cb, 0, t);
      if (any_flag)
        reconstruct_quantise<D, NT>(0, BT, ldT, gK + (size_t)lh * D + 2 * t, k_new + ((size_t)ra.src * LH + lh) * D + 2 * t,
                                    k_new + ((size_t)rb.src * LH + lh) * D + 2 * t, ra, rb, ca, cb, gr, t);
      if (next < te) load_x<D>(k_new, na, nb, LH, lh, t, xka, xkb);
      project<D, NT>(P4 + NFRAG, P2 + NFRAG, lane, xva, xvb, ra, rb, ca, cb);
      store_coef<NT>(ra, ca, 1, t);
      store_coef<NT>(rb, cb, 1, t);
      if (any_flag)
        reconstruct_quantise<D, NT>(1, BT + D * ldT, ldT, gV + (size_t)lh * D + 2 * t, v_new + ((size_t)ra.src * LH + lh) * D + 2 * t,
                                    v_new + ((size_t)rb.src * LH + lh) * D + 2 * t, ra, rb, ca, cb, gr, t);
      if (next >= te) break;
      ra = na; rb = nb; tile = next;
    }
  }
}

}  // namespace

int launch_compress_mma(const uint8_t* arena, const CacheGeom& g, const TokDst* dst, int n, int n_flagged, const __nv_bfloat16* k_new,
                        const __nv_bfloat16* v_new, const __nv_bfloat16* BK, const __nv_bfloat16* BV, const __nv_bfloat16* gK,
                        const __nv_bfloat16* gV, int n_sms, cudaStream_t s) {
  if (n <= 0) return 0;
  const int nfrag = (g.d / 16) * (g.r / 8) * 32;
  const size_t smem = (size_t)2 * nfrag * 24 + (size_t)2 * g.d * (g.r + 8) * 2;
  const long long tiles = (long long)g.L * g.H * ((n + 15) / 16);
  const int per_sm = 1;
  const int grid = (int)std::max<long long>(1, std::min<long long>((long long)per_sm * n_sms, tiles));
  const int nft = (n_flagged + 15) / 16;
  bool ok = true;
#define DWKV_COMPRESS_CASE(DD, NN)                                                                                              \
  case NN:                                                                                                                      \
    cudaFuncSetAttribute(compress_mma_kernel<DD, NN>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);                  \
    compress_mma_kernel<DD, NN><<<grid, kCompressWarps * 32, smem, s>>>(arena, g, dst, n, nft, k_new, v_new, BK, BV, gK, gV);    \
    break;
  if (g.d == 128) {
    switch (g.r / 8) { DWKV_COMPRESS_CASE(128, 1) DWKV_COMPRESS_CASE(128, 2) DWKV_COMPRESS_CASE(128, 3) DWKV_COMPRESS_CASE(128, 4)
                       DWKV_COMPRESS_CASE(128, 6) DWKV_COMPRESS_CASE(128, 8) default: ok = false; }
  } else {
    switch (g.r / 8) { DWKV_COMPRESS_CASE(64, 1) DWKV_COMPRESS_CASE(64, 2) DWKV_COMPRESS_CASE(64, 3) DWKV_COMPRESS_CASE(64, 4)
                       DWKV_COMPRESS_CASE(64, 6) DWKV_COMPRESS_CASE(64, 8) default: ok = false; }
  }
#undef DWKV_COMPRESS_CASE
  if (!ok) return 0;
  return 1;
}

}  // namespace dwkv
