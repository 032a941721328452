// dwkv_compress.cu -- a4: append / compress on the tensor cores (PAPER.md:56
// "projecting the original cache vector onto the current basis"; readings A13, A14).
//
// For a tile of 16 new tokens and one (layer, kv head), per Z in {K, V}:
//   C   = (X / g) . B^T        [16 x r]   x/g as x * rn(1/g) in fp32, split hi + mid + lo bf16 (24 bits), fp32 accumulate
//   c   = bf16(C), columns >= r_t of a token dropped (leading-r_t coefficients of its tier)
//   rec = c . B                [16 x d]   exact bf16 products, fp32 accumulate     (only if a token of the tile is flagged)
//   e   = x - g * rec  ->  int4 / group 16 / fp16 scale  (quantiser A14, fp32 IEEE, no reciprocal)
// One warp per tile; a CTA of 4 warps shares the basis of its (layer, head) in shared memory (row-major for the projection,
// transposed for the reconstruction, both padded to be bank-conflict free as MMA B fragments). Results go straight to their
// fragment-native positions in the class pages (dwkv_layout.cuh): every 32-bit coefficient word, 16-byte K-code row, V-code
// byte and scale is owned by exactly one (token, lane), so no atomics are needed (pages are zeroed when allocated).
#include <algorithm>

#include "dwkv_internal.h"
#include "dwkv_mma.cuh"

namespace dwkv {
namespace {
using namespace dwkv::dev;

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

struct RowDst {          // destination of one token row of the tile for this (layer, head)
  uint8_t* blk;          // sub-block base
  int slot;              // slot inside the sub-block
  int rk;                // rank of the token's tier
  int tb;                // tiles per sub-block (2 flagged / 4 unflagged)
  int coef_bytes;        // bytes of [K coef] (= [V coef]) of the sub-block
  bool valid, flagged;
  int src;               // row of the token in k_new / v_new
};

__device__ __forceinline__ RowDst row_dst(const uint8_t* arena, const CacheGeom& g, const TokDst* dst, int tok, int n_tok, int lh) {
  RowDst r;
  r.valid = tok < n_tok;
  const TokDst td = dst[r.valid ? tok : 0];
  const ClassLayout cl = make_class_layout(g.tier_rank[td.cls >> 1], td.cls & 1, g.d);
  r.rk = g.tier_rank[td.cls >> 1];
  r.tb = cl.tb;
  r.coef_bytes = cl.coef_bytes;
  r.flagged = r.valid && td.ridx >= 0;
  r.src = td.src;
  r.blk = const_cast<uint8_t*>(arena) + td.page_off + (size_t)lh * kPageLhBytes + (size_t)td.blk * cl.block_bytes + sub_off(cl, td.slot);
  r.slot = sub_slot(cl, td.slot);
  return r;
}

template <int D, int NT>      // NT = basis rank / 8
__global__ void __launch_bounds__(128) compress_mma_kernel(const uint8_t* arena, const CacheGeom g, const TokDst* dst, const int n_tok,
                                                           const __nv_bfloat16* k_new, const __nv_bfloat16* v_new,
                                                           const __nv_bfloat16* BK, const __nv_bfloat16* BV,
                                                           const __nv_bfloat16* gK, const __nv_bfloat16* gV) {
  constexpr int NKK = D / 16, NG = D / 16;
  extern __shared__ __align__(16) uint8_t smem_raw[];
  constexpr int r = 8 * NT;
  constexpr int ldB = D + 8, ldT = r + 8;                                   // padded leading dimensions (elements)
  __nv_bfloat16* Bs = reinterpret_cast<__nv_bfloat16*>(smem_raw);       // [2][r][ldB]   basis rows        (projection B operand)
  __nv_bfloat16* BT = Bs + 2 * r * ldB;                                 // [2][D][ldT]   transposed basis  (reconstruction B operand)
  float* ig = reinterpret_cast<float*>(BT + 2 * D * ldT);                // [2][D]        1 / gate (x / g as x * (1/g): one division per channel and CTA)
  const int lh = blockIdx.y, l = lh / g.H, h = lh % g.H, LH = g.L * g.H;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, gr = lane >> 2, t = lane & 3;
  for (int z = 0; z < 2; ++z) {
    const __nv_bfloat16* B = (z ? BV : BK) + ((size_t)(l / g.w) * g.H + h) * (size_t)r * D;
    for (int idx0 = tid; idx0 < r * D / 2; idx0 += 128 * 8) {           // pairs of channels, 8 loads in flight per thread
      uint32_t w[8];
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        const int idx = idx0 + 128 * u;
        w[u] = idx < r * D / 2 ? __ldg(reinterpret_cast<const uint32_t*>(B) + idx) : 0u;
      }
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        const int idx = idx0 + 128 * u;
        if (idx < r * D / 2) {
          const int j = idx / (D / 2), i = (idx - j * (D / 2)) * 2;
          *reinterpret_cast<uint32_t*>(Bs + (z * r + j) * ldB + i) = w[u];
          *reinterpret_cast<uint16_t*>(BT + (z * D + i) * ldT + j) = (uint16_t)(w[u] & 0xffff);
          *reinterpret_cast<uint16_t*>(BT + (z * D + i + 1) * ldT + j) = (uint16_t)(w[u] >> 16);
        }
      }
    }
  }
  for (int i = tid; i < 2 * D; i += 128) ig[i] = __frcp_rn(__bfloat162float(((i < D) ? gK : gV)[(size_t)lh * D + (i % D)]));
  __syncthreads();
#pragma unroll 1
  for (int tok0 = (blockIdx.x * 4 + warp) * 16; tok0 < n_tok; tok0 += gridDim.x * 64) {     // this warp's tiles
  const RowDst ra = row_dst(arena, g, dst, tok0 + gr, n_tok, lh), rb = row_dst(arena, g, dst, tok0 + gr + 8, n_tok, lh);
  const bool any_flag = __any_sync(kFull, ra.flagged || rb.flagged);
#pragma unroll 1
  for (int z = 0; z < 2; ++z) {
    const __nv_bfloat16* X = z ? v_new : k_new;
    const __nv_bfloat16* xa = X + ((size_t)(ra.valid ? ra.src : 0) * LH + lh) * D + 2 * t;
    const __nv_bfloat16* xb = X + ((size_t)(rb.valid ? rb.src : 0) * LH + lh) * D + 2 * t;
    const __nv_bfloat16* gt = (z ? gV : gK) + (size_t)lh * D + 2 * t;
    const float* igz = ig + z * D + 2 * t;
    const __nv_bfloat16* Bz = Bs + z * r * ldB;
    const __nv_bfloat16* BTz = BT + z * D * ldT;
    // ---- projection C = (X / g) . B^T; loops are kept rolled: the kernel must stay inside the instruction cache --------------
    float c[NT][4];
#pragma unroll
    for (int nt = 0; nt < NT; ++nt) c[nt][0] = c[nt][1] = c[nt][2] = c[nt][3] = 0.f;
#pragma unroll 2
    for (int kk = 0; kk < NKK; ++kk) {
      // A-fragment order: [0] row g ch 16kk+2t, [1] row g+8, [2] row g ch 16kk+8+2t, [3] row g+8
      const uint32_t w0 = ra.valid ? __ldg(reinterpret_cast<const uint32_t*>(xa + 16 * kk)) : 0u;
      const uint32_t w1 = rb.valid ? __ldg(reinterpret_cast<const uint32_t*>(xb + 16 * kk)) : 0u;
      const uint32_t w2 = ra.valid ? __ldg(reinterpret_cast<const uint32_t*>(xa + 16 * kk + 8)) : 0u;
      const uint32_t w3 = rb.valid ? __ldg(reinterpret_cast<const uint32_t*>(xb + 16 * kk + 8)) : 0u;
      const float2 i0 = *reinterpret_cast<const float2*>(igz + 16 * kk), i2 = *reinterpret_cast<const float2*>(igz + 16 * kk + 8);
      const float2 x0 = bf2(w0), x1 = bf2(w1), x2 = bf2(w2), x3 = bf2(w3);
      uint32_t ah[4], am[4], al[4];
      split3(x0.x * i0.x, x0.y * i0.y, ah[0], am[0], al[0]);
      split3(x1.x * i0.x, x1.y * i0.y, ah[1], am[1], al[1]);
      split3(x2.x * i2.x, x2.y * i2.y, ah[2], am[2], al[2]);
      split3(x3.x * i2.x, x3.y * i2.y, ah[3], am[3], al[3]);
#pragma unroll
      for (int nt = 0; nt < NT; ++nt) {
        {
          const __nv_bfloat16* br = Bz + (8 * nt + gr) * ldB + 16 * kk + 2 * t;
          const uint32_t b0 = *reinterpret_cast<const uint32_t*>(br), b1 = *reinterpret_cast<const uint32_t*>(br + 8);
          mma16(c[nt], al[0], al[1], al[2], al[3], b0, b1);      // small terms first
          mma16(c[nt], am[0], am[1], am[2], am[3], b0, b1);
          mma16(c[nt], ah[0], ah[1], ah[2], ah[3], b0, b1);
        }
      }
    }
    // ---- round, drop columns beyond the token's rank, store coefficients ------------------------------------------------------
    uint32_t ca[NT], cb[NT];          // bf16x2 (cols 8nt+2t, +1) of rows g and g+8
#pragma unroll
    for (int nt = 0; nt < NT; ++nt) {
      ca[nt] = (8 * nt < ra.rk && ra.valid) ? pack_bf16x2(c[nt][0], c[nt][1]) : 0u;
      cb[nt] = (8 * nt < rb.rk && rb.valid) ? pack_bf16x2(c[nt][2], c[nt][3]) : 0u;
    }
#pragma unroll
    for (int row = 0; row < 2; ++row) {
      const RowDst& rd = row ? rb : ra;
      if (rd.valid) {
        uint8_t* base = rd.blk + (z ? rd.coef_bytes : 0);
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) {
          if (8 * nt < rd.rk) {
            const uint32_t w = row ? cb[nt] : ca[nt];
            if (z == 0) {
              *reinterpret_cast<uint32_t*>(base + kcoef_elem_off(rd.slot, 8 * nt + 2 * t, rd.tb)) = w;
            } else {
              *reinterpret_cast<uint16_t*>(base + vcoef_elem_off(rd.slot, 8 * nt + 2 * t, rd.tb)) = (uint16_t)(w & 0xffff);
              *reinterpret_cast<uint16_t*>(base + vcoef_elem_off(rd.slot, 8 * nt + 2 * t + 1, rd.tb)) = (uint16_t)(w >> 16);
            }
          }
        }
      }
    }
    if (!any_flag) continue;
    // ---- reconstruction rec = c . B, residual e = x - g * rec, int4 quantiser, stores ------------------------------------------
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
          const float2 x0 = bf2(rd.valid ? __ldg(reinterpret_cast<const uint32_t*>(xp + 16 * grp)) : 0u);
          const float2 x2 = bf2(rd.valid ? __ldg(reinterpret_cast<const uint32_t*>(xp + 16 * grp + 8)) : 0u);
          float e[4];
          e[0] = fmaf(-g0.x, rec[0][2 * row], x0.x); e[1] = fmaf(-g0.y, rec[0][2 * row + 1], x0.y);
          e[2] = fmaf(-g2.x, rec[1][2 * row], x2.x); e[3] = fmaf(-g2.y, rec[1][2 * row + 1], x2.y);
          float amax = fmaxf(fmaxf(fabsf(e[0]), fabsf(e[1])), fmaxf(fabsf(e[2]), fabsf(e[3])));
          amax = fmaxf(amax, __shfl_xor_sync(kFull, amax, 1));
          amax = fmaxf(amax, __shfl_xor_sync(kFull, amax, 2));
          if (rd.flagged) {
            const __half s = quant_scale(amax);
            const float sf = __half2float(s);
            int code[4];
#pragma unroll
            for (int x = 0; x < 4; ++x) code[x] = (quant_code(e[x], sf) + 8) & 15;     // offset binary
            uint8_t* res = rd.blk + 2 * rd.coef_bytes;          // [K code | K scale | V code | V scale], sub-block of 16 slots
            const int j = rd.slot >> 3, p = rd.slot & 7;
            if (z == 0) {
              const uint32_t bits = ((uint32_t)code[0] << (8 * gg)) | ((uint32_t)code[1] << (16 + 8 * gg)) |
                                    ((uint32_t)code[2] << (8 * gg + 4)) | ((uint32_t)code[3] << (16 + 8 * gg + 4));
              if (row) kwb |= bits; else kwa |= bits;
              if (t == 0) *reinterpret_cast<__half*>(res + 8 * D + scale_elem_off(rd.slot, grp, D)) = s;
            } else {
              // V codes: byte (2*hi + tile) of word (4*gch + ts)*(D/4) + 4*grp holds channels gch (low nibble) and gch + 8
              const int ts = p >> 1, hi = p & 1;
              uint8_t* cv = res + 10 * D + 4 * grp + 2 * hi + j;
              cv[(4 * (2 * t) + ts) * (D / 4)] = (uint8_t)(code[0] | (code[2] << 4));
              cv[(4 * (2 * t + 1) + ts) * (D / 4)] = (uint8_t)(code[1] | (code[3] << 4));
              if (t == 0) *reinterpret_cast<__half*>(res + 18 * D + scale_elem_off(rd.slot, grp, D)) = s;
            }
          }
        }
      }
      if (z == 0) {
        if (ra.flagged) *reinterpret_cast<uint32_t*>(ra.blk + 2 * ra.coef_bytes + (ra.slot >> 3) * 4 * D + (4 * (ra.slot & 7) + t) * (D / 8) + 4 * wx) = kwa;
        if (rb.flagged) *reinterpret_cast<uint32_t*>(rb.blk + 2 * rb.coef_bytes + (rb.slot >> 3) * 4 * D + (4 * (rb.slot & 7) + t) * (D / 8) + 4 * wx) = kwb;
      }
    }
  }
  }   // tiles
}

}  // namespace

int launch_compress_mma(const uint8_t* arena, const CacheGeom& g, const TokDst* dst, int n, const __nv_bfloat16* k_new,
                        const __nv_bfloat16* v_new, const __nv_bfloat16* BK, const __nv_bfloat16* BV, const __nv_bfloat16* gK,
                        const __nv_bfloat16* gV, cudaStream_t s) {
  if (n <= 0) return 0;
  const size_t smem = (size_t)2 * g.r * (g.d + 8) * 2 + (size_t)2 * g.d * (g.r + 8) * 2 + (size_t)2 * g.d * 4;
  // a CTA refills the basis of its (layer, head) once and loops over token tiles: a few CTAs per (layer, head)
  const int gx = std::max(1, std::min((n + 63) / 64, (4 * 148 + g.L * g.H - 1) / (g.L * g.H)));
  dim3 grid(gx, g.L * g.H);
  bool ok = true;
#define DWKV_COMPRESS_CASE(DD, NN)                                                                                              \
  case NN:                                                                                                                      \
    cudaFuncSetAttribute(compress_mma_kernel<DD, NN>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);                  \
    compress_mma_kernel<DD, NN><<<grid, 128, smem, s>>>(arena, g, dst, n, k_new, v_new, BK, BV, gK, gV);                        \
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
