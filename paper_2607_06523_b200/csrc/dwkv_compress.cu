// dwkv_compress.cu -- a4: append / compress on the tensor cores (PAPER.md:56
// "projecting the original cache vector onto the current basis"; readings A13, A14).
//
// For a tile of 16 new tokens and one (layer, kv head), per Z in {K, V}:
//   C   = X . B'^T             [16 x r]   B'[j][i] = B[j][i] / g[i] (fp32 IEEE division), split hi + mid + lo bf16 (24 bits)
//                                         once per (layer, head) and CTA; x is bf16 already, so the A operand needs no work
//   c   = bf16(C), columns >= r_t of a token dropped (leading-r_t coefficients of its tier)
//   rec = c . B                [16 x d]   exact bf16 products, fp32 accumulate     (only if a token of the tile is flagged)
//   e   = x - g * rec  ->  int4 / group 16 / fp16 scale  (quantiser A14, fp32 IEEE, no reciprocal)
// Persistent grid: the (layer-head, tile) items are cut into equal-cost contiguous ranges, one per CTA (the host sorts the call's tokens
// flagged-first and by descending rank, so a tile's tokens share a rank; a tile costs compress_tile_cost(flagged, rank / 8) and
// only the rank chunks its tokens keep are multiplied); a CTA stages B' of its current (layer, head) in shared memory in the register
// order of the MMA B fragments (one 16-byte + one 8-byte ld.shared per MMA triple) and its 8 or 12 warps take tiles round-robin.
// Every warp streams its token rows through a private shared-memory ring filled by cp.async 2-4 stages ahead (a stage = the 16
// rows of one tile and one Z) and reads the A fragments back with ldmatrix. Results go straight
// to their fragment-native positions in the class pages (dwkv_layout.cuh): every 32-bit coefficient word, 16-byte K-code row,
// V-code byte and scale is owned by exactly one (token, lane), so no atomics are needed (pages are zeroed when allocated).
#include <algorithm>

#include <cuda.h>

#include "dwkv_internal.h"
#include "dwkv_mma.cuh"

namespace dwkv {
namespace {
using namespace dwkv::dev;

constexpr int kCompressMaxWarps = 16;

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
  int meta;              // slot inside the sub-block | rank of the token's tier << 8 | valid << 16 | flagged << 17 | 8-bit planes << 18
  int src;               // row of the token in k_new / v_new
  __device__ __forceinline__ int slot() const { return meta & 0xff; }
  __device__ __forceinline__ int rk() const { return (meta >> 8) & 0xff; }
  __device__ __forceinline__ bool valid() const { return (meta >> 16) & 1; }
  __device__ __forceinline__ bool flagged() const { return (meta >> 17) & 1; }
  __device__ __forceinline__ int tb() const { return flagged() ? 2 : 4; }          // tiles per sub-block
  __device__ __forceinline__ bool i8() const { return (meta >> 18) & 1; }
  // bytes of [K coef] (= [V coef]); 8-bit planes: one byte per coefficient + 8 * tb exponent bytes per 32-column block
  __device__ __forceinline__ int coef_bytes() const { return i8() ? rk() * 8 * tb() + ((rk() + 31) >> 5) * 8 * tb() : rk() * 16 * tb(); }
};

// the ClassLayout arithmetic of dwkv_layout.cuh with shifts only (tb is 2 or 4); tier ranks come as 4 bytes of one word
__device__ __forceinline__ RowDst row_dst_from(const uint8_t* arena, const uint32_t ranks4, const int d, const TokDst& td, const bool valid, int lh,
                                                const bool i8 = false) {
  RowDst r;
  const int resid = td.cls & 1;
  const int rk = (ranks4 >> (8 * (td.cls >> 1))) & 0xff;
  const int tb = resid ? 2 : 4;
  const int coef_bytes = i8 ? rk * 8 * tb + ((rk + 31) >> 5) * 8 * tb : rk * 16 * tb;
  const int sub_bytes = 2 * coef_bytes + (resid ? 2 * 5 * tb * d : 0);
  const int block_bytes = resid ? 2 * sub_bytes : sub_bytes;
  r.src = valid ? td.src : 0;
  r.blk = const_cast<uint8_t*>(arena) + td.page_off + (size_t)lh * kPageLhBytes + (size_t)td.blk * block_bytes +
          ((resid && td.slot >= 16) ? sub_bytes : 0);
  r.meta = (resid ? (td.slot & 15) : td.slot) | (rk << 8) | ((int)valid << 16) | ((int)(valid && resid) << 17) | ((int)i8 << 18);
  return r;
}
__device__ __forceinline__ RowDst row_dst(const uint8_t* arena, const uint32_t ranks4, const int d, const TokDst* dst, int tok, int n_tok, int lh,
                                          const bool i8 = false) {
  const bool valid = tok < n_tok;
  const TokDst td = dst[valid ? tok : 0];
  return row_dst_from(arena, ranks4, d, td, valid, lh, i8);
}

// item position in cost space -> (layer-head, tile). Per layer-head the tiles come in runs of equal cost (CompressRuns).
__device__ __forceinline__ void cost_to_item(long long pos, const CompressRuns& R, int* lh, int* tile) {
  *lh = (int)(pos / R.per_lh);
  int rem = (int)(pos - (long long)*lh * R.per_lh), t0 = 0;
#pragma unroll 1
  for (int i = 0; i < R.n; ++i) {
    const int c = R.count[i] * R.cost[i];
    if (rem < c) { *tile = t0 + rem / R.cost[i]; return; }
    rem -= c; t0 += R.count[i];
  }
  *tile = t0;
}

// ---- per-warp shared-memory ring of token-row stages -------------------------------------------------------------------------
// A stage holds the 16 token rows of one tile for one Z, row-major with a row pitch of 2 * D + 16 bytes (ldmatrix and 4-byte
// reads of 8 consecutive rows are then bank-conflict free). Lane (g, t) copies channels 32u + 8t .. +7 of rows g and g + 8 with
// 16-byte cp.async (zero-filled for rows beyond n_tok); one ldmatrix.x4 per k step returns the A fragment of the projection as
// an aligned register quad. A stage is complete for the warp after cp.async.wait_group + __syncwarp.
__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src, int src_bytes) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait(int pending) {     // pending = stages - 1 (2..4 stages)
  if (pending >= 3) asm volatile("cp.async.wait_group 3;" ::: "memory");
  else if (pending == 2) asm volatile("cp.async.wait_group 2;" ::: "memory");
  else asm volatile("cp.async.wait_group 1;" ::: "memory");
}
__device__ __forceinline__ uint32_t lds32(uint32_t a) {
  uint32_t r;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(r) : "r"(a));
  return r;
}

__device__ __forceinline__ void ldmatrix_x4(uint32_t a, uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];" : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(a));
}

template <int D>
__device__ __forceinline__ void issue_rows(uint32_t stage, const __nv_bfloat16* X, int2 src, int LH, int lh, int lane) {
  constexpr int PITCH = 2 * D + 16;
  const int g = lane >> 2, t = lane & 3;
  const char* pa = reinterpret_cast<const char*>(X + ((size_t)max(src.x, 0) * LH + lh) * D + 8 * t);
  const char* pb = reinterpret_cast<const char*>(X + ((size_t)max(src.y, 0) * LH + lh) * D + 8 * t);
  const int sa = src.x >= 0 ? 16 : 0, sb = src.y >= 0 ? 16 : 0;
  const uint32_t da = stage + g * PITCH + 16 * t, db = da + 8 * PITCH;
#pragma unroll
  for (int u = 0; u < D / 32; ++u) {
    cp_async16(da + 64 * u, pa + 64 * u, sa);
    cp_async16(db + 64 * u, pb + 64 * u, sb);
  }
}

// bf16 pair (channels ch, ch+1; ch even) of row `row` of a stage
template <int D>
__device__ __forceinline__ uint32_t stage_x(uint32_t stage, int row, int ch) { return lds32(stage + row * (2 * D + 16) + ch * 2); }

// C = X . B'^T for one Z: 3 MMAs (lo, mid, hi term of B') per (k step, rank chunk); returns the rounded coefficients of rows g (ca) and g+8 (cb), columns 8nt + 2t, +1, zero beyond the rank
// 8-bit planes (I8; reading A27): the fp32 coefficients of a row are quantised per 32-column block (exponent from the
// block's amax over the row's leading r_t columns: the quad's four lanes hold the row), ca / cb then carry the DEQUANTISED values
// code * 2^e (exactly bf16) so that the residual absorbs the quantisation error, qa / qb the stored bytes (code + 128) of the two
// columns, xa / xb the exponent bytes (e + 127) of the row's blocks.
template <int D, int NT, int NTM, bool I8>      // NTM = rank chunks any token of the tile keeps: only those are multiplied
__device__ __forceinline__ void project_n(const uint4* P4, const uint2* P2, int lane, uint32_t stage, const RowDst& ra, const RowDst& rb,
                                          uint32_t (&ca)[NT], uint32_t (&cb)[NT], uint32_t (&qa)[NT], uint32_t (&qb)[NT], uint32_t& xa, uint32_t& xb) {
  // few chunks: one accumulator chain per term of B' (lo, mid, hi) so that the MMAs of a k step are independent
  constexpr int NA = NTM <= 2 ? 3 : 1;
  float c[NA][NTM][4];
#pragma unroll
  for (int a = 0; a < NA; ++a)
#pragma unroll
    for (int nt = 0; nt < NTM; ++nt) c[a][nt][0] = c[a][nt][1] = c[a][nt][2] = c[a][nt][3] = 0.f;
  // ldmatrix: lanes 8i .. 8i+7 address the rows of matrix i = (rows 0-7 | 8-15) x (channels +0 | +8) of the k step
  const uint32_t am = stage + ((lane & 7) + 8 * ((lane >> 3) & 1)) * (2 * D + 16) + 16 * (lane >> 4);
#pragma unroll
  for (int kk = 0; kk < D / 16; ++kk) {
    uint32_t a0, a1, a2, a3;
    ldmatrix_x4(am + 32 * kk, a0, a1, a2, a3);
#pragma unroll
    for (int nt = 0; nt < NTM; ++nt) {
      const uint4 hm = P4[(kk * NT + nt) * 32 + lane];
      const uint2 lo = P2[(kk * NT + nt) * 32 + lane];
      mma16(c[0][nt], a0, a1, a2, a3, lo.x, lo.y);      // small terms first
      mma16(c[NA == 3 ? 1 : 0][nt], a0, a1, a2, a3, hm.z, hm.w);
      mma16(c[NA == 3 ? 2 : 0][nt], a0, a1, a2, a3, hm.x, hm.y);
    }
  }
  if constexpr (I8) {
    constexpr int NB = (NT + 3) / 4;             // 32-column blocks of the basis rank
    float v[NTM][4];
    float ama[NB], amb[NB];
#pragma unroll
    for (int b = 0; b < NB; ++b) ama[b] = amb[b] = 0.f;
#pragma unroll
    for (int nt = 0; nt < NTM; ++nt) {
#pragma unroll
      for (int x = 0; x < 4; ++x) v[nt][x] = NA == 3 ? (c[0][nt][x] + c[1][nt][x]) + c[NA - 1][nt][x] : c[0][nt][x];
      if (8 * nt < ra.rk()) ama[nt >> 2] = fmaxf(ama[nt >> 2], fmaxf(fabsf(v[nt][0]), fabsf(v[nt][1])));
      if (8 * nt < rb.rk()) amb[nt >> 2] = fmaxf(amb[nt >> 2], fmaxf(fabsf(v[nt][2]), fabsf(v[nt][3])));
    }
    int ea[NB], eb[NB];
    xa = xb = 0u;
#pragma unroll
    for (int b = 0; b < NB; ++b) {
      ama[b] = fmaxf(ama[b], __shfl_xor_sync(kFull, ama[b], 1)); ama[b] = fmaxf(ama[b], __shfl_xor_sync(kFull, ama[b], 2));
      amb[b] = fmaxf(amb[b], __shfl_xor_sync(kFull, amb[b], 1)); amb[b] = fmaxf(amb[b], __shfl_xor_sync(kFull, amb[b], 2));
      ea[b] = coef8_exponent(ama[b]); eb[b] = coef8_exponent(amb[b]);
      xa |= (uint32_t)(ea[b] + 127) << (8 * b); xb |= (uint32_t)(eb[b] + 127) << (8 * b);
    }
#pragma unroll
    for (int nt = 0; nt < NT; ++nt) {
      ca[nt] = cb[nt] = 0u; qa[nt] = qb[nt] = 0u;
      if (nt < NTM) {
        if (8 * nt < ra.rk() && ra.valid()) {
          const int e = ea[nt >> 2], k0 = coef8_code(v[nt][0], e), k1 = coef8_code(v[nt][1], e);
          const float sc = __uint_as_float((uint32_t)(e + 127) << 23);
          ca[nt] = pack_bf16x2((float)k0 * sc, (float)k1 * sc);
          qa[nt] = (uint32_t)(k0 + 128) | ((uint32_t)(k1 + 128) << 8);
        }
        if (8 * nt < rb.rk() && rb.valid()) {
          const int e = eb[nt >> 2], k0 = coef8_code(v[nt][2], e), k1 = coef8_code(v[nt][3], e);
          const float sc = __uint_as_float((uint32_t)(e + 127) << 23);
          cb[nt] = pack_bf16x2((float)k0 * sc, (float)k1 * sc);
          qb[nt] = (uint32_t)(k0 + 128) | ((uint32_t)(k1 + 128) << 8);
        }
      }
    }
  } else {
#pragma unroll
  for (int nt = 0; nt < NT; ++nt) {
    ca[nt] = cb[nt] = 0u;
    if (nt < NTM) {
      float v[4];
#pragma unroll
      for (int x = 0; x < 4; ++x) v[x] = NA == 3 ? (c[0][nt][x] + c[1][nt][x]) + c[NA - 1][nt][x] : c[0][nt][x];
      if (8 * nt < ra.rk() && ra.valid()) ca[nt] = pack_bf16x2(v[0], v[1]);
      if (8 * nt < rb.rk() && rb.valid()) cb[nt] = pack_bf16x2(v[2], v[3]);
    }
  }
  }
}

template <int D, int NT, bool I8>
__device__ __forceinline__ void project(const uint4* P4, const uint2* P2, int lane, uint32_t stage, const RowDst& ra, const RowDst& rb,
                                        const int ntmax /* warp-uniform */, uint32_t (&ca)[NT], uint32_t (&cb)[NT], uint32_t (&qa)[NT],
                                        uint32_t (&qb)[NT], uint32_t& xa, uint32_t& xb) {
  if (ntmax <= 1) project_n<D, NT, 1, I8>(P4, P2, lane, stage, ra, rb, ca, cb, qa, qb, xa, xb);
  else if (NT >= 2 && ntmax == 2) project_n<D, NT, (NT >= 2 ? 2 : NT), I8>(P4, P2, lane, stage, ra, rb, ca, cb, qa, qb, xa, xb);
  else if (NT >= 3 && ntmax == 3) project_n<D, NT, (NT >= 3 ? 3 : NT), I8>(P4, P2, lane, stage, ra, rb, ca, cb, qa, qb, xa, xb);
  else project_n<D, NT, NT, I8>(P4, P2, lane, stage, ra, rb, ca, cb, qa, qb, xa, xb);
}

// 8-bit planes: the row's code bytes (two columns per chunk and lane) and, from lane t = 0, the exponent bytes of its blocks
template <int NT>
__device__ __forceinline__ void store_coef8(const RowDst& rd, const uint32_t (&q)[NT], const uint32_t xexp, int z, int t) {
  if (!rd.valid()) return;
  uint8_t* base = rd.blk + (z ? rd.coef_bytes() : 0);
#pragma unroll
  for (int nt = 0; nt < NT; ++nt) {
    if (8 * nt < rd.rk()) {
      if (z == 0) {
        *reinterpret_cast<uint16_t*>(base + kcoef8_elem_off(rd.slot(), 8 * nt + 2 * t, rd.tb())) = (uint16_t)q[nt];
      } else {
        base[vcoef8_elem_off(rd.slot(), 8 * nt + 2 * t, rd.tb())] = (uint8_t)(q[nt] & 0xff);
        base[vcoef8_elem_off(rd.slot(), 8 * nt + 2 * t + 1, rd.tb())] = (uint8_t)(q[nt] >> 8);
      }
    }
  }
  if (t == 0) {
#pragma unroll
    for (int b = 0; b < (NT + 3) / 4; ++b)
      if (32 * b < rd.rk()) base[coef8_exp_off(rd.slot(), rd.rk() >> 3, rd.tb(), b)] = (uint8_t)(xexp >> (8 * b));
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
// x is read from the shared-memory stage in the unpermuted channel order of the reconstruction's n dimension; the loop is kept
// rolled so the kernel stays inside the instruction cache.
template <int D, int NT>
__device__ __forceinline__ void reconstruct_quantise(const int z, const __nv_bfloat16* BTz, const int ldT, const __nv_bfloat16* gt,
                                                     const uint32_t stage, const RowDst& ra, const RowDst& rb,
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
        const float2 x0 = bf2(stage_x<D>(stage, gr + 8 * row, 16 * grp + 2 * t));          // rows beyond n_tok were zero-filled
        const float2 x2 = bf2(stage_x<D>(stage, gr + 8 * row, 16 * grp + 8 + 2 * t));
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

template <int D, int NT, bool I8>      // NT = basis rank / 8; I8 = 8-bit coefficient planes (option "coef_int8")
__global__ void __launch_bounds__(kCompressMaxWarps * 32, 1)
compress_mma_kernel(const uint8_t* arena, const CacheGeom g, const TokDst* dst, const int n_tok, const CompressRuns runs, const int n_stages,
                    const __nv_bfloat16* k_new, const __nv_bfloat16* v_new, const __nv_bfloat16* BK, const __nv_bfloat16* BV,
                    const __nv_bfloat16* gK, const __nv_bfloat16* gV) {
  constexpr int NKK = D / 16, r = 8 * NT, ldT = r + 8, NFRAG = NKK * NT * 32, STAGE = 16 * (2 * D + 16);
  extern __shared__ __align__(16) uint8_t smem_raw[];
  uint4* P4 = reinterpret_cast<uint4*>(smem_raw);                        // [2][NFRAG]  (hi.b0, hi.b1, mid.b0, mid.b1) of B'
  uint2* P2 = reinterpret_cast<uint2*>(P4 + 2 * NFRAG);                  // [2][NFRAG]  (lo.b0, lo.b1)
  __nv_bfloat16* BT = reinterpret_cast<__nv_bfloat16*>(P2 + 2 * NFRAG);  // [2][D][ldT] transposed basis (reconstruction B operand)
  const int LH = g.L * g.H;
  const uint32_t ranks4 = (uint32_t)g.tier_rank[0] | ((uint32_t)g.tier_rank[1] << 8) | ((uint32_t)g.tier_rank[2] << 16) | ((uint32_t)g.tier_rank[3] << 24);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, gr = lane >> 2, t = lane & 3;
  const int NTHR = blockDim.x, W = NTHR >> 5;
  const uint32_t ring = (uint32_t)__cvta_generic_to_shared(BT + 2 * D * ldT) + (uint32_t)(warp * n_stages) * STAGE;   // this warp's stages
  const int nt_lh = (n_tok + 15) >> 4;
  const long long total = (long long)LH * runs.per_lh;
  int lh0, t0, lh1, t1;
  cost_to_item(total * blockIdx.x / gridDim.x, runs, &lh0, &t0);
  cost_to_item(total * (blockIdx.x + 1) / gridDim.x, runs, &lh1, &t1);
#pragma unroll 1
  for (int lh = lh0; lh <= lh1 && lh < LH; ++lh) {
    const int tb = lh == lh0 ? t0 : 0, te = lh == lh1 ? t1 : nt_lh;
    if (tb >= te) continue;
    const int l = lh / g.H, h = lh - l * g.H;
    // ---- this warp's tiles of the segment: tb + warp, + W, ...; their row copies start before the basis is staged ----------
    const int n = (te - tb - warp + W - 1) / W;                          // tiles of this warp (may be <= 0)
    const int nst = 2 * n;                                               // stages: (tile 0, K), (tile 0, V), (tile 1, K), ...
    int issued = 0, slot_i = 0;
    int2 src_cur = make_int2(-1, -1), src_nxt = make_int2(-1, -1);       // source rows (-1: beyond n_tok) of the tile being issued / the next
    auto fetch_src = [&](int i) {
      const int tok = 16 * (tb + warp + W * i) + gr;
      return make_int2(tok < n_tok ? __ldg(&dst[tok].src) : -1, tok + 8 < n_tok ? __ldg(&dst[tok + 8].src) : -1);
    };
    auto issue_one = [&]() {
      if (issued < nst) {
        issue_rows<D>(ring + slot_i * STAGE, (issued & 1) ? v_new : k_new, src_cur, LH, lh, lane);
        if (issued & 1) {
          src_cur = src_nxt;
          const int ni = (issued >> 1) + 2;
          if (ni < n) src_nxt = fetch_src(ni);
        }
        ++issued;
        slot_i = slot_i + 1 == n_stages ? 0 : slot_i + 1;
      }
      cp_async_commit();                                                 // always: uniform group counting
    };
    if (n > 0) src_cur = fetch_src(0);
    if (n > 1) src_nxt = fetch_src(1);
    for (int k = 0; k + 1 < n_stages; ++k) issue_one();
    __syncthreads();                                                     // the previous segment's readers of B' are done
    // ---- stage B' = B / g (hi + mid + lo) in B-fragment order and the transposed basis --------------------------------------
#pragma unroll 1
    for (int z = 0; z < 2; ++z) {
      const __nv_bfloat16* B = (z ? BV : BK) + ((size_t)(l / g.w) * g.H + h) * (size_t)r * D;
      const __nv_bfloat16* gz = (z ? gV : gK) + (size_t)lh * D;
      for (int idx = tid; idx < NFRAG; idx += NTHR) {
        const int fl = idx & 31, fnt = (idx >> 5) % NT, fkk = (idx >> 5) / NT;
        const int fg = fl >> 2, ft = fl & 3;
        const int ch = 16 * fkk + 2 * ft;                                  // k slots 2t, 2t+1 | 8+2t, 8+2t+1 <-> channels ch, ch+1 | ch+8, ch+9
        const __nv_bfloat16* bp = B + (size_t)(8 * fnt + fg) * D + ch;
        const float2 b01 = bf2(__ldg(reinterpret_cast<const uint32_t*>(bp))), b23 = bf2(__ldg(reinterpret_cast<const uint32_t*>(bp + 8)));
        const float2 g01 = bf2(__ldg(reinterpret_cast<const uint32_t*>(gz + ch))), g23 = bf2(__ldg(reinterpret_cast<const uint32_t*>(gz + ch + 8)));
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
    // destination rows of the current tile and (loaded one stage early, so the table read is off the critical path) of the next
    RowDst ra, rb, na, nb;
    if (n > 0) {
      na = row_dst(arena, ranks4, g.d, dst, 16 * (tb + warp) + gr, n_tok, lh, I8);
      nb = row_dst(arena, ranks4, g.d, dst, 16 * (tb + warp) + gr + 8, n_tok, lh, I8);
    }
    bool any_flag = false;
    int ntmax = NT;
    int slot_c = 0;
#pragma unroll 1
    for (int s = 0; s < nst; ++s) {
      __syncwarp();                                                      // every lane is done with the stage that is refilled now
      issue_one();
      cp_async_wait(n_stages - 1);                                       // this lane's copies of stage s have landed ...
      __syncwarp();                                                      // ... and so have the other lanes' (the reconstruction reads across lanes)
      const uint32_t stage = ring + slot_c * STAGE;
      const int z = s & 1;
      if (z == 0) {
        ra = na; rb = nb;
        any_flag = __any_sync(kFull, ra.flagged() || rb.flagged());
        ntmax = __reduce_max_sync(kFull, max(ra.valid() ? ra.rk() : 0, rb.valid() ? rb.rk() : 0)) >> 3;
      } else if (s + 1 < nst) {
        const int tile = tb + warp + W * ((s + 1) >> 1);
        na = row_dst(arena, ranks4, g.d, dst, 16 * tile + gr, n_tok, lh, I8);
        nb = row_dst(arena, ranks4, g.d, dst, 16 * tile + gr + 8, n_tok, lh, I8);
      }
      uint32_t ca[NT], cb[NT], qa[NT], qb[NT], xa = 0u, xb = 0u;
      project<D, NT, I8>(P4 + z * NFRAG, P2 + z * NFRAG, lane, stage, ra, rb, ntmax, ca, cb, qa, qb, xa, xb);
      if constexpr (I8) {
        store_coef8<NT>(ra, qa, xa, z, t);
        store_coef8<NT>(rb, qb, xb, z, t);
      } else {
        store_coef<NT>(ra, ca, z, t);
        store_coef<NT>(rb, cb, z, t);
      }
      if (any_flag)
        reconstruct_quantise<D, NT>(z, BT + z * D * ldT, ldT, (z ? gV : gK) + (size_t)lh * D + 2 * t, stage, ra, rb, ca, cb, gr, t);
      slot_c = slot_c + 1 == n_stages ? 0 : slot_c + 1;
    }
    asm volatile("cp.async.wait_group 0;" ::: "memory");                 // only empty groups are left
  }
}

// =====================================================================================================================================
// tcgen05 variant (d = 128): the projection and the reconstruction as UMMA tiles of 128 tokens, accumulators in TMEM.
//   tile   = 128 consecutive rows of the call (no sorting: a thread of the epilogue owns one token row = one TMEM lane)
//   MMA 1  : acc[128 x N1] = X[128 x 128] . B1^T, B1 = the three bf16 terms of B' = B / g as separate output columns, ordered
//            [chunk b][term][8 columns] so that one chunk's lo / mid / hi partial sums are three 8-column TMEM loads; N1 = 3r (to 16)
//   epi 1  : c = bf16((lo + mid) + hi), tier mask, fragment-native coefficient stores; the rows of FLAGGED tokens join a batch:
//            coefficients into the A operand of MMA 2, token row and destination into side buffers. The batch (<= 128 rows, gathered
//            over the tiles of one (layer, head, Z) run) is flushed when the run ends or the next tile's flagged rows would not fit
//   MMA 2  : rec[p x 128] = c[p x 64] . B2^T, B2 = the transposed basis padded to 64 ranks
//   epi 2  : thread p < batch rows: e = x - g * rec, int4 quantiser A14, code / scale stores (one thread per row: batching over
//            tiles is what keeps all 128 threads busy -- a single tile has only a handful of flagged rows)
// Warps 0-3: epilogue (and the per-(layer, head) staging of B1 / B2); warp 4 lane 0: TMA producer (two 64-channel halves of 128
// token rows per (tile, Z), hardware 128-byte swizzle); warp 5 lane 0: MMA issuer. mbarrier rings: x_full / x_empty (token
// stages), acc_full / acc_empty (two accumulators), a2_ready / rec_full (second product), basis_ready (operands of a new (l, h)).
constexpr int kCuS = 3;                               // token stages of 32 KB
constexpr int kCuXBytes = 32768;
constexpr int kCuAccCols = 192;                       // columns reserved per projection accumulator (N1 <= 192)

__device__ __forceinline__ void cu_mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void cu_mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void cu_mbar_wait(uint32_t bar, uint32_t parity) {
  // bounded (about 10 s with the back-off): a protocol error traps instead of hanging the GPU
  for (uint32_t spin = 0; spin < (1u << 26); ++spin) {
    uint32_t ok;
    asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                 : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    if (ok) return;
    if (spin > 4096) __nanosleep(128);
  }
  __trap();
}
__device__ __forceinline__ uint64_t cu_desc(uint32_t saddr) {     // K-major, SWIZZLE_128B, 8-row groups 1024 bytes apart, version 1
  return (uint64_t)((saddr >> 4) & 0x3fff) | (1ull << 16) | ((uint64_t)(1024 >> 4) << 32) | (1ull << 46) | (2ull << 61);
}
__device__ __forceinline__ void cu_mma(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t acc) {
  asm volatile("{ .reg .pred p; setp.ne.b32 p, %4, 0; tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p; }"
               ::"r"(tmem_d), "l"(da), "l"(db), "r"(idesc), "r"(acc) : "memory");
}
__device__ __forceinline__ void cu_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void cu_tma_3d(uint32_t dst, const CUtensorMap* map, uint32_t bar, int c0, int c1, int c2) {
  asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
               ::"r"(dst), "l"(map), "r"(bar), "r"(c0), "r"(c1), "r"(c2) : "memory");
}
__device__ __forceinline__ void cu_tmem_ld8(uint32_t taddr, float (&v)[8]) {
  uint32_t r[8];
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]) : "r"(taddr));
#pragma unroll
  for (int i = 0; i < 8; ++i) v[i] = __uint_as_float(r[i]);
}
constexpr int kCuEpiGroups = 2;                       // epilogue warpgroups (each 4 warps = the 4 TMEM lane quadrants)
constexpr int kCuEpi = 128 * kCuEpiGroups, kCuThreads = kCuEpi + 64;
__device__ __forceinline__ void cu_bar_epi() { asm volatile("bar.sync 1, %0;" ::"n"(kCuEpi) : "memory"); }      // the epilogue threads

// the steps of a CTA: its (layer-head, tile) items [item0, item1), per layer-head first all tiles for K, then all for V
struct CuIter {
  int n_tiles, left, lh, z, tile, ta, tb;
  __device__ CuIter(int item0, int item1, int nt) : n_tiles(nt), left(item1 - item0), lh(item0 / nt), z(0) {
    ta = item0 - lh * nt; tb = min(nt, ta + left); tile = ta;
  }
  __device__ bool last_of_run() const { return tile == tb - 1; }
  __device__ void next() {
    if (++tile < tb) return;
    if (z == 0) { z = 1; tile = ta; return; }
    left -= tb - ta; ++lh; z = 0; ta = 0; tb = min(n_tiles, left); tile = 0;
  }
};

struct CuParams {
  const uint8_t* arena;
  const TokDst* dst;            // row order of the call's chunk (unsorted): row i of the chunk = global row row0 + i
  const __nv_bfloat16 *BK, *BV, *gK, *gV, *k_new, *v_new;
  int n_rows;                   // rows of this chunk
  int row0;                     // first global row of the chunk in k_new / v_new
  int N1;                       // 3 r rounded up to 16
  uint32_t ranks4;
  CacheGeom g;
};

__global__ void __launch_bounds__(kCuThreads, 1) compress_umma_kernel(const __grid_constant__ CUtensorMap mapK, const __grid_constant__ CUtensorMap mapV,
                                                               const CuParams p) {
  constexpr int D = 128;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  __shared__ __align__(8) uint64_t bars[2 * kCuS + 8];
  __shared__ uint32_t tmem_base_sh;
  __shared__ int nflag_sh[2], wcount_sh[8];
  const CacheGeom& g = p.g;
  const int r = g.r, N1 = p.N1, LH = g.L * g.H, NC = r / 8;
  const uint32_t sm = ((uint32_t)__cvta_generic_to_shared(smem_raw) + 1023u) & ~1023u;
  // shared-memory map (all 1024-aligned): token stages | B1[z][atom] | B2[z] | A2 | gate[z][128] floats | flagged-row list
  const uint32_t xs0 = sm, b1_0 = xs0 + kCuS * kCuXBytes, b1_atom = (uint32_t)N1 * 128, b2_0 = b1_0 + 4 * b1_atom, a2 = b2_0 + 2 * 16384,
                 gam = a2 + 16384, flist = gam + 1024;
  const uint32_t bar0 = (uint32_t)__cvta_generic_to_shared(bars);
  // a2_ready is a pair (step parity): the epilogue can post two steps before the MMA thread has looked at the first, and a waiter
  // may lag an mbarrier by one phase only
  const uint32_t x_full = bar0, x_empty = bar0 + 8 * kCuS, acc_full = bar0 + 16 * kCuS, acc_empty = acc_full + 16, a2_ready = acc_empty + 16,
                 rec_full = a2_ready + 16, basis_ready = rec_full + 8;
  const int tid_all = threadIdx.x, lane = tid_all & 31, warp = tid_all >> 5;
  const int tid = tid_all & 127, grp_e = tid_all >> 7;       // epilogue: row / TMEM lane of the thread, and its warpgroup (splits chunks)
  const int n_tiles = (p.n_rows + 127) >> 7;
  const long long items = (long long)LH * n_tiles;
  const int item0 = (int)(items * blockIdx.x / gridDim.x), item1 = (int)(items * (blockIdx.x + 1) / gridDim.x);
  const int n_idx = 2 * (item1 - item0);                     // (item, Z) steps of this CTA
  if (tid_all == 0) {
    for (int i = 0; i < 2 * kCuS + 8; ++i) cu_mbar_init(bar0 + 8 * i, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(&mapK) : "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(&mapV) : "memory");
  }
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"((uint32_t)__cvta_generic_to_shared(&tmem_base_sh)) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  for (int i = tid_all; i < 3 * 16384 / 16; i += kCuThreads)            // B2 (both Z) and A2: the ranks >= r stay zero for the whole kernel
    asm volatile("st.shared.v4.u32 [%0], {%1, %1, %1, %1};" ::"r"(b2_0 + 16 * i), "r"(0u) : "memory");
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tmem = tmem_base_sh;
  const uint32_t idesc1 = (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(N1 >> 3) << 17) | ((128u >> 4) << 24);      // both operands K-major
  const uint32_t idesc2 = (1u << 4) | (1u << 7) | (1u << 10) | ((128u >> 3) << 17) | ((128u >> 4) << 24);
  if (warp == 4 * kCuEpiGroups) {
    // ===== TMA producer =========================================================================================================
    if (lane == 0) {
      CuIter it(item0, item1, n_tiles);
      for (int idx = 0; idx < n_idx; ++idx, it.next()) {
        const int s = idx % kCuS;
        if (idx >= kCuS) cu_mbar_wait(x_empty + 8 * s, (uint32_t)(((idx / kCuS) - 1) & 1));
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(x_full + 8 * s), "r"((uint32_t)kCuXBytes) : "memory");
        const CUtensorMap* map = it.z ? &mapV : &mapK;
        cu_tma_3d(xs0 + s * kCuXBytes, map, x_full + 8 * s, 0, it.lh, p.row0 + 128 * it.tile);
        cu_tma_3d(xs0 + s * kCuXBytes + 16384, map, x_full + 8 * s, 64, it.lh, p.row0 + 128 * it.tile);
      }
    }
  } else if (warp == 4 * kCuEpiGroups + 1) {
    // ===== MMA issuer ===========================================================================================================
    if (lane == 0) {
      int n_seg = 0, cur_lh = -1;
      CuIter it(item0, item1, n_tiles);          // the step MMA 1 is issued for next
      auto mma1 = [&](int idx) {
        const int s = idx % kCuS, buf = idx & 1;
        if (it.lh != cur_lh) { cu_mbar_wait(basis_ready, (uint32_t)(n_seg & 1)); ++n_seg; cur_lh = it.lh; }
        cu_mbar_wait(x_full + 8 * s, (uint32_t)((idx / kCuS) & 1));
        if (idx >= 2) cu_mbar_wait(acc_empty + 8 * buf, (uint32_t)(((idx >> 1) - 1) & 1));
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        const uint32_t xs = xs0 + s * kCuXBytes, b1 = b1_0 + (uint32_t)(2 * it.z) * b1_atom;
#pragma unroll
        for (int k = 0; k < 8; ++k)       // channels 16k .. 16k+15: atom k / 4, 32 bytes per step inside the swizzled 128-byte rows
          cu_mma(tmem + buf * kCuAccCols, cu_desc(xs + (k >> 2) * 16384 + 32 * (k & 3)), cu_desc(b1 + (k >> 2) * b1_atom + 32 * (k & 3)), idesc1, k > 0);
        cu_commit(acc_full + 8 * buf);
        cu_commit(x_empty + 8 * s);           // the token stage is free as soon as these products have read it
        it.next();
      };
      int z_cur = 0;
      if (n_idx > 0) { z_cur = it.z; mma1(0); }
      for (int idx = 0; idx < n_idx; ++idx) {
        const int z_this = z_cur;
        const bool more = idx + 1 < n_idx, same_lh = more && it.lh == cur_lh;
        if (same_lh) { z_cur = it.z; mma1(idx + 1); }      // run ahead into the other accumulator while the epilogue of idx works
        cu_mbar_wait(a2_ready + 8 * (idx & 1), (uint32_t)((idx >> 1) & 1));
        if (nflag_sh[idx & 1] > 0) {                       // the epilogue flushes its batch of flagged rows: rec = c . B2^T
          asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
          const uint32_t b2 = b2_0 + (uint32_t)z_this * 16384;
#pragma unroll
          for (int k = 0; k < 4; ++k) cu_mma(tmem + 2 * kCuAccCols, cu_desc(a2 + 32 * k), cu_desc(b2 + 32 * k), idesc2, k > 0);
          cu_commit(rec_full);
        }
        if (!same_lh && more) { z_cur = it.z; mma1(idx + 1); }     // a new (layer, head): staged only after idx is finished
      }
    }
  } else {
    // ===== epilogue warps (128 threads = TMEM lanes) ============================================================================
    const uint32_t rows_sh = flist + 256;                       // RowDst (16 bytes) of the batch of flagged rows
    int cur_lh = -1, n_rec = 0, nb = 0;                         // nb = flagged rows waiting in the batch (CTA-uniform)
    const int wq = warp & 3;                                    // TMEM lane quadrant of this warp
    const uint32_t lane_taddr = (uint32_t)(32 * wq) << 16;
    CuIter it(item0, item1, n_tiles);
    // destination of my row in the current and in the next step (the table read of the next step is off the critical path)
    RowDst rd = row_dst(p.arena, p.ranks4, D, p.dst, 128 * it.tile + tid, p.n_rows, it.lh);
    for (int idx = 0; idx < n_idx; ++idx) {
      const int z = it.z, lh = it.lh, tile_cur = it.tile, buf = idx & 1;
      const bool last_of_run = it.last_of_run();
      it.next();
      // the table row of the next step: the load is issued here, its first use is at the end of this step
      const bool more = idx + 1 < n_idx, vn = more && 128 * it.tile + tid < p.n_rows;
      const TokDst tdn = p.dst[vn ? 128 * it.tile + tid : 0];
      const int lh_next = it.lh;
      if (lh != cur_lh) {
        // ---- operands of this (layer, head): B1 = three-term split of B / g in [chunk][term][8] row order, B2 = B^T, gates ------
        const int l = lh / g.H, h = lh - l * g.H;
        for (int zz = 0; zz < 2; ++zz) {
          const __nv_bfloat16* B = (zz ? p.BV : p.BK) + ((size_t)(l / g.w) * g.H + h) * (size_t)r * D;
          const __nv_bfloat16* gz = (zz ? p.gV : p.gK) + (size_t)lh * D;
          const uint32_t b1 = b1_0 + (uint32_t)(2 * zz) * b1_atom, b2 = b2_0 + (uint32_t)zz * 16384;
          for (int i0 = tid_all; i0 < r * 64; i0 += kCuEpi * 8) {       // 8 (rank, channel pair) items per thread with all loads issued first
            uint32_t bwv[8], gwv[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) {
              const int i = i0 + kCuEpi * u, j = i >> 6, ch = (i & 63) * 2;
              const bool ok = i < r * 64;
              bwv[u] = ok ? __ldg(reinterpret_cast<const uint32_t*>(B + (size_t)j * D + ch)) : 0u;
              gwv[u] = ok ? __ldg(reinterpret_cast<const uint32_t*>(gz + ch)) : 0x3f803f80u;
            }
#pragma unroll
            for (int u = 0; u < 8; ++u) {
              const int i = i0 + kCuEpi * u, j = i >> 6, ch = (i & 63) * 2;
              if (i >= r * 64) break;
              const uint32_t bw = bwv[u];
              const float2 bb = bf2(bw), gg = bf2(gwv[u]);
              uint32_t t3[3];
              split3(__fdiv_rn(bb.x, gg.x), __fdiv_rn(bb.y, gg.y), t3[0], t3[1], t3[2]);
              const uint32_t col = (uint32_t)(ch >> 6) * b1_atom + (uint32_t)(ch & 7) * 2, chunk = (uint32_t)(ch & 63) >> 3;
#pragma unroll
              for (int term = 0; term < 3; ++term) {
                const uint32_t nrow = (uint32_t)(j >> 3) * 24 + 8 * term + (j & 7);
                asm volatile("st.shared.u32 [%0], %1;" ::"r"(b1 + col + nrow * 128 + ((chunk ^ (nrow & 7)) << 4)), "r"(t3[term]) : "memory");
              }
              // B2[ch][j] = B[j][ch]
              asm volatile("st.shared.u16 [%0], %1;" ::"r"(b2 + (uint32_t)ch * 128 + ((((uint32_t)j >> 3) ^ (ch & 7)) << 4) + (j & 7) * 2), "h"((uint16_t)(bw & 0xffff)) : "memory");
              asm volatile("st.shared.u16 [%0], %1;" ::"r"(b2 + (uint32_t)(ch + 1) * 128 + ((((uint32_t)j >> 3) ^ ((ch + 1) & 7)) << 4) + (j & 7) * 2), "h"((uint16_t)(bw >> 16)) : "memory");
            }
          }
          for (int i = tid_all; i < (N1 - 3 * r) * 16; i += kCuEpi) {     // padding rows 3r .. N1-1 of both atoms
            const uint32_t nrow = 3 * r + (i >> 4) % (N1 - 3 * r), c16 = i & 15;
            asm volatile("st.shared.v4.u32 [%0], {%1, %1, %1, %1};" ::"r"(b1 + (c16 >> 3) * b1_atom + nrow * 128 + ((c16 & 7) << 4)), "r"(0u) : "memory");
          }
          for (int i = tid_all; i < D; i += kCuEpi) {
            const float gv = __bfloat162float(gz[i]);
            asm volatile("st.shared.f32 [%0], %1;" ::"r"(gam + (uint32_t)(zz * 128 + i) * 4), "f"(gv) : "memory");
          }
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        cu_bar_epi();
        if (tid_all == 0) cu_mbar_arrive(basis_ready);
        cur_lh = lh;
      }
      // ---- positions of this tile's flagged rows in the batch, and the flagged count of the next tile ---------------------------
      const unsigned bal = __ballot_sync(kFull, rd.flagged());
      if (lane == 0 && grp_e == 0) wcount_sh[wq] = __popc(bal);
      cu_bar_epi();
      int pre = 0, n_flag = 0;
#pragma unroll
      for (int ww = 0; ww < 4; ++ww) { const int cnt = wcount_sh[ww]; pre += ww < wq ? cnt : 0; n_flag += cnt; }
      const int my_p = nb + pre + __popc(bal & ((1u << lane) - 1u));      // nb + n_flag <= 128 by the flush rule below
      // ---- epilogue 1: coefficients ---------------------------------------------------------------------------------------------
      cu_mbar_wait(acc_full + 8 * buf, (uint32_t)((idx >> 1) & 1));
      asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
      {
        const uint32_t taddr = tmem + buf * kCuAccCols + lane_taddr;
        const bool valid = rd.valid(), fl = rd.flagged();
        const int rk = rd.rk(), slot = rd.slot(), tb = rd.tb();
        uint8_t* base = rd.blk + (z ? rd.coef_bytes() : 0);
#pragma unroll 1
        for (int b = grp_e; b < NC; b += kCuEpiGroups) {       // the warpgroups split the rank chunks
          float hi[8], mid[8], lo[8];
          cu_tmem_ld8(taddr + 24 * b, hi);
          cu_tmem_ld8(taddr + 24 * b + 8, mid);
          cu_tmem_ld8(taddr + 24 * b + 16, lo);
          asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
          const bool keep = valid && 8 * b < rk;
          uint32_t wv[4];
#pragma unroll
          for (int k = 0; k < 4; ++k)
            wv[k] = keep ? pack_bf16x2((lo[2 * k] + mid[2 * k]) + hi[2 * k], (lo[2 * k + 1] + mid[2 * k + 1]) + hi[2 * k + 1]) : 0u;
          if (keep) {
            if (z == 0) {
#pragma unroll
              for (int k = 0; k < 4; ++k) *reinterpret_cast<uint32_t*>(base + kcoef_elem_off(slot, 8 * b + 2 * k, tb)) = wv[k];
            } else {
#pragma unroll
              for (int k = 0; k < 4; ++k) {
                *reinterpret_cast<uint16_t*>(base + vcoef_elem_off(slot, 8 * b + 2 * k, tb)) = (uint16_t)(wv[k] & 0xffff);
                *reinterpret_cast<uint16_t*>(base + vcoef_elem_off(slot, 8 * b + 2 * k + 1, tb)) = (uint16_t)(wv[k] >> 16);
              }
            }
          }
          if (fl)
            asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(a2 + (uint32_t)my_p * 128 + (((uint32_t)b ^ (my_p & 7)) << 4)),
                         "r"(wv[0]), "r"(wv[1]), "r"(wv[2]), "r"(wv[3]) : "memory");
        }
        if (fl && grp_e == 0)        // a flagged row joins the batch: its destination and its row index in k_new / v_new (re-read from L2 at the flush)
          asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(rows_sh + 16 * my_p), "r"((uint32_t)(uintptr_t)rd.blk),
                       "r"((uint32_t)((uintptr_t)rd.blk >> 32)), "r"((uint32_t)rd.meta), "r"((uint32_t)(p.row0 + 128 * tile_cur + tid)) : "memory");
      }
      nb += n_flag;
      {   // flagged rows of the next tile (first use of the table row loaded at the top of the step)
        const unsigned baln = __ballot_sync(kFull, vn && tdn.ridx >= 0);
        if (lane == 0 && grp_e == 0) wcount_sh[4 + wq] = __popc(baln);
      }
      asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      cu_bar_epi();
      // flush the batch through MMA 2 when the (layer, head, Z) run ends or the next tile's flagged rows would not fit
      const int n_flag_next = wcount_sh[4] + wcount_sh[5] + wcount_sh[6] + wcount_sh[7];
      const int flush = (nb > 0 && (last_of_run || nb + n_flag_next > 128)) ? nb : 0;
      if (tid_all == 0) {
        cu_mbar_arrive(acc_empty + 8 * buf);
        nflag_sh[idx & 1] = flush;
        cu_mbar_arrive(a2_ready + 8 * (idx & 1));
      }
      // ---- epilogue 2: residuals of the batch (thread p owns batch row p; its rec is in TMEM lane p) ------------------------------
      if (flush > 0) {
        cu_mbar_wait(rec_full, (uint32_t)(n_rec & 1));
        ++n_rec;
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        if (32 * wq < flush) {                                   // warp-uniform: this warp's lanes hold batch rows
          const bool act = tid < flush;
          RowDst rq = rd;
          if (act) {
            uint32_t b0, b1w, mt, sr;
            asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(b0), "=r"(b1w), "=r"(mt), "=r"(sr) : "r"(rows_sh + 16 * tid));
            rq.blk = reinterpret_cast<uint8_t*>((uintptr_t)b0 | ((uintptr_t)b1w << 32)); rq.meta = (int)mt; rq.src = (int)sr;
          }
          const uint4* xg = reinterpret_cast<const uint4*>((z ? p.v_new : p.k_new) + ((size_t)(act ? rq.src : 0) * LH + lh) * D);
          const uint32_t taddr = tmem + 2 * kCuAccCols + lane_taddr;
          const int slot = rq.slot(), sj = slot >> 3, sg = slot & 7;
          uint8_t* res = rq.blk + 2 * rq.coef_bytes();            // [K code | K scale | V code | V scale], sub-block of 16 slots
          uint4 xn[4];
#pragma unroll
          for (int c = 0; c < 4; ++c) xn[c] = __ldg(xg + 4 * grp_e + c);
#pragma unroll 1
          for (int gp = grp_e; gp < D / 32; gp += kCuEpiGroups) {  // pairs of 16-channel groups (split over the warpgroups): channels 32 gp .. + 31
            uint4 xc[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) { xc[c] = xn[c]; xn[c] = __ldg(xg + 4 * min(gp + kCuEpiGroups, D / 32 - 1) + c); }     // next pair's row chunks in flight
            float rec[32];
#pragma unroll
            for (int c = 0; c < 4; ++c) cu_tmem_ld8(taddr + 32 * gp + 8 * c, *reinterpret_cast<float(*)[8]>(rec + 8 * c));
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
            if (act) {
              int code[32];
              __half sc[2];
#pragma unroll
              for (int gg = 0; gg < 2; ++gg) {
                float e[16];
                float amax = 0.f;
#pragma unroll
                for (int c = 0; c < 2; ++c) {                      // two 8-channel chunks of the group
                  const int ch0 = 32 * gp + 16 * gg + 8 * c;
                  uint4 xv, g0, g1;
                  xv = xc[2 * gg + c];
                  asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(g0.x), "=r"(g0.y), "=r"(g0.z), "=r"(g0.w) : "r"(gam + (uint32_t)(z * 128 + ch0) * 4));
                  asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(g1.x), "=r"(g1.y), "=r"(g1.z), "=r"(g1.w) : "r"(gam + (uint32_t)(z * 128 + ch0 + 4) * 4));
                  const uint32_t xw[4] = {xv.x, xv.y, xv.z, xv.w};
                  const float gm[8] = {__uint_as_float(g0.x), __uint_as_float(g0.y), __uint_as_float(g0.z), __uint_as_float(g0.w),
                                       __uint_as_float(g1.x), __uint_as_float(g1.y), __uint_as_float(g1.z), __uint_as_float(g1.w)};
#pragma unroll
                  for (int k = 0; k < 4; ++k) {
                    const float2 xx = bf2(xw[k]);
                    e[8 * c + 2 * k] = fmaf(-gm[2 * k], rec[16 * gg + 8 * c + 2 * k], xx.x);
                    e[8 * c + 2 * k + 1] = fmaf(-gm[2 * k + 1], rec[16 * gg + 8 * c + 2 * k + 1], xx.y);
                    amax = fmaxf(amax, fmaxf(fabsf(e[8 * c + 2 * k]), fabsf(e[8 * c + 2 * k + 1])));
                  }
                }
                sc[gg] = quant_scale(amax);
                const float sf = __half2float(sc[gg]);
#pragma unroll
                for (int i = 0; i < 16; ++i) code[16 * gg + i] = (quant_code(e[i], sf) + 8) & 15;     // offset binary
              }
              if (z == 0) {
                // K codes: word (slot, t) of group pair gp holds, for gg, b, hi: channel 32gp + 16gg + 8b + 2t + hi at bit 4(2gg + b) + 16hi
#pragma unroll
                for (int t = 0; t < 4; ++t) {
                  uint32_t wd = 0u;
#pragma unroll
                  for (int gg = 0; gg < 2; ++gg)
#pragma unroll
                    for (int b = 0; b < 2; ++b)
#pragma unroll
                      for (int hi = 0; hi < 2; ++hi) wd |= (uint32_t)code[16 * gg + 8 * b + 2 * t + hi] << (4 * (2 * gg + b) + 16 * hi);
                  *reinterpret_cast<uint32_t*>(res + sj * 4 * D + (4 * sg + t) * (D / 8) + 4 * gp) = wd;
                }
#pragma unroll
                for (int gg = 0; gg < 2; ++gg) *reinterpret_cast<__half*>(res + 8 * D + scale_elem_off(slot, 2 * gp + gg, D)) = sc[gg];
              } else {
                // V codes: byte (2 * hi + tile) of word (4 * gch + ts) * (D / 4) + 4 * grp holds channels gch (low nibble) and gch + 8
                const int ts = sg >> 1, hs = sg & 1;
#pragma unroll
                for (int gg = 0; gg < 2; ++gg) {
                  uint8_t* cv = res + 10 * D + 4 * (2 * gp + gg) + 2 * hs + sj;
#pragma unroll
                  for (int gch = 0; gch < 8; ++gch) cv[(4 * gch + ts) * (D / 4)] = (uint8_t)(code[16 * gg + gch] | (code[16 * gg + 8 + gch] << 4));
                  *reinterpret_cast<__half*>(res + 18 * D + scale_elem_off(slot, 2 * gp + gg, D)) = sc[gg];
                }
              }
            }
          }
        }
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        cu_bar_epi();                                               // the batch buffers and the rec columns are free again
        nb = 0;
      }
      if (more) rd = row_dst_from(p.arena, p.ranks4, D, tdn, vn, lh_next);
    }
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem) : "memory");
}

typedef CUresult (*CuEncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                    const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
bool cu_make_row_map(CUtensorMap* m, const void* base, uint64_t LH, uint64_t rows) {     // dims (128 channels, LH, rows), box (64, 1, 128)
  static CuEncodeTiledFn fn = [] {
    void* q = nullptr;
    cudaDriverEntryPointQueryResult st;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &q, cudaEnableDefault, &st) != cudaSuccess || st != cudaDriverEntryPointSuccess) q = nullptr;
    return (CuEncodeTiledFn)q;
  }();
  if (!fn) return false;
  const cuuint64_t dims[3] = {128, LH, rows}, strides[2] = {256, LH * 256};
  const cuuint32_t box[3] = {64, 1, 128}, es[3] = {1, 1, 1};
  return fn(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(base), dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

}  // namespace

bool compress_umma_supported(const CacheGeom& g, const void* k_new, const void* v_new) {
  return g.d == 128 && g.r <= 48 && ((((uintptr_t)k_new | (uintptr_t)v_new) & 15) == 0);
}

// rows [row0, row0 + n_rows) of k_new / v_new (total_rows rows in all), dst = their destinations in row order (not sorted)
int launch_compress_umma(const uint8_t* arena, const CacheGeom& g, const TokDst* dst, int n_rows, int row0, long long total_rows,
                         const __nv_bfloat16* k_new, const __nv_bfloat16* v_new, const __nv_bfloat16* BK, const __nv_bfloat16* BV,
                         const __nv_bfloat16* gK, const __nv_bfloat16* gV, int n_sms, cudaStream_t s) {
  if (n_rows <= 0) return 0;
  CUtensorMap mapK, mapV;
  const uint64_t LH = (uint64_t)g.L * g.H;
  if (!cu_make_row_map(&mapK, k_new, LH, (uint64_t)total_rows) || !cu_make_row_map(&mapV, v_new, LH, (uint64_t)total_rows)) return 0;
  CuParams p;
  p.arena = arena; p.dst = dst; p.BK = BK; p.BV = BV; p.gK = gK; p.gV = gV; p.k_new = k_new; p.v_new = v_new; p.n_rows = n_rows; p.row0 = row0;
  p.N1 = (3 * g.r + 15) / 16 * 16;
  p.ranks4 = (uint32_t)g.tier_rank[0] | ((uint32_t)g.tier_rank[1] << 8) | ((uint32_t)g.tier_rank[2] << 16) | ((uint32_t)g.tier_rank[3] << 24);
  p.g = g;
  const size_t smem = 1024 + (size_t)kCuS * kCuXBytes + (size_t)4 * p.N1 * 128 + 2 * 16384 + 16384 + 1024 + 256 + 2048;
  const long long items = (long long)LH * ((n_rows + 127) / 128);
  const int grid = (int)std::max<long long>(1, std::min<long long>(n_sms, items));
  cudaFuncSetAttribute(compress_umma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  compress_umma_kernel<<<grid, kCuThreads, smem, s>>>(mapK, mapV, p);
  return 1;
}

int launch_compress_mma(const uint8_t* arena, const CacheGeom& g, const TokDst* dst, int n, const CompressRuns& runs, const __nv_bfloat16* k_new,
                        const __nv_bfloat16* v_new, const __nv_bfloat16* BK, const __nv_bfloat16* BV, const __nv_bfloat16* gK,
                        const __nv_bfloat16* gV, int n_sms, cudaStream_t s) {
  if (n <= 0) return 0;
  const int nfrag = (g.d / 16) * (g.r / 8) * 32;
  const size_t fixed = (size_t)2 * nfrag * 24 + (size_t)2 * g.d * (g.r + 8) * 2, stage = (size_t)16 * (2 * g.d + 16);
  const size_t cap = 227 * 1024;
  // warps per CTA and ring stages per warp: 16 warps (the kernel is latency-bound: 4 warps per scheduler) if they can have 2
  // stages each, else 8 warps
  int warps = kCompressMaxWarps, stages = (int)std::min<size_t>(4, (cap - fixed) / (warps * stage));
  if (stages < 2) { warps = 8; stages = (int)std::min<size_t>(4, (cap - fixed) / (warps * stage)); }
  if (stages < 2) return 0;
  const size_t smem = fixed + (size_t)warps * stages * stage;
  const long long tiles = (long long)g.L * g.H * ((n + 15) / 16);
  const int grid = (int)std::max<long long>(1, std::min<long long>((long long)n_sms, tiles));
  bool ok = true;
#define DWKV_COMPRESS_CASE(DD, NN)                                                                                              \
  case NN:                                                                                                                      \
    if (g.i8) {                                                                                                                 \
      cudaFuncSetAttribute(compress_mma_kernel<DD, NN, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);          \
      compress_mma_kernel<DD, NN, true><<<grid, warps * 32, smem, s>>>(arena, g, dst, n, runs, stages, k_new, v_new, BK, BV, gK, gV); \
    } else {                                                                                                                    \
      cudaFuncSetAttribute(compress_mma_kernel<DD, NN, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);         \
      compress_mma_kernel<DD, NN, false><<<grid, warps * 32, smem, s>>>(arena, g, dst, n, runs, stages, k_new, v_new, BK, BV, gK, gV); \
    }                                                                                                                           \
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
