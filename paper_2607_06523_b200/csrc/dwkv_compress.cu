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
// V-code byte and scale is owned by exactly one (token, lane), so no atomics are needed (free pages are always all zero: dwkv_api.cu, zero_pages).
#include <algorithm>

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

// Reading A14: fp32 IEEE, round-to-nearest-even, no FMA contraction: code = clamp(rint(RN(e / sf)), -7, 7), stored as code + 8.
// Fast path, for a scale that is a normal fp16 number below the fp16 maximum (then |e / sf| <= 7 (1 + 2^-24) / (1 - 2^-11) < 7.004
// for every element of the group and the clamp can never act): ONE approximate reciprocal per group and per code
//     s8 = fma(e, rinv, 8)      r8 = rint(s8)      code + 8 = (int) r8
// s8 differs from e / sf + 8 by less than 2^-19 (reciprocal: 2^-22 relative of a value below 8) + 2^-21 (one rounding in [8, 16)),
// and RN(e / sf) differs from e / sf by at most 2^-21; so if s8 is further than 2^-16 from every half-integer, r8 - 8 is the
// correctly rounded quotient's integer. Only a group with a code inside that margin (a few per 10^5), or with a subnormal / saturated
// scale, takes the IEEE divisions (one cold non-inlined copy). The result is bit-identical to the plain form for every input.
__device__ __forceinline__ float rcp_approx(float x) {
  float y;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
static __device__ __noinline__ float quant_code_exact(float e, float sf) {      // cold: clamp(rint(RN(e / sf)), -7, 7) + 8
  return fminf(fmaxf(rintf(__fdiv_rn(e, sf)), -7.f), 7.f) + 8.f;
}
// the four codes (+ 8) a lane owns of one group; sf != 0
__device__ __forceinline__ void quant_codes4(const float (&e)[4], float sf, int (&code)[4]) {
  const float rinv = rcp_approx(sf);
  float r8[4], dev = 0.f;
#pragma unroll
  for (int x = 0; x < 4; ++x) {
    const float s8 = fmaf(e[x], rinv, 8.f);
    r8[x] = rintf(s8);
    dev = fmaxf(dev, fabsf(s8 - r8[x]));
  }
  if (dev > 0.5f - 0x1p-16f || sf < 0x1p-14f || sf >= 65504.f) {        // rare
#pragma unroll
    for (int x = 0; x < 4; ++x) r8[x] = quant_code_exact(e[x], sf);
  }
#pragma unroll
  for (int x = 0; x < 4; ++x) code[x] = (int)r8[x];
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
// A stage holds the 16 token rows of one tile for one Z, row-major with a row pitch of 2 * D bytes and the 16-byte chunks of a
// row XOR-swizzled: chunk c of row r sits at chunk c ^ f(r), f(r) = ((r & 1) << 2) | ((r >> 1) & 3) (a bijection of r mod 8 whose
// bit 2 is the row's parity). Lane (g, t) copies channels 32u + 8t .. +7 of rows g and g + 8 with 16-byte cp.async (zero-filled
// for rows beyond n_tok): a quarter warp writes two neighbouring rows, which the swizzle sends to different 64-byte halves of the
// banks; ldmatrix (8 rows, one chunk) and the reconstruction's 4-byte reads (8 rows x 4 words of one chunk) see 8 distinct chunk
// positions: all three patterns are conflict-free (the padded layout this replaces cost 2 - 3 wavefronts per cp.async quarter).
// One ldmatrix.x4 per k step returns the A fragment of the projection as an aligned register quad. A stage is complete for the
// warp after cp.async.wait_group + __syncwarp. Stages are 256-byte aligned (the swizzle is applied by XOR on the address).
__device__ __forceinline__ uint32_t stage_swz(int row) { return (uint32_t)(((row & 1) << 2) | ((row >> 1) & 3)); }
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
__device__ __forceinline__ void issue_rows(uint32_t stage, const char* xlh /* X + (lh * D + 8t) elements */, int2 src, uint32_t row_bytes,
                                           int lane) {
  constexpr int PITCH = 2 * D;
  const int g = lane >> 2, t = lane & 3;
  const char* pa = xlh + (size_t)(uint32_t)max(src.x, 0) * row_bytes;
  const char* pb = xlh + (size_t)(uint32_t)max(src.y, 0) * row_bytes;
  const int sa = src.x >= 0 ? 16 : 0, sb = src.y >= 0 ? 16 : 0;
  const uint32_t da = (stage + g * PITCH) | (16u * ((uint32_t)t ^ stage_swz(g))), db = da + 8 * PITCH;     // f(g + 8) = f(g)
#pragma unroll
  for (int u = 0; u < D / 32; ++u) {
    cp_async16(da ^ (64u * u), pa + 64 * u, sa);
    cp_async16(db ^ (64u * u), pb + 64 * u, sb);
  }
}

// bf16 pair (channels ch, ch+1; ch even) of row `row` of a stage
template <int D>
__device__ __forceinline__ uint32_t stage_x(uint32_t stage, int row, int ch) {
  return lds32((stage + row * (2 * D)) | ((((uint32_t)ch >> 3) ^ stage_swz(row)) << 4) | ((ch & 7) * 2));
}

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
  const int arow = (lane & 7) + 8 * ((lane >> 3) & 1);
  const uint32_t am = (stage + arow * (2 * D)) | (16u * ((uint32_t)(lane >> 4) ^ stage_swz(arow)));       // chunk 2kk + (lane >> 4), swizzled
#pragma unroll
  for (int kk = 0; kk < D / 16; ++kk) {
    uint32_t a0, a1, a2, a3;
    ldmatrix_x4(am ^ (32u * kk), a0, a1, a2, a3);
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

// Coefficient stores of one row: the position of (slot, lane) inside the class plane is formed once, the rank chunks follow at a
// constant stride (kcoef_elem_off / vcoef_elem_off of dwkv_layout.cuh with col = 8 nt + 2t, TB = tiles per sub-block: 2 if the
// token is flagged, else 4; compile-time so that the chunk offsets are immediates).
// 8-bit planes: the row's code bytes (two columns per chunk and lane) and, from lane t = 0, the exponent bytes of its blocks
template <int NT, int TB>
__device__ __forceinline__ void store_coef8_tb(const RowDst& rd, const uint32_t (&q)[NT], const uint32_t xexp, int z, int t) {
  const int sl = rd.slot(), rk = rd.rk();
  uint8_t* plane = rd.blk + (z ? rd.coef_bytes() : 0);
  if (z == 0) {
    uint8_t* p = plane + (4 * (sl & 7) + t) * 2 * TB + (sl >> 3) * 2;
#pragma unroll
    for (int nt = 0; nt < NT; ++nt)
      if (8 * nt < rk) *reinterpret_cast<uint16_t*>(p + nt * 64 * TB) = (uint16_t)q[nt];
  } else {
    uint8_t* p = plane + (8 * t + ((sl & 7) >> 1)) * 2 * TB + (sl >> 3) * 2 + (sl & 1);
#pragma unroll
    for (int nt = 0; nt < NT; ++nt)
      if (8 * nt < rk) {
        p[nt * 64 * TB] = (uint8_t)(q[nt] & 0xff);
        p[nt * 64 * TB + 8 * TB] = (uint8_t)(q[nt] >> 8);
      }
  }
  if (t == 0) {
#pragma unroll
    for (int b = 0; b < (NT + 3) / 4; ++b)
      if (32 * b < rk) plane[coef8_exp_off(sl, rk >> 3, TB, b)] = (uint8_t)(xexp >> (8 * b));
  }
}
template <int NT>
__device__ __forceinline__ void store_coef8(const RowDst& rd, const uint32_t (&q)[NT], const uint32_t xexp, int z, int t) {
  if (!rd.valid()) return;
  if (rd.flagged()) store_coef8_tb<NT, 2>(rd, q, xexp, z, t);
  else store_coef8_tb<NT, 4>(rd, q, xexp, z, t);
}

template <int NT, int TB>
__device__ __forceinline__ void store_coef_tb(const RowDst& rd, const uint32_t (&cw)[NT], int z, int t) {
  const int sl = rd.slot(), rk = rd.rk();
  if (z == 0) {
    uint8_t* p = rd.blk + (4 * (sl & 7) + t) * 4 * TB + (sl >> 3) * 4;
#pragma unroll
    for (int nt = 0; nt < NT; ++nt)
      if (8 * nt < rk) *reinterpret_cast<uint32_t*>(p + nt * 128 * TB) = cw[nt];
  } else {
    uint8_t* p = rd.blk + rd.coef_bytes() + (8 * t + ((sl & 7) >> 1)) * 4 * TB + (sl >> 3) * 4 + (sl & 1) * 2;
#pragma unroll
    for (int nt = 0; nt < NT; ++nt)
      if (8 * nt < rk) {
        *reinterpret_cast<uint16_t*>(p + nt * 128 * TB) = (uint16_t)(cw[nt] & 0xffff);
        *reinterpret_cast<uint16_t*>(p + nt * 128 * TB + 16 * TB) = (uint16_t)(cw[nt] >> 16);
      }
  }
}
template <int NT>
__device__ __forceinline__ void store_coef(const RowDst& rd, const uint32_t (&cw)[NT], int z, int t) {
  if (!rd.valid()) return;
  if (rd.flagged()) store_coef_tb<NT, 2>(rd, cw, z, t);
  else store_coef_tb<NT, 4>(rd, cw, z, t);
}

// rec = c . B, e = x - g * rec, int4 quantiser (A14), fragment-native code / scale stores: tiles with a flagged token only.
// x is read from the shared-memory stage in the unpermuted channel order of the reconstruction's n dimension; the loop is kept
// rolled so the kernel stays inside the instruction cache. The store positions of a row depend on (z, slot, t) only: they are
// formed once, as 32-bit offsets from the row's sub-block base, and advance by 4 bytes per group.
template <int D, int NT>
__device__ __forceinline__ void reconstruct_quantise(const int z, const __nv_bfloat16* BTz, const int ldT, const __nv_bfloat16* gt,
                                                     const uint32_t stage, const RowDst& ra, const RowDst& rb,
                                                     const uint32_t (&ca)[NT], const uint32_t (&cb)[NT], const int gr, const int t) {
  // residual planes of a sub-block of 16 slots, behind the two coefficient planes: [K code 8D | K scale 2D | V code 8D | V scale 2D]
  int code_off[2], scale_off[2];
#pragma unroll
  for (int row = 0; row < 2; ++row) {
    const RowDst& rd = row ? rb : ra;
    const int sl = rd.slot(), j = sl >> 3, p = sl & 7, res = 2 * rd.coef_bytes();
    // K: 16-byte code row of (slot, t): word wx at + 4 wx.  V: byte (2 hi + j) of word (4 gch + ts) * (D / 4) + 4 grp, gch = 2t, 2t + 1
    code_off[row] = z == 0 ? res + j * 4 * D + (4 * p + t) * (D / 8) : res + 10 * D + 2 * (p & 1) + j + (8 * t + (p >> 1)) * (D / 4);
    scale_off[row] = res + (z == 0 ? 8 * D : 18 * D) + scale_elem_off(sl, 0, D);
  }
  const bool fa = ra.flagged(), fb = rb.flagged();
#pragma unroll 1
  for (int wx = 0; wx < D / 32; ++wx) {     // K code word wx of a row = groups 2wx, 2wx+1 (registers q = 4wx .. 4wx+3)
    uint32_t kw[2] = {0u, 0u};
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
        const float2 x0 = bf2(stage_x<D>(stage, gr + 8 * row, 16 * grp + 2 * t));          // rows beyond n_tok were zero-filled
        const float2 x2 = bf2(stage_x<D>(stage, gr + 8 * row, 16 * grp + 8 + 2 * t));
        float e[4];
        e[0] = fmaf(-g0.x, rec[0][2 * row], x0.x); e[1] = fmaf(-g0.y, rec[0][2 * row + 1], x0.y);
        e[2] = fmaf(-g2.x, rec[1][2 * row], x2.x); e[3] = fmaf(-g2.y, rec[1][2 * row + 1], x2.y);
        float amax = fmaxf(fmaxf(fabsf(e[0]), fabsf(e[1])), fmaxf(fabsf(e[2]), fabsf(e[3])));
        amax = fmaxf(amax, __shfl_xor_sync(kFull, amax, 1));
        amax = fmaxf(amax, __shfl_xor_sync(kFull, amax, 2));
        if (row ? fb : fa) {
          uint8_t* blk = row ? rb.blk : ra.blk;
          const __half s = quant_scale(amax);
          const float sf = __half2float(s);
          int code[4] = {8, 8, 8, 8};                  // sf == 0 (amax / 7 rounds to zero in fp16): codes 0
          if (sf != 0.f) quant_codes4(e, sf, code);
          if (z == 0) {
            kw[row] |= ((uint32_t)code[0] << (8 * gg)) | ((uint32_t)code[1] << (16 + 8 * gg)) |
                       ((uint32_t)code[2] << (8 * gg + 4)) | ((uint32_t)code[3] << (16 + 8 * gg + 4));
          } else {
            uint8_t* cv = blk + code_off[row] + 4 * grp;
            cv[0] = (uint8_t)(code[0] | (code[2] << 4));
            cv[D] = (uint8_t)(code[1] | (code[3] << 4));
          }
          if (t == 0) *reinterpret_cast<__half*>(blk + scale_off[row] + 4 * grp) = s;
        }
      }
    }
    if (z == 0) {
      if (fa) *reinterpret_cast<uint32_t*>(ra.blk + code_off[0] + 4 * wx) = kw[0];
      if (fb) *reinterpret_cast<uint32_t*>(rb.blk + code_off[1] + 4 * wx) = kw[1];
    }
  }
}

template <int D, int NT, bool I8>      // NT = basis rank / 8; I8 = 8-bit coefficient planes (option "coef_int8")
__global__ void __launch_bounds__(kCompressMaxWarps * 32, 1)
compress_mma_kernel(const uint8_t* arena, const CacheGeom g, const TokDst* dst, const int n_tok, const CompressRuns runs, const int n_stages,
                    const __nv_bfloat16* k_new, const __nv_bfloat16* v_new, const __nv_bfloat16* BK, const __nv_bfloat16* BV,
                    const __nv_bfloat16* gK, const __nv_bfloat16* gV) {
  constexpr int NKK = D / 16, r = 8 * NT, ldT = r + 8, NFRAG = NKK * NT * 32, STAGE = 16 * (2 * D);
  extern __shared__ __align__(256) uint8_t smem_raw[];
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
    const char* xk = reinterpret_cast<const char*>(k_new + (size_t)lh * D + 8 * t);      // row 0 of this (layer, head), this lane's channels
    const char* xv = reinterpret_cast<const char*>(v_new + (size_t)lh * D + 8 * t);
    const uint32_t row_bytes = (uint32_t)LH * D * 2;
    int2 src_cur = make_int2(-1, -1), src_nxt = make_int2(-1, -1);       // source rows (-1: beyond n_tok) of the tile being issued / the next
    auto fetch_src = [&](int i) {
      const int tok = 16 * (tb + warp + W * i) + gr;
      return make_int2(tok < n_tok ? __ldg(&dst[tok].src) : -1, tok + 8 < n_tok ? __ldg(&dst[tok + 8].src) : -1);
    };
    auto issue_one = [&]() {
      if (issued < nst) {
        issue_rows<D>(ring + slot_i * STAGE, (issued & 1) ? xv : xk, src_cur, row_bytes, lane);
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
      }
      // table entries of the next tile: requested here, turned into destinations after this stage's arithmetic (the conversion is
      // a chain of dependent integer operations: placed right behind the loads it was the kernel's largest single stall)
      TokDst tda, tdb;
      bool va = false, vb = false;
      const bool fetch_next = z == 1 && s + 1 < nst;
      if (fetch_next) {
        const int tok = 16 * (tb + warp + W * ((s + 1) >> 1)) + gr;
        va = tok < n_tok; vb = tok + 8 < n_tok;
        tda = dst[va ? tok : 0]; tdb = dst[vb ? tok + 8 : 0];
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
      if (fetch_next) {
        na = row_dst_from(arena, ranks4, g.d, tda, va, lh, I8);
        nb = row_dst_from(arena, ranks4, g.d, tdb, vb, lh, I8);
      }
      slot_c = slot_c + 1 == n_stages ? 0 : slot_c + 1;
    }
    asm volatile("cp.async.wait_group 0;" ::: "memory");                 // only empty groups are left
  }
}

}  // namespace

int launch_compress_mma(const uint8_t* arena, const CacheGeom& g, const TokDst* dst, int n, const CompressRuns& runs, const __nv_bfloat16* k_new,
                        const __nv_bfloat16* v_new, const __nv_bfloat16* BK, const __nv_bfloat16* BV, const __nv_bfloat16* gK,
                        const __nv_bfloat16* gV, int n_sms, cudaStream_t s) {
  if (n <= 0) return 0;
  const int nfrag = (g.d / 16) * (g.r / 8) * 32;
  const size_t fixed = (size_t)2 * nfrag * 24 + (size_t)2 * g.d * (g.r + 8) * 2, stage = (size_t)16 * (2 * g.d);
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
