// dwkv_scan3.cuh -- the fused decode kernel (SURVEY.md section 8a steps a1 + a2; "fused kernel").
//
// ONE persistent launch per decode call covers the q -> basis pre-projection and the split-T scan of every class:
//   * grid = one CTA of 8 warps per SM; every WARP owns a contiguous, cost-balanced slice of the linear order
//         (sequence b, layer*head lh, unit u of b, sub-block)            -- "lh-major": a slice stays inside one or two
//     (b, lh) SEGMENTS, so the online-softmax state (m, l, a[r], e[d]) lives in registers across units and classes and
//     a warp writes ONE partial per segment it touches (a handful per segment instead of one per unit);
//   * at the start of a segment the warp projects q into basis space itself (a1): q~ = cscale * BK . (gK * q) on the
//     tensor cores, hi/lo bf16 split of both operands (16 significant bits), result left in MMA A-fragment registers;
//   * cache bytes stream through a private shared-memory ring filled by cp.async.bulk (TMA engine, 1-D, no tensor map)
//     with one mbarrier per slot; a fetch cursor runs up to NS stages ahead ACROSS unit / class / segment boundaries and
//     leaves a 16-byte stage descriptor for the compute side, so the pipeline never drains inside a slice;
//   * contractions are mma.sync.m16n8k16 on fragment-native data (dwkv_layout.cuh). With G <= 4 query heads per kv head
//     the kernel runs in PAIR mode: the 16 MMA rows carry (4 heads) x (2 token tiles) x (hi, lo part) through
//     block-diagonal A operands, so all 32 lanes hold live scores and q~ / p keep 16 bits at no extra MMA;
//     with 4 < G <= 8 (FULL mode) rows are (8 heads) x (hi, lo);
//   * softmax uses a lazily raised reference (rescale only when a score exceeds it by 2^8).
// K-hat / V-hat are never formed. Algebra: SURVEY.md section 8 box (log2 domain, cscale = softmax_scale * log2 e).
#pragma once
#include "dwkv_internal.h"
#include "dwkv_mma.cuh"

namespace dwkv {
namespace s3 {
using namespace dwkv::dev;

constexpr int kWarps = 8;
constexpr int kRingBytes = 27648;   // per warp
constexpr int kMaxSlots = 8;
constexpr int kWarpSmem = kRingBytes + kMaxSlots * 16 + kMaxSlots * 8;
constexpr float kLazy = 8.0f;       // rescale when a score exceeds the reference by more than this (log2 units)

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
               "l"(src), "r"(bytes), "r"(bar)
               : "memory");
}
__device__ __forceinline__ bool mbar_try(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
      : "=r"(ok)
      : "r"(bar), "r"(parity)
      : "memory");
  return ok != 0;
}
// the common case (the stage has landed) is one try; the slow path is bounded: a bulk copy that never lands (a bad plan, a lost
// expect_tx) traps after 2^28 polls (seconds) instead of hanging the GPU
static __device__ __noinline__ void mbar_wait_slow(uint32_t bar, uint32_t parity) {
  for (uint32_t spins = 0; !mbar_try(bar, parity); ++spins)
    if (spins == (1u << 28)) __trap();
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  if (!mbar_try(bar, parity)) mbar_wait_slow(bar, parity);
}
__device__ __forceinline__ uint4 lds128(uint32_t a) {
  uint4 r;
  asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "r"(a));
  return r;
}
__device__ __forceinline__ uint2 lds64(uint32_t a) {
  uint2 r;
  asm volatile("ld.shared.v2.u32 {%0,%1}, [%2];" : "=r"(r.x), "=r"(r.y) : "r"(a));
  return r;
}
__device__ __forceinline__ uint32_t lds32(uint32_t a) {
  uint32_t r;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(r) : "r"(a));
  return r;
}
// 8-bit coefficient mode: bytes 2k, 2k+1 of w (offset-binary codes u = code + 128) -> bf16x2 (code_lo, code_hi), exact.
// PRMT builds the float 2^23 + u (bytes u, 0, 0, 0x4B), the subtraction of 2^23 + 128 is exact, the pack rounds nothing (|code| <= 128).
__device__ __forceinline__ uint32_t u8pair_to_bf16x2(uint32_t w, int k) {
  uint32_t f0, f1;
  asm("prmt.b32 %0, %1, %2, %3;" : "=r"(f0) : "r"(w), "r"(0x4B000000u), "r"(0x7440u | (uint32_t)(2 * k)));
  asm("prmt.b32 %0, %1, %2, %3;" : "=r"(f1) : "r"(w), "r"(0x4B000000u), "r"(0x7440u | (uint32_t)(2 * k + 1)));
  return pack_bf16x2(__uint_as_float(f0) - 8388736.f, __uint_as_float(f1) - 8388736.f);
}
// 8-bit coefficient mode, K side: bytes 2k, 2k+1 of w -> f16x2 (code_lo, code_hi), exact: one PRMT builds (0x6400 | u) = 1024 + u
// twice, one packed subtraction of 1152 = 1024 + 128 removes the offset (fp16 has ulp 1 in [1024, 2048)).
__device__ __forceinline__ uint32_t u8pair_to_f16x2(uint32_t w, int k) {
  uint32_t x, r;
  asm("prmt.b32 %0, %1, %2, %3;" : "=r"(x) : "r"(w), "r"(0x64646464u), "r"(k ? 0x4342u : 0x4140u));
  asm("sub.f16x2 %0, %1, %2;" : "=r"(r) : "r"(x), "r"(0x64806480u));
  return r;
}
// score MMAs of the 8-bit mode: q~ (hi + lo in fp16) x integer codes in fp16
__device__ __forceinline__ void mma16h(float (&d)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t b0, uint32_t b1) {
  asm("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
      : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
      : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
__device__ __forceinline__ void mma8h(float (&d)[4], uint32_t a0, uint32_t a1, uint32_t b0) {
  asm("mma.sync.aligned.m16n8k8.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5}, {%6}, {%0,%1,%2,%3};"
      : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
      : "r"(a0), "r"(a1), "r"(b0));
}
// exponent byte (e + 127) at bit position sh of w -> 2^e
// (one PRMT isolates the byte, the multiply by 2^23 can issue on the FMA pipe: the ALU pipe is the busy one in this mode)
__device__ __forceinline__ float exp_byte_to_scale(uint32_t w, int sh) {
  return __uint_as_float(__byte_perm(w, 0u, 0x4440u + (uint32_t)(sh >> 3)) * 0x00800000u);
}
__device__ __forceinline__ void sts128(uint32_t a, int x, int y, int z, int w) {
  asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};" ::"r"(a), "r"(x), "r"(y), "r"(z), "r"(w) : "memory");
}
// D(16x8) += A(16x16) . B(16x8), bf16 operands, fp32 accumulate, all four accumulator registers live
__device__ __forceinline__ void mma16(float (&d)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t b0,
                                      uint32_t b1) {
  asm("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
      : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
      : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
// D = A . B + C with C in registers of its own (the persistent (-m_ref, -m_ref, 0, 0) quad of the score MMAs: no per-sub-block copy)
__device__ __forceinline__ void mma16c(float (&d)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t b0, uint32_t b1,
                                       const float (&c)[4]) {
  asm("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%10,%11,%12,%13};"
      : "=f"(d[0]), "=f"(d[1]), "=f"(d[2]), "=f"(d[3])
      : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1), "f"(c[0]), "f"(c[1]), "f"(c[2]), "f"(c[3]));
}
__device__ __forceinline__ void mma8c(float (&d)[4], uint32_t a0, uint32_t a1, uint32_t b0, const float (&c)[4]) {
  asm("mma.sync.aligned.m16n8k8.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5}, {%6}, {%7,%8,%9,%10};"
      : "=f"(d[0]), "=f"(d[1]), "=f"(d[2]), "=f"(d[3])
      : "r"(a0), "r"(a1), "r"(b0), "f"(c[0]), "f"(c[1]), "f"(c[2]), "f"(c[3]));
}
// D = A . B (C = 0): fresh outputs, no accumulator initialisation
__device__ __forceinline__ void mma16z(float (&d)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t b0, uint32_t b1) {
  asm("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%10,%10,%10,%10};"
      : "=f"(d[0]), "=f"(d[1]), "=f"(d[2]), "=f"(d[3])
      : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1), "f"(0.f));
}
__device__ __forceinline__ void mma8(float (&d)[4], uint32_t a0, uint32_t a1, uint32_t b0) {
  asm("mma.sync.aligned.m16n8k8.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5}, {%6}, {%0,%1,%2,%3};"
      : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
      : "r"(a0), "r"(a1), "r"(b0));
}
// (x, y) -> bf16x2 hi part (round to nearest) and bf16x2 lo part of the remainders: x = hi.x + lo.x to 16 bits
__device__ __forceinline__ void split_bf16x2(float x, float y, uint32_t& hi, uint32_t& lo) {
  hi = pack_bf16x2(x, y);
  const float hx = __uint_as_float(hi << 16), hy = __uint_as_float(hi & 0xffff0000u);
  lo = pack_bf16x2(x - hx, y - hy);
}

// the same split in fp16 (8-bit coefficient mode: q~ feeds an f16 MMA): 11 + 11 bits; clamped to the fp16 range so that an
// absurdly large q saturates the score instead of producing inf - inf
__device__ __forceinline__ void split_f16x2(float x, float y, uint32_t& hi, uint32_t& lo) {
  x = fminf(fmaxf(x, -65504.f), 65504.f); y = fminf(fmaxf(y, -65504.f), 65504.f);
  const __half2 h = __floats2half2_rn(x, y);
  const float2 hf = __half22float2(h);
  const __half2 l = __floats2half2_rn(x - hf.x, y - hf.y);
  hi = *reinterpret_cast<const uint32_t*>(&h);
  lo = *reinterpret_cast<const uint32_t*>(&l);
}

__device__ __forceinline__ Unit load_unit(const Unit* u) {
  const uint4 a = __ldg(reinterpret_cast<const uint4*>(u));
  const uint4 b = __ldg(reinterpret_cast<const uint4*>(u) + 1);
  Unit r;
  r.page_off = (int64_t)(((uint64_t)a.y << 32) | a.x);
  r.blk0 = (int32_t)a.z; r.nblk = (int32_t)a.w;
  r.ntok = (int32_t)b.x; r.cls = (int16_t)(b.y & 0xffff); r.b = (int16_t)(b.y >> 16);
  r.epart = (int32_t)b.z; r.rk = (int32_t)b.w;
  return r;
}

// geometry of the ring for a kernel instance (NKB = basis rank / 8 rounded up to even, D = head dim)
template <int NKB, int D>
struct Ring {
  static constexpr int SLOT_RAW = (NKB * 1024 > NKB * 512 + 20 * D) ? NKB * 1024 : NKB * 512 + 20 * D;
  static constexpr int SLOT1 = (SLOT_RAW + 127) & ~127;                 // bytes of the fattest sub-block
  static constexpr int NS = 2;  /* (3 stages of 9 KB measured 2-17 % slower: the per-stage overhead is ~100 instructions) */                                        // few, large stages: per-stage overhead is amortised
  static constexpr int SLOT = (kRingBytes / NS) / SLOT1 * SLOT1;        // a whole number of fattest sub-blocks
  static_assert(NS >= 2, "ring too small for this rank");
};

// Per-segment register state. Row r of the MMA M dimension: PAIR: (head r & 3, token tile parity (r >> 2) & 1), rows
// 8..15 = lo parts of rows 0..7; FULL: head r, rows 8..15 = lo parts. Lane (g, t) owns row g (and g + 8).
template <int NKB, int D>
struct State {
  float m;                 // reference of row g (log2 units), -inf = none yet
  float thr;               // -inf while unreferenced, kLazy afterwards
  float cq[4];             // C operand of the score MMAs: (-m, -m, 0, 0), (0, 0, 0, 0) while unreferenced; changes only on a rescale
  float l;                 // this lane's share of sum p of row g
  float acc[NKB][4];       // a[row g][8i + 2t + {0,1}] hi-part accumulators (0,1) and lo-part accumulators (2,3)
  float eacc[D / 16][4];   // TRANSPOSED e^T[channel 16grp + g (+8)][column 2t + {0,1}], column n <-> row n
};

// Query-side operands of a segment, already in MMA A-fragment order.
template <int NKB, int D, bool PAIR>
struct QRegs {
  // PAIR: qa[i] = {selA ? hi : 0, selA ? lo : 0, selA ? 0 : hi, selA ? 0 : lo}  (selA = lane's row is a tile-A row)
  // FULL: qa[i] = {hi, lo} of chunk i
  uint32_t qa[NKB][PAIR ? 4 : 2];
  // raw q (residual-K term) as ready-made A-operand quads (a0, a1, a2, a3) = (row g | row g+8) x (channels +0 | +8). Rows g+8 of these
  // MMAs are "don't care" rows for one of the two products that share a quad, so no register is spent on zeros and none is moved:
  // PAIR, group grp:      qr[grp]   = {selA ? q0 : 0, selA ? 0 : q0, selA ? q2 : 0, selA ? 0 : q2}: the tile-A product reads rows g,
  //                                   the tile-B product (same quad, tile B codes) reads rows g+8
  // FULL, groups 2p, 2p+1: qr[p]    = {q0(2p), q0(2p+1), q2(2p), q2(2p+1)}: group 2p reads rows g, group 2p+1 rows g+8
  uint32_t qr[PAIR ? D / 16 : D / 32][4];
  float qbias[D / 16];     // -136 * sum_{i in grp} q[head][i]: removes the offset of the biased codes
};

}  // namespace s3
}  // namespace dwkv
