// dwkv_layout.cuh -- the packed, tier-segregated cache layout.
//
// The cache is a pool of fixed-size pages. A page belongs to one (sequence, class) where class = 2*tier + flag,
// and holds, for EVERY (layer, kv head), PAGE_LH_BYTES of that class's token records:
//     page[(l*H_kv + h) * PAGE_LH_BYTES + block * block_bytes(class) + ...]
// Tokens are stored in blocks of 32 slots. A block is a sequence of independent "sub-blocks": ONE sub-block of 32 slots
// for unflagged classes, TWO sub-blocks of 16 slots for flagged classes (so that a streaming stage of the scan stays
// <= 4.5 KB). Inside a sub-block every field is laid out in the register order of the mma.sync.m16n8k16 fragments that
// consume it ("fragment-native"): a warp-wide vector load brings exactly the operand registers of the tensor-core
// instruction and every load is a contiguous run.
//
//   lane = 4*g + t  (g = lane>>2, t = lane&3), tile j = 8 consecutive slots, TB = tiles per sub-block (4 or 2),
//   chunk i = 8 rank columns, nk = rank/8, d = head dim, ng = d/16 groups
//   [K coef]  nk vectors of 128*TB B.  vector i, lane (g,t), word j : ( cK[slot 8j+g][8i+2t], cK[slot 8j+g][8i+2t+1] )
//             = B-fragment register (k = rank cols, n = token) of the score MMA  S = q~ . cK^T
//   [V coef]  nk vectors of 128*TB B.  vector i, lane (g,t), word j : ( cV[slot 8j+2t][8i+g], cV[slot 8j+2t+1][8i+g] )
//             = B-fragment register (k = tokens, n = rank col) of the value MMA  a += P . cV
//   flagged classes only (TB = 2):
//   [K code]  tile j, lane (g,t): d/8 bytes = d/32 words; word x, nibble pair s (bits 4s.. and 16+4s..) is register
//             q = 4x+s = (group q>>1, half b = q&1): offset-binary codes (code+8) of slot 8j+g, channels
//             16*grp + 8*b + 2t (low half-word) and +1 (high half-word)
//   [K scale] word (j, t, grp) = fp16x2 ( scale[slot 8j+2t][grp], scale[slot 8j+2t+1][grp] )
//   [V code]  lane (g,t): d/4 bytes = d/16 words; word grp, nibble pair a (bits 4a.. and 16+4a..) is A-fragment register a
//             of the transposed value MMA e^T += codeV^T . (P*scaleV): offset-binary codes of slots 8*(a>>1)+2t (low
//             half-word) and +1 (high), channel 16*grp + 8*(a&1) + g
//   [V scale] same arrangement as [K scale]
//
// 8-bit coefficient mode ("8-bit blockwise quantized"; reading A27): a block
// is 32 consecutive rank columns of a token's coefficient vector (ranks <= 32: one block, ranks 48 / 64: two): the same fragment
// order with one BYTE per coefficient (offset-binary code + 128) and, behind the nk code vectors of each of K and V, one
// exponent byte (e + 127) per slot and block ([K exp] of block 0, then of block 1):
//   [K coef8] nk vectors of 64*TB B.  vector i, lane (g,t), half-word j : ( uK[slot 8j+g][8i+2t], uK[slot 8j+g][8i+2t+1] )
//   [K exp]   8*TB B.                 byte (t, j, hi) = exponent byte of slot 8j + 2t + hi   (the C-fragment columns of lane t)
//   [V coef8] nk vectors of 64*TB B.  vector i, lane (g,t), half-word j : ( uV[slot 8j+2t][8i+g], uV[slot 8j+2t+1][8i+g] )
//   [V exp]   as [K exp]
#pragma once
#include <stdint.h>

#if defined(__CUDACC__)
#define DWKV_HD __host__ __device__ __forceinline__
#else
#define DWKV_HD inline
#endif

namespace dwkv {

constexpr int kBlockTok = 32;              // token slots per block
constexpr int kPageLhBytes = 64 * 1024;    // bytes per (layer, kv head) per page
constexpr int kMaxNk = 8;                  // basis rank <= 64
constexpr int kMaxClasses = 8;             // 2 * DWKV_MAX_TIERS

struct ClassLayout {
  int nk;            // rank / 8
  int resid;         // 0 / 1
  int i8;            // 8-bit coefficient mode
  int tb;            // tiles (of 8 slots) per sub-block: 4 (unflagged) or 2 (flagged)
  int sub_tok;       // slots per sub-block = 8 * tb
  int coef_bytes;    // nk * 128 * tb  (per K or V, per sub-block); 8-bit mode: nk * 64 * tb codes + 8 * tb exponent bytes per 32-column block
  int code_bytes;    // per K or V, per sub-block: tb * 4 * d, 0 if !resid
  int scale_bytes;   // tb * d
  int sub_bytes;     // 2*coef + resid * 2*(code + scale)
  int block_bytes;   // (32 / sub_tok) * sub_bytes
  int blocks_per_page;
  int tokens_per_page;
};

DWKV_HD ClassLayout make_class_layout(int rank, int resid, int d, int i8 = 0) {
  ClassLayout c;
  c.nk = rank / 8;
  c.resid = resid;
  c.i8 = i8;
  c.tb = resid ? 2 : 4;
  c.sub_tok = 8 * c.tb;
  c.coef_bytes = i8 ? c.nk * 64 * c.tb + ((rank + 31) / 32) * 8 * c.tb : c.nk * 128 * c.tb;
  c.code_bytes = resid ? c.tb * 4 * d : 0;
  c.scale_bytes = resid ? c.tb * d : 0;
  c.sub_bytes = 2 * c.coef_bytes + 2 * (c.code_bytes + c.scale_bytes);
  c.block_bytes = (kBlockTok / c.sub_tok) * c.sub_bytes;
  c.blocks_per_page = kPageLhBytes / c.block_bytes;
  c.tokens_per_page = c.blocks_per_page * kBlockTok;
  return c;
}

// byte offsets of the fields inside a sub-block ---------------------------------------------------------------------
DWKV_HD int off_coefK(const ClassLayout&) { return 0; }
DWKV_HD int off_coefV(const ClassLayout& c) { return c.coef_bytes; }
DWKV_HD int off_codeK(const ClassLayout& c) { return 2 * c.coef_bytes; }
DWKV_HD int off_scaleK(const ClassLayout& c) { return 2 * c.coef_bytes + c.code_bytes; }
DWKV_HD int off_codeV(const ClassLayout& c) { return 2 * c.coef_bytes + c.code_bytes + c.scale_bytes; }
DWKV_HD int off_scaleV(const ClassLayout& c) { return 2 * c.coef_bytes + 2 * c.code_bytes + c.scale_bytes; }
// byte offset of the sub-block holding slot s (0..31) of a block, and the slot index inside it
DWKV_HD int sub_off(const ClassLayout& c, int s) { return (s / c.sub_tok) * c.sub_bytes; }
DWKV_HD int sub_slot(const ClassLayout& c, int s) { return s % c.sub_tok; }

// element addressing inside a sub-block (slot s in 0..sub_tok-1, rank column col, channel ch) -----------------------
DWKV_HD int kcoef_elem_off(int s, int col, int tb) {     // byte offset of the bf16 element inside [K coef]
  const int j = s >> 3, g = s & 7, i = col >> 3, t = (col & 7) >> 1, hi = col & 1;
  return i * 128 * tb + (4 * g + t) * 4 * tb + j * 4 + hi * 2;
}
DWKV_HD int vcoef_elem_off(int s, int col, int tb) {     // byte offset of the bf16 element inside [V coef]
  const int j = s >> 3, p = s & 7, t = p >> 1, hi = p & 1, i = col >> 3, g = col & 7;
  return i * 128 * tb + (4 * g + t) * 4 * tb + j * 4 + hi * 2;
}
// 8-bit coefficient mode: byte offsets inside [K coef8] / [V coef8] and of the exponent byte behind the nk code vectors
DWKV_HD int kcoef8_elem_off(int s, int col, int tb) {
  const int j = s >> 3, g = s & 7, i = col >> 3, t = (col & 7) >> 1, hi = col & 1;
  return i * 64 * tb + (4 * g + t) * 2 * tb + j * 2 + hi;
}
DWKV_HD int vcoef8_elem_off(int s, int col, int tb) {
  const int j = s >> 3, p = s & 7, t = p >> 1, hi = p & 1, i = col >> 3, g = col & 7;
  return i * 64 * tb + (4 * g + t) * 2 * tb + j * 2 + hi;
}
DWKV_HD int coef8_exp_off(int s, int nk, int tb, int blk = 0) {     // blk = rank column / 32
  const int j = s >> 3, p = s & 7, t = p >> 1, hi = p & 1;
  return nk * 64 * tb + blk * 8 * tb + t * 2 * tb + j * 2 + hi;
}
DWKV_HD void kcode_nibble(int s, int ch, int d, int* word_off, int* bit) {   // inside [K code] (s in 0..15)
  const int j = s >> 3, g = s & 7, grp = ch >> 4, wi = ch & 15, b = wi >> 3, t = (wi & 7) >> 1, hi = wi & 1;
  const int q = 2 * grp + b;
  *word_off = j * 4 * d + (4 * g + t) * (d / 8) + (q >> 2) * 4;
  *bit = 4 * (q & 3) + 16 * hi;
}
DWKV_HD void vcode_nibble(int s, int ch, int d, int* word_off, int* bit) {   // inside [V code] (s in 0..15)
  const int tile = (s >> 3) & 1, p = s & 7, t = p >> 1, hi = p & 1;
  const int grp = ch >> 4, wi = ch & 15, g = wi & 7, upper = wi >> 3;
  const int a = upper + 2 * tile;        // A-fragment register index of the transposed value MMA
  *word_off = (4 * g + t) * (d / 4) + grp * 4;
  *bit = 4 * a + 16 * hi;
}
DWKV_HD int scale_elem_off(int s, int grp, int d) {   // byte offset of the fp16 element inside [K scale] / [V scale]
  const int j = s >> 3, p = s & 7, t = p >> 1, hi = p & 1, ng = d / 16;
  return j * d + t * (ng * 4) + grp * 4 + hi * 2;
}

}  // namespace dwkv
