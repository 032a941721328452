// dwkv_cache_ops.cu -- load / dump auxiliaries of the cache (the append/compress kernel, step a4, is dwkv_compress.cu):
//   scatter_raw_kernel  load pre-compressed token-ordered entries into the fragment-native pages
//   gather_kernel       token-ordered dump of stored entries (bit-exact checks of routing and int4 dequantisation)
//   stats_* kernels     router features of a probe step (per-token attention mass / spike), probe_error_kernel (Eq. 3)
#include <algorithm>
#include "dwkv_internal.h"
#include "dwkv_mma.cuh"

namespace dwkv {
namespace {
using dwkv::dev::coef8_exponent;
using dwkv::dev::coef8_code;

constexpr uint32_t kFull = 0xffffffffu;

// Reading A14: fp32 IEEE, round-to-nearest-even, no FMA contraction, no reciprocal.
//   s32 = amax / 7 ; s32 = min(s32, 65504) ; s = fp16_rn(s32) ; s == 0 -> 0 else clamp(rint(e / float(s)), -7, 7)
__device__ __forceinline__ int quant_code(float e, float amax, __half* s_out) {
  float s32 = __fdiv_rn(amax, 7.0f);
  s32 = fminf(s32, 65504.0f);
  const __half s = __float2half_rn(s32);
  const float sf = __half2float(s);
  *s_out = s;
  if (sf == 0.f) return 0;
  float r = rintf(__fdiv_rn(e, sf));
  r = fminf(fmaxf(r, -7.f), 7.f);
  return (int)r;
}

__device__ __forceinline__ float group16_amax(float a) {   // max over the 16 lanes of a half-warp
  a = fmaxf(a, __shfl_xor_sync(kFull, a, 8));
  a = fmaxf(a, __shfl_xor_sync(kFull, a, 4));
  a = fmaxf(a, __shfl_xor_sync(kFull, a, 2));
  a = fmaxf(a, __shfl_xor_sync(kFull, a, 1));
  return a;
}

struct BlockPtr {
  uint8_t* blk;     // start of the sub-block that holds the token
  int slot;         // slot inside the sub-block
  ClassLayout cl;
  int rk;
};

__device__ __forceinline__ BlockPtr block_ptr(const uint8_t* arena, const CacheGeom& g, const TokDst& td, int lh) {
  BlockPtr b;
  b.rk = g.tier_rank[td.cls >> 1];
  b.cl = make_class_layout(b.rk, td.cls & 1, g.d, g.i8);
  b.blk = const_cast<uint8_t*>(arena) + td.page_off + (size_t)lh * kPageLhBytes + (size_t)td.blk * b.cl.block_bytes +
          sub_off(b.cl, td.slot);
  b.slot = sub_slot(b.cl, td.slot);
  return b;
}

__device__ __forceinline__ float warp_max(float a) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) a = fmaxf(a, __shfl_xor_sync(kFull, a, o));
  return a;
}
// store one token's coefficient of column col (stored byte = code + 128) and, from the first column of a 32-column block, the
// block's exponent byte (e + 127)
__device__ __forceinline__ void store_coef8(const BlockPtr& bp, int z, int col, int code, int e) {
  uint8_t* base = bp.blk + (z ? off_coefV(bp.cl) : off_coefK(bp.cl));
  base[z ? vcoef8_elem_off(bp.slot, col, bp.cl.tb) : kcoef8_elem_off(bp.slot, col, bp.cl.tb)] = (uint8_t)(code + 128);
  if ((col & 31) == 0) base[coef8_exp_off(bp.slot, bp.cl.nk, bp.cl.tb, col >> 5)] = (uint8_t)(e + 127);
}
__device__ __forceinline__ float load_coef8(const BlockPtr& bp, int z, int col) {
  const uint8_t* base = bp.blk + (z ? off_coefV(bp.cl) : off_coefK(bp.cl));
  const int u = base[z ? vcoef8_elem_off(bp.slot, col, bp.cl.tb) : kcoef8_elem_off(bp.slot, col, bp.cl.tb)];
  const uint32_t eb = base[coef8_exp_off(bp.slot, bp.cl.nk, bp.cl.tb, col >> 5)];
  return (float)(u - 128) * __uint_as_float(eb << 23);
}

__device__ __forceinline__ void store_code(uint8_t* region, int word_off, int bit, int code) {
  atomicOr(reinterpret_cast<unsigned int*>(region + word_off), (unsigned int)((code + 8) & 15) << bit);
}

__device__ __forceinline__ int load_code(const uint8_t* region, int word_off, int bit) {
  const unsigned int w = *reinterpret_cast<const unsigned int*>(region + word_off);
  return (int)((w >> bit) & 15u) - 8;
}

// ---------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) scatter_raw_kernel(const uint8_t* arena, CacheGeom g, const TokDst* dst,
                                                          const __nv_bfloat16* coefK, const __nv_bfloat16* coefV,
                                                          const float* residK, const float* residV,
                                                          const uint8_t* codeK, const uint8_t* codeV,
                                                          const __half* scaleK, const __half* scaleV) {
  const int tok = blockIdx.x, lh = blockIdx.y, LH = g.L * g.H, tid = threadIdx.x;
  const TokDst td = dst[tok];
  const BlockPtr bp = block_ptr(arena, g, td, lh);
  const size_t row = (size_t)tok * LH + lh;
  if (g.i8) {                 // quantise the given coefficients: warp b holds the 32-column block b of the vector (rank <= 64)
    if (tid < 64 && (tid & ~31) < bp.rk) {
      for (int z = 0; z < 2; ++z) {
        const float cf = tid < bp.rk ? __bfloat162float((z ? coefV : coefK)[row * g.r + tid]) : 0.f;
        const int e = coef8_exponent(warp_max(fabsf(cf)));
        if (tid < bp.rk) store_coef8(bp, z, tid, coef8_code(cf, e), e);
      }
    }
  } else if (tid < bp.rk) {
    *reinterpret_cast<__nv_bfloat16*>(bp.blk + off_coefK(bp.cl) + kcoef_elem_off(bp.slot, tid, bp.cl.tb)) = coefK[row * g.r + tid];
    *reinterpret_cast<__nv_bfloat16*>(bp.blk + off_coefV(bp.cl) + vcoef_elem_off(bp.slot, tid, bp.cl.tb)) = coefV[row * g.r + tid];
  }
  if (td.ridx < 0) return;
  const size_t rrow = (size_t)td.ridx * LH + lh;
  const int d = g.d, ng = d / 16;
  if (tid < d) {
    const int ch = tid, grp = ch >> 4;
    for (int z = 0; z < 2; ++z) {
      const float* resid = z ? residV : residK;
      const uint8_t* codes = z ? codeV : codeK;
      const __half* scales = z ? scaleV : scaleK;
      int code;
      __half s;
      if (resid) {
        const float e = resid[rrow * d + ch];
        const float amax = group16_amax(fabsf(e));
        code = quant_code(e, amax, &s);
      } else {
        const uint8_t byte = codes[rrow * (d / 2) + (ch >> 1)];
        const int nib = (ch & 1) ? (byte >> 4) : (byte & 15);
        code = (nib < 8) ? nib : nib - 16;
        s = scales[rrow * ng + grp];
      }
      int wo, bit;
      if (z == 0) kcode_nibble(bp.slot, ch, d, &wo, &bit); else vcode_nibble(bp.slot, ch, d, &wo, &bit);
      store_code(bp.blk + (z ? off_codeV(bp.cl) : off_codeK(bp.cl)), wo, bit, code);
      if ((ch & 15) == 0)
        *reinterpret_cast<__half*>(bp.blk + (z ? off_scaleV(bp.cl) : off_scaleK(bp.cl)) + scale_elem_off(bp.slot, grp, d)) = s;
    }
  }
}

// ---------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) gather_kernel(const uint8_t* arena, CacheGeom g, const TokDst* dst, DumpPtrs o) {
  const int tok = blockIdx.x, lh = blockIdx.y, LH = g.L * g.H, tid = threadIdx.x;
  const TokDst td = dst[tok];
  const BlockPtr bp = block_ptr(arena, g, td, lh);
  const size_t row = (size_t)tok * LH + lh;
  const int d = g.d, ng = d / 16;
  if (g.i8 && tid < g.r) {     // code * 2^e has <= 7 significant bits: exactly a bf16 value (g.r <= 64 < blockDim)
    const __nv_bfloat16 zero = __float2bfloat16_rn(0.f);
    if (o.coefK) o.coefK[row * g.r + tid] = tid < bp.rk ? __float2bfloat16_rn(load_coef8(bp, 0, tid)) : zero;
    if (o.coefV) o.coefV[row * g.r + tid] = tid < bp.rk ? __float2bfloat16_rn(load_coef8(bp, 1, tid)) : zero;
  } else if (tid < g.r) {
    const __nv_bfloat16 zero = __float2bfloat16_rn(0.f);
    if (o.coefK)
      o.coefK[row * g.r + tid] = tid < bp.rk ? *reinterpret_cast<const __nv_bfloat16*>(bp.blk + off_coefK(bp.cl) + kcoef_elem_off(bp.slot, tid, bp.cl.tb)) : zero;
    if (o.coefV)
      o.coefV[row * g.r + tid] = tid < bp.rk ? *reinterpret_cast<const __nv_bfloat16*>(bp.blk + off_coefV(bp.cl) + vcoef_elem_off(bp.slot, tid, bp.cl.tb)) : zero;
  }
  const bool fl = (td.cls & 1) != 0;
  for (int z = 0; z < 2; ++z) {
    uint8_t* codes = z ? o.codeV : o.codeK;
    __half* scales = z ? o.scaleV : o.scaleK;
    float* deq = z ? o.deqV : o.deqK;
    const uint8_t* creg = bp.blk + (z ? off_codeV(bp.cl) : off_codeK(bp.cl));
    const uint8_t* sreg = bp.blk + (z ? off_scaleV(bp.cl) : off_scaleK(bp.cl));
    if (tid < d) {
      int code = 0;
      __half s = __float2half_rn(0.f);
      if (fl) {
        int wo, bit;
        if (z == 0) kcode_nibble(bp.slot, tid, d, &wo, &bit); else vcode_nibble(bp.slot, tid, d, &wo, &bit);
        code = load_code(creg, wo, bit);
        s = *reinterpret_cast<const __half*>(sreg + scale_elem_off(bp.slot, tid >> 4, d));
      }
      if (deq) deq[row * d + tid] = (float)code * __half2float(s);
      if (scales && (tid & 15) == 0) scales[row * ng + (tid >> 4)] = s;
      const int other = __shfl_down_sync(kFull, code, 1);
      if (codes && (tid & 1) == 0) codes[row * (d / 2) + (tid >> 1)] = (uint8_t)((code & 15) | ((other & 15) << 4));
    }
  }
}

__global__ void gate_check_kernel(const __nv_bfloat16* g, int64_t n, int* bad) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) {
    const float v = __bfloat162float(g[i]);
    if (!(fabsf(v) > 0.f) || isinf(v) || isnan(v)) atomicOr(bad, 1);
  }
}

}  // namespace

int launch_scatter_raw(const uint8_t* arena, const CacheGeom& g, const TokDst* dst, int n, const __nv_bfloat16* coefK,
                       const __nv_bfloat16* coefV, const float* residK, const float* residV, const uint8_t* codeK,
                       const uint8_t* codeV, const __half* scaleK, const __half* scaleV, cudaStream_t s) {
  if (n <= 0) return 0;
  dim3 grid(n, g.L * g.H);
  scatter_raw_kernel<<<grid, 128, 0, s>>>(arena, g, dst, coefK, coefV, residK, residV, codeK, codeV, scaleK, scaleV);
  return 1;
}

int launch_gather(const uint8_t* arena, const CacheGeom& g, const TokDst* dst, int n, const DumpPtrs& o, cudaStream_t s) {
  if (n <= 0) return 0;
  dim3 grid(n, g.L * g.H);
  gather_kernel<<<grid, 128, 0, s>>>(arena, g, dst, o);
  return 1;
}

int launch_gate_check(const __nv_bfloat16* g, int64_t n, int* bad_flag, cudaStream_t s) {
  gate_check_kernel<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(g, n, bad_flag);
  return 1;
}

// Eq. (3) of the paper: e[h] = ||ref - cmp||_2 / (||ref||_2 + eps) over the G query heads of kv head h, the
// n_q probed positions and all channels. One CTA per kv head; ref, cmp: fp32 [n_q, H*G, d].
namespace {
__global__ void __launch_bounds__(256) probe_error_kernel(const float* ref, const float* cmp, float* e, int n_q, int H, int G, int d, float eps) {
  __shared__ float sn[8], sd[8];
  const int h = blockIdx.x, tid = threadIdx.x, per_q = G * d;
  float num = 0.f, den = 0.f;
  for (int i = tid; i < n_q * per_q; i += 256) {
    const int qi = i / per_q, r = i - qi * per_q;
    const size_t off = ((size_t)qi * H + h) * per_q + r;
    const float a = ref[off], b = cmp[off];
    num = fmaf(a - b, a - b, num);
    den = fmaf(a, a, den);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) { num += __shfl_xor_sync(0xffffffffu, num, o); den += __shfl_xor_sync(0xffffffffu, den, o); }
  if ((tid & 31) == 0) { sn[tid >> 5] = num; sd[tid >> 5] = den; }
  __syncthreads();
  if (tid == 0) {
    num = 0.f; den = 0.f;
    for (int w = 0; w < 8; ++w) { num += sn[w]; den += sd[w]; }
    e[h] = sqrtf(num) / (sqrtf(den) + eps);
  }
}

// ---------------------------------------------------------------------------------------------------------------
// Router features from the decode path (reading A28): per-token softmax probabilities of one (sequence,
// layer, query vector) over the compressed cache, summed / maximised over the query heads. A probe-path kernel set (runs every p
// decode steps on one layer), written plainly in fp32: scores with the decode kernel's algebra (q~ = cscale * BK (gK * q) once per
// block; s = q~ . cK + cscale * sum_g scale_g * (q_g . code_g); nothing is reconstructed), then log-sum-exp per query head, then
// mass[t] += sum_hq p, spike[t] = max(spike[t], max_hq p).
constexpr int kStatsTok = 128;      // tokens (threads) per block of the score kernel

__global__ void __launch_bounds__(kStatsTok) stats_scores_kernel(const uint8_t* arena, CacheGeom g, const TokDst* dst, int T, int layer,
                                                               const __nv_bfloat16* q, const __nv_bfloat16* BK, const __nv_bfloat16* gK,
                                                               float cscale, float* scores /* [T][Hq] log2 units */) {
  extern __shared__ float sh[];
  const int h = blockIdx.y, tid = threadIdx.x, d = g.d, r = g.r, G = g.G;
  float* qt = sh;                 // [G][r]   q~ (log2 units)
  float* qr = sh + G * r;         // [G][d]   cscale * q (residual term)
  float* qg = qr + G * d;         // [G][d]   gK * q
  const __nv_bfloat16* qh = q + (size_t)h * G * d;
  const __nv_bfloat16* gk = gK + ((size_t)layer * g.H + h) * d;
  const __nv_bfloat16* B = BK + ((size_t)(layer / g.w) * g.H + h) * (size_t)r * d;
  for (int i = tid; i < G * d; i += kStatsTok) {
    const float x = __bfloat162float(qh[i]);
    qr[i] = cscale * x;
    qg[i] = x * __bfloat162float(gk[i % d]);
  }
  __syncthreads();
  for (int i = tid; i < G * r; i += kStatsTok) {
    const int gq = i / r, j = i - gq * r;
    float acc = 0.f;
    for (int ch = 0; ch < d; ++ch) acc = fmaf(__bfloat162float(B[(size_t)j * d + ch]), qg[gq * d + ch], acc);
    qt[i] = cscale * acc;
  }
  __syncthreads();
  const int t = blockIdx.x * kStatsTok + tid;
  if (t >= T) return;
  const TokDst td = dst[t];
  const BlockPtr bp = block_ptr(arena, g, td, layer * g.H + h);
  float sc[8];
#pragma unroll
  for (int gq = 0; gq < 8; ++gq) sc[gq] = 0.f;
  for (int j = 0; j < bp.rk; ++j) {
    const float c = g.i8 ? load_coef8(bp, 0, j)
                         : __bfloat162float(*reinterpret_cast<const __nv_bfloat16*>(bp.blk + off_coefK(bp.cl) + kcoef_elem_off(bp.slot, j, bp.cl.tb)));
#pragma unroll
    for (int gq = 0; gq < 8; ++gq)
      if (gq < G) sc[gq] = fmaf(qt[gq * r + j], c, sc[gq]);
  }
  if (td.cls & 1) {
    const uint8_t* creg = bp.blk + off_codeK(bp.cl);
    const uint8_t* sreg = bp.blk + off_scaleK(bp.cl);
    for (int grp = 0; grp < d / 16; ++grp) {
      const float s = __half2float(*reinterpret_cast<const __half*>(sreg + scale_elem_off(bp.slot, grp, d)));
      float dot[8];
#pragma unroll
      for (int gq = 0; gq < 8; ++gq) dot[gq] = 0.f;
      for (int i = 0; i < 16; ++i) {
        int wo, bit;
        kcode_nibble(bp.slot, 16 * grp + i, d, &wo, &bit);
        const float code = (float)load_code(creg, wo, bit);
#pragma unroll
        for (int gq = 0; gq < 8; ++gq)
          if (gq < G) dot[gq] = fmaf(qr[gq * d + 16 * grp + i], code, dot[gq]);
      }
#pragma unroll
      for (int gq = 0; gq < 8; ++gq)
        if (gq < G) sc[gq] = fmaf(s, dot[gq], sc[gq]);
    }
  }
#pragma unroll
  for (int gq = 0; gq < 8; ++gq)
    if (gq < G) scores[(size_t)t * (g.H * G) + h * G + gq] = sc[gq];
}

// one block per query head: lse[hq] = m + log2(sum_t 2^(s - m))
__global__ void __launch_bounds__(256) stats_lse_kernel(const float* scores, int T, int Hq, float* lse) {
  __shared__ float red[8];
  const int hq = blockIdx.x, tid = threadIdx.x;
  float m = -INFINITY;
  for (int t = tid; t < T; t += 256) m = fmaxf(m, scores[(size_t)t * Hq + hq]);
  m = warp_max(m);
  if ((tid & 31) == 0) red[tid >> 5] = m;
  __syncthreads();
  m = red[0];
  for (int w = 1; w < 8; ++w) m = fmaxf(m, red[w]);
  __syncthreads();
  float sum = 0.f;
  for (int t = tid; t < T; t += 256) sum += exp2f(scores[(size_t)t * Hq + hq] - m);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(kFull, sum, o);
  if ((tid & 31) == 0) red[tid >> 5] = sum;
  __syncthreads();
  if (tid == 0) {
    sum = 0.f;
    for (int w = 0; w < 8; ++w) sum += red[w];
    lse[hq] = m + log2f(sum);
  }
}

__global__ void __launch_bounds__(256) stats_emit_kernel(const float* scores, const float* lse, int T, int Hq, float* mass, float* spike) {
  const int t = blockIdx.x * 256 + threadIdx.x;
  if (t >= T) return;
  float sum = 0.f, mx = 0.f;
  for (int hq = 0; hq < Hq; ++hq) {
    const float p = exp2f(scores[(size_t)t * Hq + hq] - lse[hq]);
    sum += p;
    mx = fmaxf(mx, p);
  }
  mass[t] += sum;
  spike[t] = fmaxf(spike[t], mx);
}
}  // namespace

size_t token_stats_scratch_bytes(const CacheGeom& g, int64_t T) { return ((size_t)T * g.H * g.G + (size_t)g.H * g.G) * sizeof(float); }

int launch_token_stats(const uint8_t* arena, const CacheGeom& g, const TokDst* dst, int T, int layer, const __nv_bfloat16* q,
                       const __nv_bfloat16* BK, const __nv_bfloat16* gK, float cscale, float* scratch, float* mass, float* spike,
                       cudaStream_t s) {
  const int Hq = g.H * g.G;
  float* scores = scratch;
  float* lse = scratch + (size_t)T * Hq;
  const size_t smem = (size_t)(g.G * g.r + 2 * g.G * g.d) * sizeof(float);
  stats_scores_kernel<<<dim3((T + kStatsTok - 1) / kStatsTok, g.H), kStatsTok, smem, s>>>(arena, g, dst, T, layer, q, BK, gK, cscale, scores);
  stats_lse_kernel<<<Hq, 256, 0, s>>>(scores, T, Hq, lse);
  stats_emit_kernel<<<(T + 255) / 256, 256, 0, s>>>(scores, lse, T, Hq, mass, spike);
  return 3;
}

int launch_probe_error(const float* ref, const float* cmp, float* e, int n_q, int H, int G, int d, float eps, cudaStream_t s) {
  probe_error_kernel<<<H, 256, 0, s>>>(ref, cmp, e, n_q, H, G, d, eps);
  return 1;
}

}  // namespace dwkv
