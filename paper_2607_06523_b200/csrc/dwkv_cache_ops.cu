// dwkv_cache_ops.cu -- load / dump auxiliaries of the cache (the append/compress kernel, step a4, is dwkv_compress.cu):
//   scatter_raw_kernel  load pre-compressed token-ordered entries into the fragment-native pages
//   gather_kernel       token-ordered dump of stored entries (bit-exact checks of routing and int4 dequantisation)
#include "dwkv_internal.h"

namespace dwkv {
namespace {

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
  b.cl = make_class_layout(b.rk, td.cls & 1, g.d);
  b.blk = const_cast<uint8_t*>(arena) + td.page_off + (size_t)lh * kPageLhBytes + (size_t)td.blk * b.cl.block_bytes +
          sub_off(b.cl, td.slot);
  b.slot = sub_slot(b.cl, td.slot);
  return b;
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
  if (tid < bp.rk) {
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
  if (tid < g.r) {
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
}  // namespace

int launch_probe_error(const float* ref, const float* cmp, float* e, int n_q, int H, int G, int d, float eps, cudaStream_t s) {
  probe_error_kernel<<<H, 256, 0, s>>>(ref, cmp, e, n_q, H, G, d, eps);
  return 1;
}

}  // namespace dwkv
