// dwkv_combine3.cu -- a3: split-combine + back-projection, and the dispatcher of the fused
// decode kernel instances. One CTA per segment (sequence b, layer, kv head): log-sum-exp merge of the few warp partials
// (m, l, a[r], e[d]) the scan left for the segment, then  o = ( gV * (BV^T a) + e ) / l  for the G query heads.
#include "dwkv_internal.h"
#include "dwkv_mma.cuh"

namespace dwkv {

bool launch_scan3_d64_p0(const Scan3Params& p, int n_sms, cudaStream_t s);
bool launch_scan3_d64_p1(const Scan3Params& p, int n_sms, cudaStream_t s);
bool launch_scan3_d128_p0(const Scan3Params& p, int n_sms, cudaStream_t s);
bool launch_scan3_d128_p1(const Scan3Params& p, int n_sms, cudaStream_t s);

namespace {
using namespace dwkv::dev;

// One warp merges the partials of one (segment, query head) and writes o[head, :]. Lanes run over partials for the
// (m, l) pass, over rank columns for a*, over channels (D / 32 each) for e* and the back-projection.
template <int D>
__device__ __forceinline__ void combine_head(const Combine3Params& p, const int seg, const int gq, const int lane) {
  constexpr int CPL = D / 32;                       // channels per lane
  const int b = seg / p.LH, lh = seg - b * p.LH;
  const int layer = p.layer0 + lh / p.H, h = lh % p.H;
  const int G = p.G, r = p.r, PR = 2 + p.r + D;
  const int P0 = __ldg(p.pstart + seg), n = __ldg(p.pstart + seg + 1) - P0;
  const float* part = p.part + ((size_t)P0 * G + gq) * PR;       // partial k of this head: part + k * G * PR
  const size_t stride = (size_t)G * PR;
  // basis rows and gate of this lane's channels: independent of the partials, issued first
  const __nv_bfloat16* BV = p.BV + ((size_t)(layer / p.w) * p.H + h) * (size_t)r * D + lane * CPL;
  const __nv_bfloat16* gVp = p.gV + ((size_t)layer * p.H + h) * D + lane * CPL;
  float mstar = -INFINITY;
  for (int k = lane; k < n; k += 32) mstar = fmaxf(mstar, part[k * stride]);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) mstar = fmaxf(mstar, __shfl_xor_sync(kFull, mstar, o));
  float lstar = 0.f, a0 = 0.f, a1 = 0.f, e[CPL];
#pragma unroll
  for (int c = 0; c < CPL; ++c) e[c] = 0.f;
  for (int k0 = 0; k0 < n; k0 += 32) {
    const int kk = k0 + lane;
    float wk = 0.f;
    if (kk < n) {
      const float2 ml = *reinterpret_cast<const float2*>(part + kk * stride);
      wk = (ml.x == -INFINITY) ? 0.f : ex2(ml.x - mstar);
      lstar = fmaf(wk, ml.y, lstar);
    }
    const int nc = min(32, n - k0);
#pragma unroll 4
    for (int k = 0; k < nc; ++k) {
      const float w = __shfl_sync(kFull, wk, k);
      const float* rec = part + (size_t)(k0 + k) * stride + 2;
      if (lane < r) a0 = fmaf(w, rec[lane], a0);
      if (lane + 32 < r) a1 = fmaf(w, rec[lane + 32], a1);
      if constexpr (CPL == 4) {
        const float2 v = *reinterpret_cast<const float2*>(rec + r + lane * 4);       // records are 8-byte aligned only
        const float2 u = *reinterpret_cast<const float2*>(rec + r + lane * 4 + 2);
        e[0] = fmaf(w, v.x, e[0]); e[1] = fmaf(w, v.y, e[1]); e[2] = fmaf(w, u.x, e[2]); e[3] = fmaf(w, u.y, e[3]);
      } else {
        const float2 v = *reinterpret_cast<const float2*>(rec + r + lane * 2);
        e[0] = fmaf(w, v.x, e[0]); e[1] = fmaf(w, v.y, e[1]);
      }
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) lstar += __shfl_xor_sync(kFull, lstar, o);
  float acc[CPL];
#pragma unroll
  for (int c = 0; c < CPL; ++c) acc[c] = 0.f;
#pragma unroll 8
  for (int j = 0; j < r; ++j) {
    const float aj = __shfl_sync(kFull, j < 32 ? a0 : a1, j & 31);
    if constexpr (CPL == 4) {
      const uint2 bw = __ldg(reinterpret_cast<const uint2*>(BV + (size_t)j * D));
      acc[0] = fmaf(aj, __uint_as_float(bw.x << 16), acc[0]); acc[1] = fmaf(aj, __uint_as_float(bw.x & 0xffff0000u), acc[1]);
      acc[2] = fmaf(aj, __uint_as_float(bw.y << 16), acc[2]); acc[3] = fmaf(aj, __uint_as_float(bw.y & 0xffff0000u), acc[3]);
    } else {
      const uint32_t bw = __ldg(reinterpret_cast<const uint32_t*>(BV + (size_t)j * D));
      acc[0] = fmaf(aj, __uint_as_float(bw << 16), acc[0]); acc[1] = fmaf(aj, __uint_as_float(bw & 0xffff0000u), acc[1]);
    }
  }
  const float inv = 1.f / lstar;
  float* out = p.out + (((size_t)b * p.Lq + (p.Lq == 1 ? 0 : layer)) * (size_t)(p.H * G) + (size_t)h * G + gq) * D + lane * CPL;
  if constexpr (CPL == 4) {
    const uint2 gw = __ldg(reinterpret_cast<const uint2*>(gVp));
    float4 o;
    o.x = (__uint_as_float(gw.x << 16) * acc[0] + e[0]) * inv; o.y = (__uint_as_float(gw.x & 0xffff0000u) * acc[1] + e[1]) * inv;
    o.z = (__uint_as_float(gw.y << 16) * acc[2] + e[2]) * inv; o.w = (__uint_as_float(gw.y & 0xffff0000u) * acc[3] + e[3]) * inv;
    *reinterpret_cast<float4*>(out) = o;
  } else {
    const uint32_t gw = __ldg(reinterpret_cast<const uint32_t*>(gVp));
    float2 o;
    o.x = (__uint_as_float(gw << 16) * acc[0] + e[0]) * inv; o.y = (__uint_as_float(gw & 0xffff0000u) * acc[1] + e[1]) * inv;
    *reinterpret_cast<float2*>(out) = o;
  }
}

// grid = segments, 4 warps per CTA: warp w merges heads w, w + 4
template <int D>
__global__ void __launch_bounds__(128) combine3_kernel(const Combine3Params p) {
  const int seg = blockIdx.x, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int gq = warp; gq < p.G; gq += 4) combine_head<D>(p, seg, gq, lane);
}

}  // namespace

int scan3_num_slices(int n_sms) { return n_sms * 8; }

int launch_scan3(const Scan3Params& p, int n_sms, cudaStream_t s) {
  const bool pair = p.G <= 4;
  bool ok = false;
  if (p.d == 128) ok = pair ? launch_scan3_d128_p1(p, n_sms, s) : launch_scan3_d128_p0(p, n_sms, s);
  else if (p.d == 64) ok = pair ? launch_scan3_d64_p1(p, n_sms, s) : launch_scan3_d64_p0(p, n_sms, s);
  return ok ? 1 : 0;
}

int launch_combine3(const Combine3Params& p, int n_segs, cudaStream_t s) {
  if (p.d == 128) combine3_kernel<128><<<n_segs, 128, 0, s>>>(p);
  else combine3_kernel<64><<<n_segs, 128, 0, s>>>(p);
  return 1;
}

}  // namespace dwkv
