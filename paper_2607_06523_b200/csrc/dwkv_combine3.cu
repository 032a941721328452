// dwkv_combine3.cu -- a3: split-combine + back-projection, and the dispatcher of the fused
// decode kernel instances. One CTA per (segment = (sequence b, layer, kv head), query head): log-sum-exp merge of the warp partials
// (m, l, a[r], e[d]) the scan left for the segment, then  o = ( gV * (BV^T a) + e ) / l  for the G query heads.
#include "dwkv_internal.h"
#include "dwkv_mma.cuh"

namespace dwkv {

bool launch_scan3_d64_p0(const Scan3Params& p, int n_sms, cudaStream_t s, cudaError_t* err);
bool launch_scan3_d64_p1(const Scan3Params& p, int n_sms, cudaStream_t s, cudaError_t* err);
bool launch_scan3_d128_p0(const Scan3Params& p, int n_sms, cudaStream_t s, cudaError_t* err);
bool launch_scan3_d128_p1(const Scan3Params& p, int n_sms, cudaStream_t s, cudaError_t* err);
bool launch_scan3_d64_p0_i8(const Scan3Params& p, int n_sms, cudaStream_t s, cudaError_t* err);
bool launch_scan3_d64_p1_i8(const Scan3Params& p, int n_sms, cudaStream_t s, cudaError_t* err);
bool launch_scan3_d128_p0_i8(const Scan3Params& p, int n_sms, cudaStream_t s, cudaError_t* err);
bool launch_scan3_d128_p1_i8(const Scan3Params& p, int n_sms, cudaStream_t s, cudaError_t* err);

namespace {
using namespace dwkv::dev;

// SPLIT (S = 4 or 16): one CTA of S warps merges the partials of one (segment, query head); the warps split the partial list
// (warp w takes partials w, w+S, ...) -- for per-layer calls, where a segment has 20-150 partials and there are only a few
// dozen (segment, head) pairs: the merge is a chain of dependent L2 round trips, so its time is set by the partials per warp. !SPLIT: one CTA per segment, warp w merges
// heads w, w+4 on its own -- for all-layer steps (1-6 partials per segment, thousands of segments). Lanes run over rank
// columns for a*, over channels (D / 32 each) for e* and the back-projection.
template <int D, int S>      // S = warps sharing one head's partial list: 1 (no split) or 4
__global__ void __launch_bounds__(128) combine3_kernel(const Combine3Params p) {
  constexpr bool SPLIT = S > 1;
  constexpr int CPL = D / 32;                       // channels per lane
  __shared__ float sh_l[S];
  __shared__ float sh_a[S][64];
  __shared__ float sh_e[S][D];
  const int seg = blockIdx.x, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int ws = SPLIT ? warp : 0;                  // this warp's offset in the split
  const int b = seg / p.LH, lh = seg - b * p.LH;
  const int layer = p.layer0 + lh / p.H, h = lh % p.H;
  const int G = p.G, r = p.r, PR = 2 + p.r + D;
  const int P0 = __ldg(p.pstart + seg), n = __ldg(p.pstart + seg + 1) - P0;
  const size_t stride = (size_t)G * PR;
  // The merge is a chain of dependent L2 round trips (~0.8 us each), so everything that does not depend on an earlier load is
  // requested up front. The basis rows and the gate of the back-projection (the same for every query head of the segment) and the
  // plan are constants: they are requested BEFORE the grid dependency resolves, i.e. while the decode kernel still drains.
  const bool finisher = !SPLIT || warp == 0;
  const __nv_bfloat16* BV = p.BV + ((size_t)(layer / p.w) * p.H + h) * (size_t)r * D + lane * CPL;
  const __nv_bfloat16* gVp = p.gV + ((size_t)layer * p.H + h) * D + lane * CPL;
  uint2 bw[32];                                     // rows 0..31 of the basis block (CPL = 2: .y unused)
  uint2 gw = make_uint2(0u, 0u);
  if (finisher) {
#pragma unroll
    for (int j = 0; j < 32; ++j) {
      if constexpr (CPL == 4) bw[j] = (j < r) ? __ldg(reinterpret_cast<const uint2*>(BV + (size_t)j * D)) : make_uint2(0u, 0u);
      else bw[j] = make_uint2((j < r) ? __ldg(reinterpret_cast<const uint32_t*>(BV + (size_t)j * D)) : 0u, 0u);
    }
    if constexpr (CPL == 4) gw = __ldg(reinterpret_cast<const uint2*>(gVp));
    else gw.x = __ldg(reinterpret_cast<const uint32_t*>(gVp));
  }
  // programmatic dependent launch: this grid may start while the decode kernel drains; wait for its completion and flush
  cudaGridDependencySynchronize();
  cudaTriggerProgrammaticLaunchCompletion();        // the next decode kernel of the stream may become resident; it waits for this grid's end
  for (int gq = SPLIT ? (int)blockIdx.y : warp; gq < G; gq += SPLIT ? G : 4) {
  const float* part = p.part + ((size_t)P0 * G + gq) * PR;       // partial k of this head: part + k * stride
  // (the maxima of all partials and the first batch of this warp's partial records are requested together: the weights need m*, the
  //  loads do not)
  const int nw = (n > ws) ? (n - ws + S - 1) / S : 0;            // partials of this warp: ws, ws + S, ...
  // first batch of this warp's partials (8), requested before m* is known
  float va0[8], va1[8], ml0[8], ml1[8];
  float2 ve[8][CPL / 2];
#pragma unroll
  for (int u = 0; u < 8; ++u) {
    const float* rec = part + (size_t)(ws + S * min(u, max(nw - 1, 0))) * stride;
    const bool ok = u < nw;
    const float2 ml = ok ? *reinterpret_cast<const float2*>(rec) : make_float2(-INFINITY, 0.f);
    ml0[u] = ml.x; ml1[u] = ml.y;
    va0[u] = (ok && lane < r) ? rec[2 + lane] : 0.f;
    va1[u] = (ok && lane + 32 < r) ? rec[2 + lane + 32] : 0.f;
#pragma unroll
    for (int c = 0; c < CPL / 2; ++c) ve[u][c] = ok ? *reinterpret_cast<const float2*>(rec + 2 + r + lane * CPL + 2 * c) : make_float2(0.f, 0.f);
  }
  // pass 1: m* over all partials (every warp computes it: n is small, the loads hit L2)
  float mstar = -INFINITY;
  for (int k0 = lane; k0 < n; k0 += 32 * 8) {       // 8 independent loads in flight per lane
    float v[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) v[u] = (k0 + 32 * u < n) ? part[(size_t)(k0 + 32 * u) * stride] : -INFINITY;
#pragma unroll
    for (int u = 0; u < 8; ++u) mstar = fmaxf(mstar, v[u]);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) mstar = fmaxf(mstar, __shfl_xor_sync(kFull, mstar, o));
  // pass 2: weighted sums; lanes hold rank columns (a*) and channels (e*); every lane computes the weights of the batch itself
  float lsum = 0.f, a0 = 0.f, a1 = 0.f, e[CPL];
#pragma unroll
  for (int c = 0; c < CPL; ++c) e[c] = 0.f;
#pragma unroll
  for (int u = 0; u < 8; ++u) {
    const float wu = (ml0[u] == -INFINITY) ? 0.f : ex2(ml0[u] - mstar);
    lsum = fmaf(wu, ml1[u], lsum);
    a0 = fmaf(wu, va0[u], a0);
    a1 = fmaf(wu, va1[u], a1);
#pragma unroll
    for (int c = 0; c < CPL / 2; ++c) { e[2 * c] = fmaf(wu, ve[u][c].x, e[2 * c]); e[2 * c + 1] = fmaf(wu, ve[u][c].y, e[2 * c + 1]); }
  }
  for (int i0 = 8; i0 < nw; i0 += 8) {               // further batches (more than 8 partials per warp: rare)
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const bool ok = i0 + u < nw;
      const float* rec = part + (size_t)(ws + S * min(i0 + u, nw - 1)) * stride;
      const float2 ml = ok ? *reinterpret_cast<const float2*>(rec) : make_float2(-INFINITY, 0.f);
      ml0[u] = ml.x; ml1[u] = ml.y;
      va0[u] = (ok && lane < r) ? rec[2 + lane] : 0.f;
      va1[u] = (ok && lane + 32 < r) ? rec[2 + lane + 32] : 0.f;
#pragma unroll
      for (int c = 0; c < CPL / 2; ++c) ve[u][c] = ok ? *reinterpret_cast<const float2*>(rec + 2 + r + lane * CPL + 2 * c) : make_float2(0.f, 0.f);
    }
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const float wu = (ml0[u] == -INFINITY) ? 0.f : ex2(ml0[u] - mstar);
      lsum = fmaf(wu, ml1[u], lsum);
      a0 = fmaf(wu, va0[u], a0);
      a1 = fmaf(wu, va1[u], a1);
#pragma unroll
      for (int c = 0; c < CPL / 2; ++c) { e[2 * c] = fmaf(wu, ve[u][c].x, e[2 * c]); e[2 * c + 1] = fmaf(wu, ve[u][c].y, e[2 * c + 1]); }
    }
  }
  float lstar = lsum;                                // (every lane accumulated every partial of the warp: no lane reduction needed)
  if constexpr (SPLIT) {
    if (lane == 0) sh_l[warp] = lsum;
    sh_a[warp][lane] = a0; sh_a[warp][lane + 32] = a1;
#pragma unroll
    for (int c = 0; c < CPL; ++c) sh_e[warp][lane * CPL + c] = e[c];
    __syncthreads();
    if (warp != 0) return;
    lstar = 0.f; a0 = 0.f; a1 = 0.f;
#pragma unroll
    for (int c = 0; c < CPL; ++c) e[c] = 0.f;
#pragma unroll
    for (int w = 0; w < S; ++w) {
      lstar += sh_l[w]; a0 += sh_a[w][lane]; a1 += sh_a[w][lane + 32];
#pragma unroll
      for (int c = 0; c < CPL; ++c) e[c] += sh_e[w][lane * CPL + c];
    }
  }
  // back-projection o = (gV * (BV^T a*) + e*) / l*: basis rows already in registers, a*_j broadcast by shuffle
  float acc[CPL];
#pragma unroll
  for (int c = 0; c < CPL; ++c) acc[c] = 0.f;
#pragma unroll
  for (int j = 0; j < 32; ++j) {
    const float aj = __shfl_sync(kFull, a0, j);
    acc[0] = fmaf(aj, __uint_as_float(bw[j].x << 16), acc[0]); acc[1] = fmaf(aj, __uint_as_float(bw[j].x & 0xffff0000u), acc[1]);
    if constexpr (CPL == 4) { acc[2] = fmaf(aj, __uint_as_float(bw[j].y << 16), acc[2]); acc[3] = fmaf(aj, __uint_as_float(bw[j].y & 0xffff0000u), acc[3]); }
  }
  if (r > 32) {                                      // basis ranks 48 / 64: the second half of the rows
    uint2 bw2[32];
#pragma unroll
    for (int j = 0; j < 32; ++j) {
      if constexpr (CPL == 4) bw2[j] = (32 + j < r) ? __ldg(reinterpret_cast<const uint2*>(BV + (size_t)(32 + j) * D)) : make_uint2(0u, 0u);
      else bw2[j] = make_uint2((32 + j < r) ? __ldg(reinterpret_cast<const uint32_t*>(BV + (size_t)(32 + j) * D)) : 0u, 0u);
    }
#pragma unroll
    for (int j = 0; j < 32; ++j) {
      const float aj = __shfl_sync(kFull, a1, j);
      acc[0] = fmaf(aj, __uint_as_float(bw2[j].x << 16), acc[0]); acc[1] = fmaf(aj, __uint_as_float(bw2[j].x & 0xffff0000u), acc[1]);
      if constexpr (CPL == 4) { acc[2] = fmaf(aj, __uint_as_float(bw2[j].y << 16), acc[2]); acc[3] = fmaf(aj, __uint_as_float(bw2[j].y & 0xffff0000u), acc[3]); }
    }
  }
  const float inv = 1.f / lstar;
  float* out = p.out + (((size_t)b * p.Lq + (p.Lq == 1 ? 0 : layer)) * (size_t)(p.H * G) + (size_t)h * G + gq) * D + lane * CPL;
  if constexpr (CPL == 4) {
    float4 o;
    o.x = (__uint_as_float(gw.x << 16) * acc[0] + e[0]) * inv; o.y = (__uint_as_float(gw.x & 0xffff0000u) * acc[1] + e[1]) * inv;
    o.z = (__uint_as_float(gw.y << 16) * acc[2] + e[2]) * inv; o.w = (__uint_as_float(gw.y & 0xffff0000u) * acc[3] + e[3]) * inv;
    *reinterpret_cast<float4*>(out) = o;
  } else {
    float2 o;
    o.x = (__uint_as_float(gw.x << 16) * acc[0] + e[0]) * inv; o.y = (__uint_as_float(gw.x & 0xffff0000u) * acc[1] + e[1]) * inv;
    *reinterpret_cast<float2*>(out) = o;
  }
  }   // heads of this warp
}

}  // namespace

int scan3_num_slices(int n_sms) { return n_sms * 8; }

int launch_scan3(const Scan3Params& p, int n_sms, cudaStream_t s, cudaError_t* err) {
  const bool pair = p.G <= 4;
  bool ok = false;
  *err = cudaSuccess;
  if (p.i8) {
    if (p.d == 128) ok = pair ? launch_scan3_d128_p1_i8(p, n_sms, s, err) : launch_scan3_d128_p0_i8(p, n_sms, s, err);
    else if (p.d == 64) ok = pair ? launch_scan3_d64_p1_i8(p, n_sms, s, err) : launch_scan3_d64_p0_i8(p, n_sms, s, err);
  } else if (p.d == 128) ok = pair ? launch_scan3_d128_p1(p, n_sms, s, err) : launch_scan3_d128_p0(p, n_sms, s, err);
  else if (p.d == 64) ok = pair ? launch_scan3_d64_p1(p, n_sms, s, err) : launch_scan3_d64_p0(p, n_sms, s, err);
  return ok ? 1 : 0;
}

int launch_combine3(const Combine3Params& p, int n_segs, int split, cudaStream_t s, cudaError_t* err) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = split > 1 ? dim3(n_segs, p.G) : dim3(n_segs);       // split: the CTA's 4 warps share the partial list of one head
  cfg.blockDim = dim3(128);
  cfg.dynamicSmemBytes = 0;
  cfg.stream = s;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;     // overlap this launch with the tail of the scan
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  if (p.d == 128) {
    if (split == 4) *err = cudaLaunchKernelEx(&cfg, combine3_kernel<128, 4>, p);
    else *err = cudaLaunchKernelEx(&cfg, combine3_kernel<128, 1>, p);
  } else {
    if (split == 4) *err = cudaLaunchKernelEx(&cfg, combine3_kernel<64, 4>, p);
    else *err = cudaLaunchKernelEx(&cfg, combine3_kernel<64, 1>, p);
  }
  return 1;
}

}  // namespace dwkv
