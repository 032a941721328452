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

constexpr int kChunk = 64;

__global__ void __launch_bounds__(128) combine3_kernel(const Combine3Params p) {
  __shared__ float red[16][8];
  __shared__ float mstar[8], lstar[8];
  __shared__ float wbuf[kChunk][8];
  __shared__ float astar[8][64];
  const int seg = blockIdx.x, tid = threadIdx.x;
  const int b = seg / p.LH, lh = seg - b * p.LH;
  const int layer = p.layer0 + lh / p.H, h = lh % p.H;
  const int G = p.G, r = p.r, d = p.d, PR = 2 + p.r + p.d;
  const int P0 = p.pstart[seg], n = p.pstart[seg + 1] - P0;
  const float* part = p.part + (size_t)P0 * (size_t)(G * PR);
  {
    const int gq = tid & 7, sl = tid >> 3;
    float mx = -INFINITY;
    if (gq < G)
      for (int k = sl; k < n; k += 16) mx = fmaxf(mx, part[(size_t)k * (G * PR) + gq * PR]);
    red[sl][gq] = mx;
    __syncthreads();
    if (tid < 8) {
      float v = red[0][tid];
      for (int s2 = 1; s2 < 16; ++s2) v = fmaxf(v, red[s2][tid]);
      mstar[tid] = v;
    }
    __syncthreads();
  }
  float lacc = 0.f;
  float areg[4] = {0.f, 0.f, 0.f, 0.f};   // elements idx = tid + 128*x of the G x r matrix a*
  float ereg[8];                          // thread i < d: e*[gq][i]
#pragma unroll
  for (int gq = 0; gq < 8; ++gq) ereg[gq] = 0.f;
  for (int c0 = 0; c0 < n; c0 += kChunk) {
    const int nc = min(kChunk, n - c0);
    const float* pc = part + (size_t)c0 * (G * PR);
    for (int idx = tid; idx < nc * G; idx += 128) {
      const int k = idx / G, gq = idx - k * G;
      const float m = pc[(size_t)k * (G * PR) + gq * PR];
      wbuf[k][gq] = (m == -INFINITY) ? 0.f : ex2(m - mstar[gq]);
    }
    __syncthreads();
    if (tid < G)
      for (int k = 0; k < nc; ++k) lacc = fmaf(wbuf[k][tid], pc[(size_t)k * (G * PR) + tid * PR + 1], lacc);
#pragma unroll
    for (int x = 0; x < 4; ++x) {
      const int idx = tid + 128 * x;
      if (idx < G * r) {
        const int gq = idx / r, j = idx - gq * r;
        float a = areg[x];
        for (int k = 0; k < nc; ++k) a = fmaf(wbuf[k][gq], pc[(size_t)k * (G * PR) + gq * PR + 2 + j], a);
        areg[x] = a;
      }
    }
    if (tid < d) {
      for (int k = 0; k < nc; ++k) {
        const float* e = pc + (size_t)k * (G * PR) + 2 + r + tid;
#pragma unroll
        for (int gq = 0; gq < 8; ++gq)
          if (gq < G) ereg[gq] = fmaf(wbuf[k][gq], e[gq * PR], ereg[gq]);
      }
    }
    __syncthreads();
  }
  if (tid < G) lstar[tid] = lacc;
#pragma unroll
  for (int x = 0; x < 4; ++x) {
    const int idx = tid + 128 * x;
    if (idx < G * r) astar[idx / r][idx % r] = areg[x];
  }
  __syncthreads();
  if (tid < d) {
    const __nv_bfloat16* BV = p.BV + ((size_t)(layer / p.w) * p.H + h) * (size_t)r * d + tid;
    const float gv = __bfloat162float(p.gV[((size_t)layer * p.H + h) * d + tid]);
    float acc[8];
#pragma unroll
    for (int gq = 0; gq < 8; ++gq) acc[gq] = 0.f;
    for (int j = 0; j < r; ++j) {
      const float bv = __bfloat162float(BV[(size_t)j * d]);
#pragma unroll
      for (int gq = 0; gq < 8; ++gq) acc[gq] = fmaf(astar[gq][j], bv, acc[gq]);
    }
    float* out = p.out + (((size_t)b * p.Lq + (p.Lq == 1 ? 0 : layer)) * (size_t)(p.H * G) + (size_t)h * G) * d + tid;
#pragma unroll
    for (int gq = 0; gq < 8; ++gq)
      if (gq < G) out[(size_t)gq * d] = (gv * acc[gq] + ereg[gq]) / lstar[gq];
  }
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
  combine3_kernel<<<n_segs, 128, 0, s>>>(p);
  return 1;
}

}  // namespace dwkv
