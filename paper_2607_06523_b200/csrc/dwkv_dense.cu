// dwkv_dense.cu -- from-scratch dense-bf16-cache decode attention, the comparison kernel of SURVEY.md section 8a
// step a5 (BASELINE.json north_star: "the same figures for a from-scratch dense-bf16-cache decode kernel").
// Plain softmax attention over K, V [n_seqs, L, H_kv, T, d] bf16 (row-major, no special packing), split-T with a
// log-sum-exp combine, all G query heads of a kv head share every cache load, mma.sync bf16 contractions.
#include <mutex>
#include <string>

#include "dwkv_internal.h"
#include "../../include/dwkv.h"

namespace dwkv {
namespace {

constexpr uint32_t kFull = 0xffffffffu;

__device__ __forceinline__ float ex2(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ uint4 ldg_stream(const void* p) {
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
               : "l"(p));
  return r;
}
__device__ __forceinline__ void mma16816(float& d0, float& d1, uint32_t a0, uint32_t a2, uint32_t b0, uint32_t b1) {
  float j2, j3;
  asm("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%5}, {%7,%8}, {%0,%1,%9,%9};"
      : "+f"(d0), "+f"(d1), "=f"(j2), "=f"(j3)
      : "r"(a0), "r"(0u), "r"(a2), "r"(b0), "r"(b1), "f"(0.f));
}
__device__ __forceinline__ uint32_t pack_bf16x2(float lo, float hi) {
  __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<uint32_t*>(&v);
}
__device__ __forceinline__ uint32_t comp(const uint4& v, int j) { return j == 0 ? v.x : j == 1 ? v.y : j == 2 ? v.z : v.w; }

struct DenseParams {
  const __nv_bfloat16 *K, *V, *q;
  float* part;     // [n_lhb][n_splits][G][2 + D]
  float* out;      // [n_seqs][L][Hq][D]
  int64_t T;
  int32_t n_splits, steps_per_split;   // a step = 16 tokens
  int32_t L, H, G;
  float cscale;
};

// grid (n_splits, n_seqs*L*H); 4 warps; warp w takes 16-token steps w, w+4, ... of the split.
template <int D>
__global__ void __launch_bounds__(128, 3) dense_scan_kernel(DenseParams p) {
  constexpr int KC = D / 32;      // 16-byte K chunks per lane per token row
  constexpr int VC = D / 64;      // 16-byte V chunks per lane per token
  constexpr int NT = D / 8;       // output n-tiles
  const int split = blockIdx.x, lhb = blockIdx.y;
  const int h = lhb % p.H;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, g = lane >> 2, t = lane & 3;
  const __nv_bfloat16* Kb = p.K + (size_t)lhb * p.T * D;
  const __nv_bfloat16* Vb = p.V + (size_t)lhb * p.T * D;
  const int b_l = lhb / p.H;   // = b*L + l
  const __nv_bfloat16* q = p.q + ((size_t)b_l * (p.H * p.G) + (size_t)h * p.G + g) * D;

  // A fragments of q: step (x, hh) covers channels 8(t+4x)+4hh .. +3 (k order permuted to match 16-byte K loads)
  uint32_t qa[KC][2][2];
#pragma unroll
  for (int x = 0; x < KC; ++x)
#pragma unroll
    for (int hh = 0; hh < 2; ++hh) {
      const int ch = 8 * (t + 4 * x) + 4 * hh;
      qa[x][hh][0] = (g < p.G) ? *reinterpret_cast<const uint32_t*>(q + ch) : 0u;
      qa[x][hh][1] = (g < p.G) ? *reinterpret_cast<const uint32_t*>(q + ch + 2) : 0u;
    }
  float m = -INFINITY, l = 0.f;
  float acc[NT][2];
#pragma unroll
  for (int c = 0; c < NT; ++c) acc[c][0] = acc[c][1] = 0.f;

  const int64_t step0 = (int64_t)split * p.steps_per_split;
  const int64_t nsteps_total = (p.T + 15) / 16;
  const int64_t step1 = min(step0 + p.steps_per_split, nsteps_total);
  for (int64_t st = step0 + warp; st < step1; st += 4) {
    const int64_t tok0 = st * 16;
    uint4 kr[2][KC], vr[4][VC];
#pragma unroll
    for (int j = 0; j < 2; ++j) {
      const int64_t tk = min(tok0 + 8 * j + g, p.T - 1);
#pragma unroll
      for (int x = 0; x < KC; ++x) kr[j][x] = ldg_stream(Kb + tk * D + 8 * (t + 4 * x));
    }
#pragma unroll
    for (int v = 0; v < 4; ++v) {      // tokens 2t, 2t+1, 2t+8, 2t+9 of the step
      const int64_t tk = min(tok0 + 2 * t + (v & 1) + 8 * (v >> 1), p.T - 1);
#pragma unroll
      for (int x = 0; x < VC; ++x) vr[v][x] = ldg_stream(Vb + tk * D + 64 * x + 8 * g);
    }
    float s[2][2];
#pragma unroll
    for (int j = 0; j < 2; ++j) {
      s[j][0] = s[j][1] = 0.f;
#pragma unroll
      for (int x = 0; x < KC; ++x)
#pragma unroll
        for (int hh = 0; hh < 2; ++hh)
          mma16816(s[j][0], s[j][1], qa[x][hh][0], qa[x][hh][1], comp(kr[j][x], 2 * hh), comp(kr[j][x], 2 * hh + 1));
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        s[j][e] *= p.cscale;
        if (tok0 + 8 * j + 2 * t + e >= p.T) s[j][e] = -INFINITY;
      }
    }
    float mx = fmaxf(fmaxf(s[0][0], s[0][1]), fmaxf(s[1][0], s[1][1]));
    mx = fmaxf(mx, __shfl_xor_sync(kFull, mx, 1));
    mx = fmaxf(mx, __shfl_xor_sync(kFull, mx, 2));
    const float m_new = fmaxf(m, mx);
    if (__any_sync(kFull, m_new > m)) {
      const float corr = ex2(m - m_new);
      l *= corr;
#pragma unroll
      for (int c = 0; c < NT; ++c) { acc[c][0] *= corr; acc[c][1] *= corr; }
      m = m_new;
    }
    const float p00 = ex2(s[0][0] - m), p01 = ex2(s[0][1] - m), p10 = ex2(s[1][0] - m), p11 = ex2(s[1][1] - m);
    l += (p00 + p01) + (p10 + p11);
    const uint32_t a0 = pack_bf16x2(p00, p01), a2 = pack_bf16x2(p10, p11);
#pragma unroll
    for (int x = 0; x < VC; ++x)
#pragma unroll
      for (int wv = 0; wv < 4; ++wv) {      // word wv of the chunk = channels 64x + 8g + 2wv, +1  -> n-tiles 8x+2wv, +1
        const uint32_t A = comp(vr[0][x], wv), B = comp(vr[1][x], wv), C = comp(vr[2][x], wv), Dd = comp(vr[3][x], wv);
        const uint32_t b0e = __byte_perm(A, B, 0x5410), b0o = __byte_perm(A, B, 0x7632);
        const uint32_t b1e = __byte_perm(C, Dd, 0x5410), b1o = __byte_perm(C, Dd, 0x7632);
        mma16816(acc[8 * x + 2 * wv][0], acc[8 * x + 2 * wv][1], a0, a2, b0e, b1e);
        mma16816(acc[8 * x + 2 * wv + 1][0], acc[8 * x + 2 * wv + 1][1], a0, a2, b0o, b1o);
      }
  }
  l += __shfl_xor_sync(kFull, l, 1);
  l += __shfl_xor_sync(kFull, l, 2);

  __shared__ float sm_m[4][8], sm_l[4][8];
  __shared__ float sm_o[4][8][D];
  if (t == 0) { sm_m[warp][g] = m; sm_l[warp][g] = l; }
#pragma unroll
  for (int c = 0; c < NT; ++c)
#pragma unroll
    for (int e = 0; e < 2; ++e) {
      const int col = 2 * t + e;                         // C-fragment column = (channel / 8) % 8
      const int ch = 64 * (c / 8) + 8 * col + (c % 8);   // n-tile c = (channel % 8) + 8 * (channel / 64)
      sm_o[warp][g][ch] = acc[c][e];
    }
  __syncthreads();
  const int G = p.G, PR = 2 + D;
  float* prec = p.part + ((size_t)lhb * p.n_splits + split) * (size_t)(G * PR);
  for (int idx = tid; idx < G * PR; idx += 128) {
    const int gq = idx / PR, k = idx % PR;
    const float ms = fmaxf(fmaxf(sm_m[0][gq], sm_m[1][gq]), fmaxf(sm_m[2][gq], sm_m[3][gq]));
    float v = 0.f;
#pragma unroll
    for (int w = 0; w < 4; ++w) {
      const float f = (sm_m[w][gq] == -INFINITY) ? 0.f : ex2(sm_m[w][gq] - ms);
      const float x = (k == 0) ? 0.f : (k == 1) ? sm_l[w][gq] : sm_o[w][gq][k - 2];
      v = fmaf(f, x, v);
    }
    prec[idx] = (k == 0) ? ms : v;
  }
}

// grid (n_lhb); thread per channel
template <int D>
__global__ void __launch_bounds__(D) dense_combine_kernel(DenseParams p) {
  const int lhb = blockIdx.x, i = threadIdx.x, G = p.G, PR = 2 + D;
  const int h = lhb % p.H, b_l = lhb / p.H;
  const float* part = p.part + (size_t)lhb * p.n_splits * (size_t)(G * PR);
  for (int gq = 0; gq < G; ++gq) {
    float ms = -INFINITY;
    for (int s = 0; s < p.n_splits; ++s) ms = fmaxf(ms, part[(size_t)s * G * PR + gq * PR]);
    float lsum = 0.f, o = 0.f;
    for (int s = 0; s < p.n_splits; ++s) {
      const float* r = part + (size_t)s * G * PR + gq * PR;
      const float f = (r[0] == -INFINITY) ? 0.f : ex2(r[0] - ms);
      lsum = fmaf(f, r[1], lsum);
      o = fmaf(f, r[2 + i], o);
    }
    p.out[((size_t)b_l * (p.H * G) + (size_t)h * G + gq) * D + i] = o / lsum;
  }
}

int dense_splits(int n_lhb, int64_t T) {
  int64_t steps = (T + 15) / 16;
  int64_t want = (148 * 12 + n_lhb - 1) / n_lhb;
  int64_t maxs = (steps + 15) / 16;   // at least 256 tokens per split
  if (want > maxs) want = maxs;
  if (want < 1) want = 1;
  return (int)want;
}

}  // namespace
}  // namespace dwkv

extern "C" uint64_t dwkv_dense_workspace_bytes(int32_t n_seqs, int32_t n_layers, int32_t n_q_heads, int32_t d_head, int64_t T) {
  // n_lhb * n_splits <= 148*12 + n_lhb, partial = G*(2+d) floats per (lhb, split), G <= 8, n_lhb*G = n_seqs*L*Hq
  (void)T;
  return ((uint64_t)148 * 12 * 8 + (uint64_t)n_seqs * n_layers * n_q_heads) * (uint64_t)(2 + d_head) * 4ull;
}

extern "C" int dwkv_dense_decode_attention(const void* K, const void* V, const void* q, float* out, void* workspace,
                                           int32_t n_seqs, int32_t n_layers, int32_t n_kv_heads, int32_t n_q_heads,
                                           int32_t d_head, int64_t T, float softmax_scale, void* stream) {
  using namespace dwkv;
  if (!K || !V || !q || !out || !workspace || n_seqs <= 0 || n_layers <= 0 || n_kv_heads <= 0 || T <= 0) return DWKV_E_INVALID;
  if (n_q_heads % n_kv_heads != 0 || n_q_heads / n_kv_heads > 8 || (d_head != 64 && d_head != 128)) return DWKV_E_INVALID;
  const int n_lhb = n_seqs * n_layers * n_kv_heads;
  if (n_lhb > 65535) return DWKV_E_INVALID;
  DenseParams p;
  p.K = (const __nv_bfloat16*)K; p.V = (const __nv_bfloat16*)V; p.q = (const __nv_bfloat16*)q;
  p.part = (float*)workspace; p.out = out; p.T = T;
  p.n_splits = dense_splits(n_lhb, T);
  const int64_t steps = (T + 15) / 16;
  p.steps_per_split = (int32_t)((steps + p.n_splits - 1) / p.n_splits);
  p.n_splits = (int32_t)((steps + p.steps_per_split - 1) / p.steps_per_split);
  p.L = n_layers; p.H = n_kv_heads; p.G = n_q_heads / n_kv_heads;
  p.cscale = (softmax_scale > 0.f ? softmax_scale : 1.0f / sqrtf((float)d_head)) * 1.4426950408889634f;
  cudaStream_t s = (cudaStream_t)stream;
  dim3 grid(p.n_splits, n_lhb);
  if (d_head == 128) {
    dense_scan_kernel<128><<<grid, 128, 0, s>>>(p);
    dense_combine_kernel<128><<<n_lhb, 128, 0, s>>>(p);
  } else {
    dense_scan_kernel<64><<<grid, 128, 0, s>>>(p);
    dense_combine_kernel<64><<<n_lhb, 64, 0, s>>>(p);
  }
  return cudaGetLastError() == cudaSuccess ? DWKV_OK : DWKV_E_CUDA;
}

// ---- allocation-free variant (include/dwkv.h: dwkv_dense_decode_attention_static) --------------------------------------------
// The split-T partial records live in a file-scope device array instead of a caller workspace, for callers that cannot allocate
// (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc). Every GPU that loads the library holds the array until the
// process exits. In host code `g_dense_static_scratch` is only the host-side stand-in of the symbol, never a device address: the
// address is resolved once per device with cudaGetSymbolAddress (that device current) and that pointer is what the kernels get.
namespace dwkv {
namespace {
constexpr size_t kDenseStaticBytes = DWKV_DENSE_STATIC_SCRATCH_BYTES;
static __device__ __align__(256) unsigned char g_dense_static_scratch[kDenseStaticBytes];

constexpr int kMaxDevices = 64;
std::mutex g_dense_static_mu;
void* g_dense_static_ptr[kMaxDevices] = {};

// device address of the array on the current device; resolved on the first call per device
int dense_static_ptr(void** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return set_error(DWKV_E_CUDA, std::string("cudaGetDevice: ") + cudaGetErrorString(e));
  if (dev < 0 || dev >= kMaxDevices) return set_error(DWKV_E_INVALID, "dwkv_dense_decode_attention_static: device ordinal beyond 63");
  std::lock_guard<std::mutex> lock(g_dense_static_mu);
  if (!g_dense_static_ptr[dev]) {
    void* ptr = nullptr;
    e = cudaGetSymbolAddress(&ptr, g_dense_static_scratch);
    if (e != cudaSuccess || !ptr)
      return set_error(DWKV_E_CUDA, std::string("cudaGetSymbolAddress(g_dense_static_scratch): ") + cudaGetErrorString(e));
    g_dense_static_ptr[dev] = ptr;
  }
  *out = g_dense_static_ptr[dev];
  return DWKV_OK;
}
}  // namespace
}  // namespace dwkv

extern "C" int dwkv_dense_decode_attention_static(const void* K, const void* V, const void* q, float* out, int32_t n_seqs,
                                                  int32_t n_layers, int32_t n_kv_heads, int32_t n_q_heads, int32_t d_head,
                                                  int64_t T, float softmax_scale, void* stream) {
  using namespace dwkv;
  if (!K || !V || !q || !out || n_seqs <= 0 || n_layers <= 0 || n_kv_heads <= 0 || n_q_heads <= 0 || T <= 0)
    return set_error(DWKV_E_INVALID, "dwkv_dense_decode_attention_static: NULL pointer or non-positive size");
  if (n_q_heads % n_kv_heads != 0 || n_q_heads / n_kv_heads > 8 || (d_head != 64 && d_head != 128))
    return set_error(DWKV_E_INVALID, "dwkv_dense_decode_attention_static: needs H_q = G * H_kv with G <= 8 and d_head 64 or 128");
  const int64_t n_lhb = (int64_t)n_seqs * n_layers * n_kv_heads;
  if (n_lhb > 65535) return set_error(DWKV_E_INVALID, "dwkv_dense_decode_attention_static: n_seqs * n_layers * n_kv_heads > 65535");
  // the partial records the launch below will write: [n_lhb][n_splits][G][2 + d] fp32, n_splits as dwkv_dense_decode_attention cuts T
  const int64_t steps = (T + 15) / 16;
  int64_t n_splits = dense_splits((int)n_lhb, T);
  const int64_t per = (steps + n_splits - 1) / n_splits;
  n_splits = (steps + per - 1) / per;
  const uint64_t need = (uint64_t)n_lhb * (uint64_t)n_splits * (uint64_t)(n_q_heads / n_kv_heads) * (uint64_t)(2 + d_head) * 4ull;
  if (need > kDenseStaticBytes)
    return set_error(DWKV_E_INVALID, "dwkv_dense_decode_attention_static: the call needs " + std::to_string(need) +
                                         " bytes of split partials, the static scratch holds " + std::to_string(kDenseStaticBytes) +
                                         " (DWKV_DENSE_STATIC_SCRATCH_BYTES); use dwkv_dense_decode_attention with a caller workspace");
  void* scratch = nullptr;
  const int rc = dense_static_ptr(&scratch);
  if (rc) return rc;
  // nothing in the array has to start at zero: the scan kernel writes every record of this launch in full before the combine
  // kernel of the same stream reads them, and records of earlier calls beyond this launch's extent are never read
  const int rc2 = dwkv_dense_decode_attention(K, V, q, out, scratch, n_seqs, n_layers, n_kv_heads, n_q_heads, d_head, T, softmax_scale, stream);
  if (rc2) return set_error(rc2, "dwkv_dense_decode_attention_static: kernel launch failed");
  return DWKV_OK;
}

