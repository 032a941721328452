// dwkv_basis.cu -- basis construction from the prefill K/V ("a small randomized
// low-rank sketch of the cached keys and values after prefill"; reading A24).
//
//   sketch_kernel<D, MT>   P[split][(l,h,Z)] = Omega_j^T X_l over a token range: bf16 x bf16 on mma.sync, fp32 accumulate.
//                          A = Omega tile (sketch rows x tokens), B = the token rows (tokens x channels); both tiles are
//                          staged by cp.async (double buffer) and read with ldmatrix / ldmatrix.trans. HBM-bound: the dense
//                          K/V of the prefill is read exactly once.
//   basis_svd_kernel<D>    per (window, head, Z): S = sum over the window's layers and the splits of P / gate, one-sided Jacobi
//                          (Hestenes) on the rows of S until they are mutually orthogonal -- they are then sigma_i * w_i^T --,
//                          the r rows of largest norm, normalised, signed (largest-magnitude entry positive), rounded to bf16.
#include <cuda.h>

#include "dwkv_internal.h"
#include "dwkv_mma.cuh"

namespace dwkv {
namespace {
using namespace dwkv::dev;

constexpr int kSketchTok = 64;       // tokens per staged tile
constexpr int kSketchWarps = 8;
constexpr int kSketchStages = 2;      // 3 stages cost a CTA per SM (73 KB each) and ran 15 % slower

__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src, int src_bytes) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void mma16(float (&d)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t b0, uint32_t b1) {
  asm("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
      : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
      : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}

// grid (L*H*2, n_split); 8 warps, warp w owns channels [w*D/8, (w+1)*D/8) of the k x D sketch block
template <int D, int MT>      // MT = sketch rows / 16
__global__ void __launch_bounds__(kSketchWarps * 32) sketch_kernel(const __nv_bfloat16* k_dense, const __nv_bfloat16* v_dense,
                                                                  const __nv_bfloat16* omega, float* part, const int n, const int LH,
                                                                  const int H, const int w) {
  constexpr int K = 16 * MT, XP = 2 * D + 16, OP = 2 * kSketchTok + 16;      // row pitches (bytes) of the X and Omega tiles
  constexpr int XT = kSketchTok * XP, OT = K * OP, NT = D / 64;                // NT = 8-channel n-tiles per warp
  extern __shared__ __align__(16) uint8_t smem_raw[];
  const uint32_t sm = (uint32_t)__cvta_generic_to_shared(smem_raw);           // [stages][X tile | Omega tile]
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int item = blockIdx.x, lh = item >> 1, z = item & 1, l = lh / H;
  const __nv_bfloat16* X = z ? v_dense : k_dense;
  const __nv_bfloat16* Om = omega + (size_t)(l % w) * K * n;                  // omega[j][i][t], j = layer inside its window
  const int per = ((n + gridDim.y - 1) / gridDim.y + kSketchTok - 1) / kSketchTok * kSketchTok;
  const int t_beg = blockIdx.y * per, t_end = min(n, t_beg + per);
  float c[MT][NT][4];
#pragma unroll
  for (int mi = 0; mi < MT; ++mi)
#pragma unroll
    for (int ni = 0; ni < NT; ++ni) c[mi][ni][0] = c[mi][ni][1] = c[mi][ni][2] = c[mi][ni][3] = 0.f;
  auto stage = [&](int buf, int t0) {
    const uint32_t xs = sm + buf * (XT + OT), os = xs + XT;
    for (int i = tid; i < kSketchTok * (D / 8); i += kSketchWarps * 32) {      // 16-byte pieces of the token rows
      const int r = i / (D / 8), p = i - r * (D / 8), t = t0 + r;
      cp_async16(xs + r * XP + 16 * p, X + ((size_t)min(t, n - 1) * LH + lh) * D + 8 * p, t < t_end ? 16 : 0);
    }
    for (int i = tid; i < K * (kSketchTok / 8); i += kSketchWarps * 32) {       // 16-byte pieces of the Omega rows (8 tokens)
      const int r = i / (kSketchTok / 8), p = i - r * (kSketchTok / 8), t = t0 + 8 * p;
      cp_async16(os + r * OP + 16 * p, Om + (size_t)r * n + min(t, n - 8), t < t_end ? 16 : 0);   // n % 8 == 0, t_end % 8 == 0
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  };
  // the next tile is being copied while tile t0 is multiplied
  for (int k = 0; k < kSketchStages - 1; ++k) {
    if (t_beg + k * kSketchTok < t_end) stage(k, t_beg + k * kSketchTok);
    else asm volatile("cp.async.commit_group;" ::: "memory");
  }
  int buf = 0;
  for (int t0 = t_beg; t0 < t_end; t0 += kSketchTok) {
    const int tn = t0 + (kSketchStages - 1) * kSketchTok;
    if (tn < t_end) stage((buf + kSketchStages - 1) % kSketchStages, tn);
    else asm volatile("cp.async.commit_group;" ::: "memory");      // empty group: uniform counting
    asm volatile("cp.async.wait_group %0;" ::"n"(kSketchStages - 1) : "memory");
    __syncthreads();
    const uint32_t xs = sm + buf * (XT + OT), os = xs + XT;
#pragma unroll
    for (int ks = 0; ks < kSketchTok / 16; ++ks) {
      // B fragments: matrices (tokens +0..7 | +8..15) x (channels c0 .. +7 | c0+8 .. +15), transposed on load
      uint32_t b[NT][2];
      {
        const int mat = lane >> 3, tok = 16 * ks + (lane & 7) + 8 * (mat & 1);
        const uint32_t a = xs + tok * XP + 2 * (warp * (D / 8) + 8 * (mat >> 1));
        if constexpr (NT == 2) {
          asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
                       : "=r"(b[0][0]), "=r"(b[0][1]), "=r"(b[1][0]), "=r"(b[1][1]) : "r"(a));
        } else {
          asm volatile("ldmatrix.sync.aligned.m8n8.x2.trans.shared.b16 {%0,%1}, [%2];" : "=r"(b[0][0]), "=r"(b[0][1]) : "r"(a));
        }
      }
#pragma unroll
      for (int mi = 0; mi < MT; ++mi) {
        uint32_t a0, a1, a2, a3;   // (sketch rows 16mi + 0..7 | +8..15) x (tokens 16ks + 0..7 | +8..15)
        const uint32_t a = os + (16 * mi + (lane & 7) + 8 * ((lane >> 3) & 1)) * OP + 2 * (16 * ks + 8 * (lane >> 4));
        asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];" : "=r"(a0), "=r"(a1), "=r"(a2), "=r"(a3) : "r"(a));
#pragma unroll
        for (int ni = 0; ni < NT; ++ni) mma16(c[mi][ni], a0, a1, a2, a3, b[ni][0], b[ni][1]);
      }
    }
    __syncthreads();
    buf = buf + 1 == kSketchStages ? 0 : buf + 1;
  }
  float* out = part + ((size_t)blockIdx.y * (2 * LH) + item) * (size_t)(K * D);
  const int g = lane >> 2, t = lane & 3;
#pragma unroll
  for (int mi = 0; mi < MT; ++mi)
#pragma unroll
    for (int ni = 0; ni < NT; ++ni) {
      const int col = warp * (D / 8) + 8 * ni + 2 * t;
      *reinterpret_cast<float2*>(out + (size_t)(16 * mi + g) * D + col) = make_float2(c[mi][ni][0], c[mi][ni][1]);
      *reinterpret_cast<float2*>(out + (size_t)(16 * mi + g + 8) * D + col) = make_float2(c[mi][ni][2], c[mi][ni][3]);
    }
}

// ---- tcgen05 variant of the sketch GEMM (d = 128) --------------------------------------------------------------------------------
// P (sketch rows, padded to M = 128) x (N = 128 channels) accumulates in TMEM over the CTA's whole token range; one elected thread
// issues tcgen05.mma (kind::f16, bf16 inputs, fp32 accumulate) on shared-memory tiles in the canonical 128-byte-swizzled layouts:
//   A = Omega tile, K-major:  row i (sketch row) = 64 tokens = 128 bytes; 8-row groups of 1024 bytes (SBO); 16-byte chunk c of row i
//       is stored at chunk c ^ (i % 8)
//   B = token rows, MN-major: k-block = 8 tokens x 64 channels = 8 rows of 128 bytes (1024 bytes, SBO between k-blocks); the two
//       64-channel halves of d = 128 lie LBO = 8 KB apart; chunk c of token t is stored at chunk c ^ (t % 8)
// All 128 threads fill the tiles with 16-byte cp.async (a ring of kUmmaStages stages); a stage is released for refilling by the
// tcgen05.commit of the MMAs that read it. The legacy mma.sync kernel above reaches 48 % of its tensor-pipe peak at 75 % of the HBM
// peak; here the tensor work is a few percent of the UMMA peak and the kernel is bound by the row loads alone.
constexpr int kUmmaStages = 3;                   // 3 x 32 KB: two CTAs per SM
constexpr int kUmmaTok = 64;                      // tokens per stage = one 128-byte swizzle row of Omega
constexpr int kUmmaXBytes = kUmmaTok * 256;       // 16 KB: 64 tokens x 128 channels bf16
constexpr int kUmmaOBytes = 128 * 128;            // 16 KB: 128 (padded) sketch rows x 64 tokens bf16
constexpr int kUmmaStageBytes = kUmmaXBytes + kUmmaOBytes;

__device__ __forceinline__ void umma_mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void umma_mbar_wait(uint32_t bar, uint32_t parity) {
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
__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
  // start address [0,14), leading byte offset [16,30), stride byte offset [32,46) (all >> 4), version 1 at [46,48), SWIZZLE_128B = 2 at [61,64)
  return (uint64_t)((saddr >> 4) & 0x3fff) | ((uint64_t)((lbo_bytes >> 4) & 0x3fff) << 16) | ((uint64_t)((sbo_bytes >> 4) & 0x3fff) << 32) |
         (1ull << 46) | (2ull << 61);
}

__global__ void __launch_bounds__(128) sketch_umma_kernel(const __nv_bfloat16* k_dense, const __nv_bfloat16* v_dense,
                                                          const __nv_bfloat16* omega, float* part, const int n, const int LH,
                                                          const int H, const int w, const int K /* sketch rows, multiple of 16 */) {
  constexpr int D = 128;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  __shared__ __align__(8) uint64_t bars[kUmmaStages + 1];
  __shared__ uint32_t tmem_base_sh;
  const uint32_t sm = ((uint32_t)__cvta_generic_to_shared(smem_raw) + 1023u) & ~1023u;
  const uint32_t bar0 = (uint32_t)__cvta_generic_to_shared(bars);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int item = blockIdx.x, lh = item >> 1, z = item & 1, l = lh / H;
  const __nv_bfloat16* X = z ? v_dense : k_dense;
  const __nv_bfloat16* Om = omega + (size_t)(l % w) * K * n;
  const int per = ((n + gridDim.y - 1) / gridDim.y + kUmmaTok - 1) / kUmmaTok * kUmmaTok;
  const int t_beg = blockIdx.y * per, t_end = min(n, t_beg + per);
  const int n_tiles = t_beg < t_end ? (t_end - t_beg + kUmmaTok - 1) / kUmmaTok : 0;
  // ---- setup: barriers, TMEM (128 fp32 columns), zero rows of the padded Omega tiles ----------------------------------------
  if (tid == 0) {
    for (int s = 0; s <= kUmmaStages; ++s) umma_mbar_init(bar0 + 8 * s, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 128;" ::"r"((uint32_t)__cvta_generic_to_shared(&tmem_base_sh)) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  for (int s = 0; s < kUmmaStages; ++s)           // sketch rows K .. 127 of every stage stay zero (the copies never touch them)
    for (int i = tid; i < (128 - K) * 8; i += 128) {
      const int row = K + i / 8, c = i % 8;
      asm volatile("st.shared.v4.u32 [%0], {%1, %1, %1, %1};" ::"r"(sm + s * kUmmaStageBytes + kUmmaXBytes + row * 128 + c * 16), "r"(0u) : "memory");
    }
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tmem = tmem_base_sh;
  auto fill = [&](int s, int t0) {
    const uint32_t xs = sm + s * kUmmaStageBytes, os = xs + kUmmaXBytes;
    for (int i = tid; i < kUmmaTok * 16; i += 128) {            // token rows: 16 chunks of 16 bytes each
      const int r = i >> 4, c16 = i & 15, t = t0 + r;
      const uint32_t dst = xs + (c16 >> 3) * 8192 + (r >> 3) * 1024 + (r & 7) * 128 + (((c16 & 7) ^ (r & 7)) << 4);
      cp_async16(dst, X + ((size_t)min(t, n - 1) * LH + lh) * D + 8 * c16, t < t_end ? 16 : 0);
    }
    for (int i = tid; i < K * 8; i += 128) {                    // Omega rows: 8 chunks of 8 tokens
      const int r = i >> 3, c = i & 7, t = t0 + 8 * c;
      const uint32_t dst = os + (r >> 3) * 1024 + (r & 7) * 128 + ((c ^ (r & 7)) << 4);
      cp_async16(dst, Om + (size_t)r * n + min(t, n - 8), t < t_end ? 16 : 0);
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  };
  // instruction descriptor: D fp32, A / B bf16, A K-major, B MN-major, N = 128, M = 128
  constexpr uint32_t idesc = (1u << 4) | (1u << 7) | (1u << 10) | (1u << 16) | ((128u >> 3) << 17) | ((128u >> 4) << 24);
  for (int k = 0; k < kUmmaStages - 1; ++k) {
    if (k < n_tiles) fill(k, t_beg + k * kUmmaTok);
    else asm volatile("cp.async.commit_group;" ::: "memory");
  }
  for (int it = 0; it < n_tiles; ++it) {
    const int s = it % kUmmaStages;
    {   // refill the stage that tile it - 1 used, once the MMAs that read it have completed
      const int nt = it + kUmmaStages - 1, sn = nt % kUmmaStages;
      if (nt < n_tiles) {
        if (it >= 1) umma_mbar_wait(bar0 + 8 * sn, (uint32_t)(((it - 1) / kUmmaStages) & 1));
        fill(sn, t_beg + nt * kUmmaTok);
      } else {
        asm volatile("cp.async.commit_group;" ::: "memory");
      }
    }
    asm volatile("cp.async.wait_group %0;" ::"n"(kUmmaStages - 1) : "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");          // generic-proxy writes -> visible to the tensor core's reads
    __syncthreads();
    if (tid == 0) {
      asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
      const uint32_t xs = sm + s * kUmmaStageBytes, os = xs + kUmmaXBytes;
#pragma unroll
      for (int ks = 0; ks < kUmmaTok / 16; ++ks) {
        const uint64_t da = umma_desc(os + 32 * ks, 16, 1024);             // K-major: 16 tokens further = 32 bytes inside the swizzled row
        const uint64_t db = umma_desc(xs + 2048 * ks, 8192, 1024);         // MN-major: 16 tokens further = two k-blocks
        const uint32_t acc = (it > 0 || ks > 0) ? 1u : 0u;
        asm volatile("{ .reg .pred p; setp.ne.b32 p, %4, 0; tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p; }"
                     ::"r"(tmem), "l"(da), "l"(db), "r"(idesc), "r"(acc) : "memory");
      }
      asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.b64 [%0];" ::"r"(bar0 + 8 * s) : "memory");
      if (it == n_tiles - 1)
        asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.b64 [%0];" ::"r"(bar0 + 8 * kUmmaStages) : "memory");
    }
  }
  // ---- epilogue: TMEM lanes = sketch rows, columns = channels -> global partial block --------------------------------------
  float* out = part + ((size_t)blockIdx.y * (2 * LH) + item) * (size_t)(K * D);
  if (n_tiles > 0) {
    umma_mbar_wait(bar0 + 8 * kUmmaStages, 0);
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  }
  const int row = 32 * warp + lane;
  if (32 * warp < K) {                           // warp-uniform: this warp's 32 lanes hold sketch rows 32 warp .. + 31
#pragma unroll
    for (int c0 = 0; c0 < D; c0 += 16) {
      uint32_t v[16];
      if (n_tiles > 0) {
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                     : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]),
                       "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
                     : "r"(tmem + ((uint32_t)(32 * warp) << 16) + (uint32_t)c0));
        asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
      } else {
#pragma unroll
        for (int x = 0; x < 16; ++x) v[x] = 0u;
      }
      if (row < K) {
#pragma unroll
        for (int x = 0; x < 16; x += 4)
          *reinterpret_cast<uint4*>(out + (size_t)row * D + c0 + x) = make_uint4(v[x], v[x + 1], v[x + 2], v[x + 3]);
      }
    }
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 128;" ::"r"(tmem) : "memory");
}

// ---- TMA-fed variant: the same tcgen05 pipeline, tiles brought in by cp.async.bulk.tensor with hardware 128-byte swizzle -----------
// Warp 0 lane 0 produces (waits for a stage's release, arms its mbarrier with the byte count, issues three tensor copies: the two
// 64-channel halves of 64 token rows and the 64-token slab of the Omega rows), warp 1 lane 0 issues the MMAs; everybody else only
// joins for the epilogue. Tokens beyond n are zero-filled by the tensor map.
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* map, uint32_t bar, int c0, int c1, int c2) {
  asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
               ::"r"(dst), "l"(map), "r"(bar), "r"(c0), "r"(c1), "r"(c2) : "memory");
}

__global__ void __launch_bounds__(128) sketch_tma_kernel(const __grid_constant__ CUtensorMap mapK, const __grid_constant__ CUtensorMap mapV,
                                                         const __grid_constant__ CUtensorMap mapO, float* part, const int n, const int LH,
                                                         const int H, const int w, const int K) {
  constexpr int D = 128, S = kUmmaStages;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  __shared__ __align__(8) uint64_t bars[2 * S + 1];              // full[S], empty[S], done
  __shared__ uint32_t tmem_base_sh;
  const uint32_t sm = ((uint32_t)__cvta_generic_to_shared(smem_raw) + 1023u) & ~1023u;
  const uint32_t bar0 = (uint32_t)__cvta_generic_to_shared(bars);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int item = blockIdx.x, lh = item >> 1, z = item & 1, l = lh / H;
  const CUtensorMap* mapX = z ? &mapV : &mapK;
  const int per = ((n + gridDim.y - 1) / gridDim.y + kUmmaTok - 1) / kUmmaTok * kUmmaTok;
  const int t_beg = blockIdx.y * per, t_end = min(n, t_beg + per);
  const int n_tiles = t_beg < t_end ? (t_end - t_beg + kUmmaTok - 1) / kUmmaTok : 0;
  if (tid == 0) {
    for (int s = 0; s <= 2 * S; ++s) umma_mbar_init(bar0 + 8 * s, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(mapX) : "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(&mapO) : "memory");
  }
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 128;" ::"r"((uint32_t)__cvta_generic_to_shared(&tmem_base_sh)) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  for (int s = 0; s < S; ++s)                     // sketch rows K .. 127 of every stage stay zero (the copies never touch them)
    for (int i = tid; i < (128 - K) * 8; i += 128) {
      const int row = K + i / 8, c = i % 8;
      asm volatile("st.shared.v4.u32 [%0], {%1, %1, %1, %1};" ::"r"(sm + s * kUmmaStageBytes + kUmmaXBytes + row * 128 + c * 16), "r"(0u) : "memory");
    }
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tmem = tmem_base_sh;
  constexpr uint32_t idesc = (1u << 4) | (1u << 7) | (1u << 10) | (1u << 16) | ((128u >> 3) << 17) | ((128u >> 4) << 24);
  if (warp == 0 && lane == 0) {
    // ===== producer =====
    const uint32_t bytes = 2 * 8192 + (uint32_t)K * 128;
    for (int it = 0; it < n_tiles; ++it) {
      const int s = it % S;
      if (it >= S) umma_mbar_wait(bar0 + 8 * (S + s), (uint32_t)(((it / S) - 1) & 1));
      const uint32_t xs = sm + s * kUmmaStageBytes, os = xs + kUmmaXBytes, full = bar0 + 8 * s;
      asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(full), "r"(bytes) : "memory");
      const int t0 = t_beg + it * kUmmaTok;
      tma_load_3d(xs, mapX, full, 0, lh, t0);
      tma_load_3d(xs + 8192, mapX, full, 64, lh, t0);
      tma_load_3d(os, &mapO, full, t0, 0, l % w);
    }
  } else if (warp == 1 && lane == 0) {
    // ===== MMA issuer =====
    for (int it = 0; it < n_tiles; ++it) {
      const int s = it % S;
      umma_mbar_wait(bar0 + 8 * s, (uint32_t)((it / S) & 1));
      asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
      const uint32_t xs = sm + s * kUmmaStageBytes, os = xs + kUmmaXBytes;
#pragma unroll
      for (int ks = 0; ks < kUmmaTok / 16; ++ks) {
        const uint64_t da = umma_desc(os + 32 * ks, 16, 1024);
        const uint64_t db = umma_desc(xs + 2048 * ks, 8192, 1024);
        const uint32_t acc = (it > 0 || ks > 0) ? 1u : 0u;
        asm volatile("{ .reg .pred p; setp.ne.b32 p, %4, 0; tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p; }"
                     ::"r"(tmem), "l"(da), "l"(db), "r"(idesc), "r"(acc) : "memory");
      }
      asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.b64 [%0];" ::"r"(bar0 + 8 * (S + s)) : "memory");
      if (it == n_tiles - 1)
        asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.b64 [%0];" ::"r"(bar0 + 8 * (2 * S)) : "memory");
    }
  }
  __syncwarp();
  // ---- epilogue: TMEM lanes = sketch rows, columns = channels -> global partial block --------------------------------------
  float* out = part + ((size_t)blockIdx.y * (2 * LH) + item) * (size_t)(K * D);
  if (n_tiles > 0) {
    umma_mbar_wait(bar0 + 8 * (2 * S), 0);
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  }
  const int row = 32 * warp + lane;
  if (32 * warp < K) {
#pragma unroll
    for (int c0 = 0; c0 < D; c0 += 16) {
      uint32_t v[16];
      if (n_tiles > 0) {
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                     : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]),
                       "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
                     : "r"(tmem + ((uint32_t)(32 * warp) << 16) + (uint32_t)c0));
        asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
      } else {
#pragma unroll
        for (int x = 0; x < 16; ++x) v[x] = 0u;
      }
      if (row < K) {
#pragma unroll
        for (int x = 0; x < 16; x += 4)
          *reinterpret_cast<uint4*>(out + (size_t)row * D + c0 + x) = make_uint4(v[x], v[x + 1], v[x + 2], v[x + 3]);
      }
    }
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 128;" ::"r"(tmem) : "memory");
}

// host: tensor maps through the driver entry point (no link against libcuda)
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                  const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn encode_tiled_fn() {
  static EncodeTiledFn fn = [] {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess) p = nullptr;
    return (EncodeTiledFn)p;
  }();
  return fn;
}
bool make_map_3d(CUtensorMap* m, const void* base, uint64_t d0, uint64_t d1, uint64_t d2, uint64_t s1_bytes, uint64_t s2_bytes, uint32_t b0,
                 uint32_t b1, uint32_t b2) {
  EncodeTiledFn fn = encode_tiled_fn();
  if (!fn) return false;
  const cuuint64_t dims[3] = {d0, d1, d2}, strides[2] = {s1_bytes, s2_bytes};
  const cuuint32_t box[3] = {b0, b1, b2}, es[3] = {1, 1, 1};
  return fn(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(base), dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// grid (M*H*2); one warp per row pair of a Jacobi step (k/2 warps, at most 32). Dynamic shared memory: S[k][D + 1] fp32, norms[k].
template <int D>
__global__ void __launch_bounds__(1024) basis_svd_kernel(const float* part, const int n_split, const __nv_bfloat16* gK,
                                                        const __nv_bfloat16* gV, __nv_bfloat16* BK, __nv_bfloat16* BV, const int K,
                                                        const int r, const int L, const int H, const int w) {
  constexpr int LD = D + 1;
  extern __shared__ __align__(16) uint8_t smem_raw[];
  float* S = reinterpret_cast<float*>(smem_raw);
  float* nrm = S + K * LD;
  __shared__ int rotated;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nthr = blockDim.x, nwarp = nthr >> 5;
  const int item = blockIdx.x, mh = item >> 1, z = item & 1, m = mh / H, h = mh - m * H, LH = L * H;
  const __nv_bfloat16* gate = z ? gV : gK;
  // ---- S = sum over the window's layers and the splits of P / gate (column scaling commutes with the sum over tokens) --------
  for (int i = tid; i < K * D; i += nthr) {
    const int row = i / D, col = i - row * D;
    float acc = 0.f;
    for (int j = 0; j < w; ++j) {
      const int lh = (m * w + j) * H + h;
      float p = 0.f;
      for (int s = 0; s < n_split; ++s) p += part[((size_t)s * (2 * LH) + 2 * lh + z) * (size_t)(K * D) + i];
      acc += __fdiv_rn(p, __bfloat162float(gate[(size_t)lh * D + col]));
    }
    S[row * LD + col] = acc;
  }
  __syncthreads();
  // ---- one-sided Jacobi: rotate row pairs until all rows are mutually orthogonal (round-robin pairing, disjoint pairs per step)
  const float tol = 1e-6f;
  for (int sweep = 0; sweep < 30; ++sweep) {
    if (tid == 0) rotated = 0;
    __syncthreads();
    for (int step = 0; step < K - 1; ++step) {
      for (int pi = warp; pi < K / 2; pi += nwarp) {
        int p, q;
        if (pi == 0) { p = K - 1; q = step; }
        else { p = (step + pi) % (K - 1); q = (step - pi + (K - 1)) % (K - 1); }
        float* sp = S + p * LD; float* sq = S + q * LD;
        float a = 0.f, b = 0.f, gmm = 0.f;
#pragma unroll
        for (int x = 0; x < D / 32; ++x) {
          const float u = sp[lane + 32 * x], v = sq[lane + 32 * x];
          a = fmaf(u, u, a); b = fmaf(v, v, b); gmm = fmaf(u, v, gmm);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
          a += __shfl_xor_sync(kFull, a, o); b += __shfl_xor_sync(kFull, b, o); gmm += __shfl_xor_sync(kFull, gmm, o);
        }
        if (fabsf(gmm) > tol * sqrtf(a * b) && gmm != 0.f) {
          const float zeta = (b - a) / (2.f * gmm);
          const float tt = copysignf(1.f, zeta) / (fabsf(zeta) + sqrtf(1.f + zeta * zeta));
          const float cs = rsqrtf(1.f + tt * tt), sn = cs * tt;
#pragma unroll
          for (int x = 0; x < D / 32; ++x) {
            const float u = sp[lane + 32 * x], v = sq[lane + 32 * x];
            sp[lane + 32 * x] = cs * u - sn * v;
            sq[lane + 32 * x] = sn * u + cs * v;
          }
          if (lane == 0) rotated = 1;
        }
      }
      __syncthreads();
    }
    if (!rotated) break;
    __syncthreads();
  }
  // ---- the r rows of largest norm, in descending order ---------------------------------------------------------------------
  for (int row = warp; row < K; row += nwarp) {
    float a = 0.f;
#pragma unroll
    for (int x = 0; x < D / 32; ++x) { const float u = S[row * LD + lane + 32 * x]; a = fmaf(u, u, a); }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) a += __shfl_xor_sync(kFull, a, o);
    if (lane == 0) nrm[row] = a;
  }
  __syncthreads();
  __nv_bfloat16* B = (z ? BV : BK) + (size_t)mh * r * D;
  for (int row = warp; row < K; row += nwarp) {
    const float a = nrm[row];
    int rank = 0;
    for (int o = 0; o < K; ++o) rank += (nrm[o] > a) || (nrm[o] == a && o < row);
    if (rank >= r) continue;
    // sign: the entry of largest magnitude is positive (first one on ties)
    float best = -1.f; int bi = 0;
#pragma unroll
    for (int x = 0; x < D / 32; ++x) {
      const float u = fabsf(S[row * LD + lane + 32 * x]);
      if (u > best) { best = u; bi = lane + 32 * x; }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      const float ob = __shfl_xor_sync(kFull, best, o); const int oi = __shfl_xor_sync(kFull, bi, o);
      if (ob > best || (ob == best && oi < bi)) { best = ob; bi = oi; }
    }
    const float inv = a > 0.f ? (S[row * LD + bi] < 0.f ? -1.f : 1.f) / sqrtf(a) : 0.f;
#pragma unroll
    for (int x = 0; x < D / 32; ++x) B[(size_t)rank * D + lane + 32 * x] = __float2bfloat16_rn(S[row * LD + lane + 32 * x] * inv);
  }
}

}  // namespace

size_t basis_scratch_bytes(const CacheGeom& g, int n_sketch, int n_split) {
  return (size_t)n_split * 2 * g.L * g.H * (size_t)n_sketch * g.d * sizeof(float);
}

int basis_num_splits(const CacheGeom& g, int n, int n_sms) {
  const int items = 2 * g.L * g.H;
  int s = (2 * n_sms + items - 1) / items;                       // about two CTAs per SM
  s = std::min(s, (n + kSketchTok - 1) / kSketchTok);
  return std::max(1, std::min(s, 16));
}

int launch_build_basis(const CacheGeom& g, int n, const __nv_bfloat16* k_dense, const __nv_bfloat16* v_dense, const __nv_bfloat16* omega,
                       int n_sketch, int n_split, float* part, const __nv_bfloat16* gK, const __nv_bfloat16* gV, __nv_bfloat16* BK,
                       __nv_bfloat16* BV, bool use_umma, cudaStream_t s) {
  const int LH = g.L * g.H, MT = n_sketch / 16;
  const size_t smem1 = kSketchStages * ((size_t)kSketchTok * (2 * g.d + 16) + (size_t)n_sketch * (2 * kSketchTok + 16));
  dim3 grid1(2 * LH, n_split);
  bool ok = true;
#define DWKV_SKETCH_CASE(DD, MM)                                                                                            \
  case MM:                                                                                                                  \
    cudaFuncSetAttribute(sketch_kernel<DD, MM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem1);                   \
    sketch_kernel<DD, MM><<<grid1, kSketchWarps * 32, smem1, s>>>(k_dense, v_dense, omega, part, n, LH, g.H, g.w);            \
    break;
  CUtensorMap mapK, mapV, mapO;
  const bool aligned = (((uintptr_t)k_dense | (uintptr_t)v_dense | (uintptr_t)omega) & 15) == 0;
  if (g.d == 128 && use_umma && aligned &&
      make_map_3d(&mapK, k_dense, 128, (uint64_t)LH, (uint64_t)n, 256, (uint64_t)LH * 256, 64, 1, kUmmaTok) &&
      make_map_3d(&mapV, v_dense, 128, (uint64_t)LH, (uint64_t)n, 256, (uint64_t)LH * 256, 64, 1, kUmmaTok) &&
      make_map_3d(&mapO, omega, (uint64_t)n, (uint64_t)n_sketch, (uint64_t)g.w, (uint64_t)n * 2, (uint64_t)n_sketch * n * 2, kUmmaTok,
                  (uint32_t)n_sketch, 1)) {
    const size_t smem_u = (size_t)kUmmaStages * kUmmaStageBytes + 1024;
    cudaFuncSetAttribute(sketch_tma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_u);
    sketch_tma_kernel<<<grid1, 128, smem_u, s>>>(mapK, mapV, mapO, part, n, LH, g.H, g.w, n_sketch);
  } else if (g.d == 128 && use_umma) {      // no driver entry point for tensor maps / unaligned inputs: cp.async-fed tcgen05 kernel
    const size_t smem_u = (size_t)kUmmaStages * kUmmaStageBytes + 1024;
    cudaFuncSetAttribute(sketch_umma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_u);
    sketch_umma_kernel<<<grid1, 128, smem_u, s>>>(k_dense, v_dense, omega, part, n, LH, g.H, g.w, n_sketch);
  } else if (g.d == 128) {
    switch (MT) { DWKV_SKETCH_CASE(128, 1) DWKV_SKETCH_CASE(128, 2) DWKV_SKETCH_CASE(128, 3) DWKV_SKETCH_CASE(128, 4) DWKV_SKETCH_CASE(128, 5)
                  default: ok = false; }
  } else {
    switch (MT) { DWKV_SKETCH_CASE(64, 1) DWKV_SKETCH_CASE(64, 2) DWKV_SKETCH_CASE(64, 3) DWKV_SKETCH_CASE(64, 4) default: ok = false; }
  }
#undef DWKV_SKETCH_CASE
  if (!ok) return 0;
  const size_t smem2 = ((size_t)n_sketch * (g.d + 1) + n_sketch) * sizeof(float);
  const int items2 = 2 * (g.L / g.w) * g.H;
  if (g.d == 128) {
    cudaFuncSetAttribute(basis_svd_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem2);
    basis_svd_kernel<128><<<items2, 32 * std::min(n_sketch / 2, 32), smem2, s>>>(part, n_split, gK, gV, BK, BV, n_sketch, g.r, g.L, g.H, g.w);
  } else {
    cudaFuncSetAttribute(basis_svd_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem2);
    basis_svd_kernel<64><<<items2, 32 * std::min(n_sketch / 2, 32), smem2, s>>>(part, n_split, gK, gV, BK, BV, n_sketch, g.r, g.L, g.H, g.w);
  }
  return 2;
}

}  // namespace dwkv
