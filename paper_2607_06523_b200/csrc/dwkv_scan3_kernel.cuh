// dwkv_scan3_kernel.cuh -- persistent fused decode kernel: fetch cursor, segment prologue (a1), stage dispatch (a2), partials.
#pragma once
#include "dwkv_scan3_sub.cuh"

namespace dwkv {
namespace s3 {

__device__ __forceinline__ uint32_t ldg32(const __nv_bfloat16* p) { return __ldg(reinterpret_cast<const uint32_t*>(p)); }
__device__ __forceinline__ float2 bf2(uint32_t w) { return make_float2(__uint_as_float(w << 16), __uint_as_float(w & 0xffff0000u)); }

// a1: q~ = cscale * BK[m,h] . (gK[l,h] * q) for the rows of this lane, straight into A-fragment registers; also the raw-q
// fragments and code-offset biases of the residual-K term. gK*q is exact in fp32 and split into hi + lo bf16 (exact);
// BK is bf16, so the tensor-core products are exact and only the fp32 accumulation rounds.
template <int NKB, int D, bool PAIR>
__device__ __forceinline__ void segment_prologue(QRegs<NKB, D, PAIR>& q, const Scan3Params& p, const int seg, const int lane) {
  const int g = lane >> 2, t = lane & 3;
  const int b = seg / p.LH, lh = seg - b * p.LH;
  const int layer = p.layer0 + lh / p.H, h = lh % p.H;
  const int hd = PAIR ? (g & 3) : g;
  const bool valid = hd < p.G;
  const uint32_t mA = (g < 4) ? 0xffffffffu : 0u;
  const __nv_bfloat16* qrow = p.q + (((size_t)b * p.Lq + (p.Lq == 1 ? 0 : layer)) * (size_t)(p.H * p.G) + (size_t)h * p.G + (valid ? hd : 0)) * D;
  const __nv_bfloat16* gk = p.gK + ((size_t)layer * p.H + h) * D;
  const __nv_bfloat16* Bk = p.BK + ((size_t)(layer / p.w) * p.H + h) * (size_t)p.r * D;
  float c[NKB][4];
#pragma unroll
  for (int jj = 0; jj < NKB; ++jj) c[jj][0] = c[jj][1] = c[jj][2] = c[jj][3] = 0.f;
#pragma unroll
  for (int kk = 0; kk < D / 16; ++kk) {
    const uint32_t q0 = valid ? ldg32(qrow + 16 * kk + 2 * t) : 0u, q2 = valid ? ldg32(qrow + 16 * kk + 8 + 2 * t) : 0u;
    const float2 g0 = bf2(ldg32(gk + 16 * kk + 2 * t)), g2 = bf2(ldg32(gk + 16 * kk + 8 + 2 * t));
    const float2 x0 = bf2(q0), x2 = bf2(q2);
    uint32_t a0, a1, a2, a3;
    split_bf16x2(x0.x * g0.x, x0.y * g0.y, a0, a1);
    split_bf16x2(x2.x * g2.x, x2.y * g2.y, a2, a3);
#pragma unroll
    for (int jj = 0; jj < NKB; ++jj) {
      const int row = 8 * jj + g;
      const bool ok = row < p.r;
      const __nv_bfloat16* br = Bk + (size_t)(ok ? row : 0) * D + 16 * kk + 2 * t;
      const uint32_t b0 = ok ? ldg32(br) : 0u, b1 = ok ? ldg32(br + 8) : 0u;
      mma16(c[jj], a0, a1, a2, a3, b0, b1);
    }
    if constexpr (PAIR) {
      q.qr[kk][0] = q0 & mA; q.qr[kk][1] = q2 & mA; q.qr[kk][2] = q0 & ~mA; q.qr[kk][3] = q2 & ~mA;
    } else {
      q.qr[kk][0] = q0; q.qr[kk][1] = q2;
    }
    float sum = (x0.x + x0.y) + (x2.x + x2.y);
    sum += __shfl_xor_sync(kFull, sum, 1);
    sum += __shfl_xor_sync(kFull, sum, 2);
    q.qbias[kk] = -136.f * sum;
  }
#pragma unroll
  for (int jj = 0; jj < NKB; ++jj) {
    uint32_t hi, lo;
    split_bf16x2((c[jj][0] + c[jj][2]) * p.cscale, (c[jj][1] + c[jj][3]) * p.cscale, hi, lo);
    if constexpr (PAIR) {
      q.qa[jj][0] = hi & mA; q.qa[jj][1] = lo & mA; q.qa[jj][2] = hi & ~mA; q.qa[jj][3] = lo & ~mA;
    } else {
      q.qa[jj][0] = hi; q.qa[jj][1] = lo;
    }
  }
}

template <int NKB, int D>
__device__ __forceinline__ void state_reset(State<NKB, D>& st) {
  st.m = -INFINITY; st.thr = -INFINITY; st.l = 0.f;
#pragma unroll
  for (int i = 0; i < NKB; ++i) st.acc[i][0] = st.acc[i][1] = st.acc[i][2] = st.acc[i][3] = 0.f;
#pragma unroll
  for (int c = 0; c < D / 16; ++c) st.eacc[c][0] = st.eacc[c][1] = st.eacc[c][2] = st.eacc[c][3] = 0.f;
}

// Write this warp's partial of a segment: per query head (m, l, a[r], e[d]) fp32. PAIR: the tile-A and tile-B rows of a
// head are merged by log-sum-exp first.
template <int NKB, int D, bool PAIR>
__device__ __forceinline__ void flush_partial(const State<NKB, D>& st, const Scan3Params& p, const int slot, const int lane) {
  constexpr int NG = D / 16;
  const int g = lane >> 2, t = lane & 3;
  const int PR = 2 + p.r + D;
  float* rec = p.part + (size_t)slot * (size_t)(p.G * PR);
  float l = st.l;
  l += __shfl_xor_sync(kFull, l, 1);
  l += __shfl_xor_sync(kFull, l, 2);
  float w = 1.f, ms = st.m;
  if constexpr (PAIR) {
    const float mp = __shfl_xor_sync(kFull, st.m, 16);
    ms = fmaxf(st.m, mp);
    w = (st.m == -INFINITY) ? 0.f : ex2(st.m - ms);
    l *= w;
    l += __shfl_xor_sync(kFull, l, 16);
  }
  const int hd = g;                       // PAIR: lanes g < 4 write head g; FULL: lane row g = head g
  const bool wr = PAIR ? (g < 4 && g < p.G) : (g < p.G);
  if (wr && t == 0) *reinterpret_cast<float2*>(rec + hd * PR) = make_float2(ms, l);
#pragma unroll
  for (int i = 0; i < NKB; ++i) {
    float a0 = (st.acc[i][0] + st.acc[i][2]) * w, a1 = (st.acc[i][1] + st.acc[i][3]) * w;
    if constexpr (PAIR) {
      a0 += __shfl_xor_sync(kFull, a0, 16);
      a1 += __shfl_xor_sync(kFull, a1, 16);
    }
    if (wr && 8 * i + 2 * t < p.r) *reinterpret_cast<float2*>(rec + hd * PR + 2 + 8 * i + 2 * t) = make_float2(a0, a1);
  }
  // e^T[channel][column n]: column n belongs to row n (lane 4n); PAIR: columns n and n + 4 are the two tiles of head n
  const float w0 = __shfl_sync(kFull, w, 8 * t), w1 = __shfl_sync(kFull, w, 8 * t + 4);
#pragma unroll
  for (int grp = 0; grp < NG; ++grp) {
    float v0 = st.eacc[grp][0] * w0, v1 = st.eacc[grp][1] * w1, v2 = st.eacc[grp][2] * w0, v3 = st.eacc[grp][3] * w1;
    if constexpr (PAIR) {
      v0 += __shfl_xor_sync(kFull, v0, 2); v1 += __shfl_xor_sync(kFull, v1, 2);
      v2 += __shfl_xor_sync(kFull, v2, 2); v3 += __shfl_xor_sync(kFull, v3, 2);
    }
    const int h0 = 2 * t, h1 = 2 * t + 1;
    const bool ok = PAIR ? (t < 2) : true;
    if (ok && h0 < p.G) {
      rec[h0 * PR + 2 + p.r + 16 * grp + g] = v0;
      rec[h0 * PR + 2 + p.r + 16 * grp + 8 + g] = v2;
    }
    if (ok && h1 < p.G) {
      rec[h1 * PR + 2 + p.r + 16 * grp + g] = v1;
      rec[h1 * PR + 2 + p.r + 16 * grp + 8 + g] = v3;
    }
  }
}

template <int NK, bool RESID, int NKB, int D, bool PAIR>
__device__ __forceinline__ void process_stage(State<NKB, D>& st, const uint32_t sp, const int n, const int ntok, const int lane,
                                              const QRegs<NKB, D, PAIR>& q, const float cscale) {
  constexpr int SUBTOK = RESID ? 16 : 32;
  constexpr int SB1 = RESID ? NK * 512 + 20 * D : NK * 1024;
  if constexpr (RESID || NK > 2) {
#pragma unroll 1
    for (int sb = 0; sb < n; ++sb) process_sub<NK, RESID, NKB, D, PAIR>(st, sp + sb * SB1, ntok - sb * SUBTOK, lane, q, cscale);
  } else {   // two independent sub-blocks per iteration: more instruction-level parallelism for the 2 warps per scheduler
    int sb = 0;
#pragma unroll 1
    for (; sb + 2 <= n; sb += 2) {
      process_sub<NK, RESID, NKB, D, PAIR>(st, sp + sb * SB1, ntok - sb * SUBTOK, lane, q, cscale);
      process_sub<NK, RESID, NKB, D, PAIR>(st, sp + (sb + 1) * SB1, ntok - (sb + 1) * SUBTOK, lane, q, cscale);
    }
    if (sb < n) process_sub<NK, RESID, NKB, D, PAIR>(st, sp + sb * SB1, ntok - sb * SUBTOK, lane, q, cscale);
  }
}

template <int NKB, int D, bool PAIR>
__global__ void __launch_bounds__(kWarps * 32, 1) scan3_kernel(const __grid_constant__ Scan3Params p) {
  using RG = Ring<NKB, D>;
  constexpr int SLOT = RG::SLOT, NS = RG::NS;
  extern __shared__ __align__(128) uint8_t smem[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t ring = smem_u32(smem) + warp * kWarpSmem;
  const uint32_t descs = ring + kRingBytes, bars = descs + kMaxSlots * 16;
  if (lane == 0) {
    for (int s = 0; s < NS; ++s) mbar_init(bars + 8 * s, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  __syncwarp();
  const int gw = warp * gridDim.x + blockIdx.x;      // consecutive slices of the linear order go to different SMs

  if (gw >= p.n_slices) return;
  const int4 ws = __ldg(p.wentry + gw), we = __ldg(p.wentry + gw + 1);
  if (ws.x == we.x && ws.y == we.y && ws.z == we.z) return;

  // ---- fetch cursor (warp-uniform) over the slice [ws, we) of the linear order ----------------------------------------------
  int f_seg = ws.x, f_u = ws.y, f_sub = ws.z;
  int f_b = f_seg / p.LH, f_lh = f_seg - f_b * p.LH;
  int f_ubeg = __ldg(p.ustart + f_b), f_uend = __ldg(p.ustart + f_b + 1);
  bool f_on = true;
  int f_code = 0, f_nsub = 0, f_per = 0, f_sb1 = 0, f_subtok = 0, f_ntok = 0;
  const uint8_t* f_base = nullptr;
  auto unit_setup = [&]() {
    const Unit un = load_unit(p.units + f_u);
    const int nk = un.rk >> 3, fl = un.cls & 1;
    f_code = nk | (fl << 8);
    f_sb1 = fl ? nk * 512 + 20 * D : nk * 1024;
    f_subtok = fl ? 16 : 32;
    f_ntok = un.ntok;
    f_nsub = (un.ntok + f_subtok - 1) / f_subtok;
    f_per = SLOT / f_sb1;
    if (f_per > 2) f_per &= ~1;       // even stages: the unflagged low-rank classes are processed two sub-blocks at a time
    f_base = p.arena + un.page_off + (size_t)(p.layer0 * p.H + f_lh) * kPageLhBytes + (size_t)un.blk0 * (size_t)(f_sb1 * (kBlockTok / f_subtok));
  };
  unit_setup();
  auto fetch_one = [&](const int k) {
    if (!f_on) {
      if (lane == 0) sts128(descs + 16 * k, 0, 0, 0, 0);
      return;
    }
    const int limit = (f_seg == we.x && f_u == we.y) ? we.z : f_nsub;
    const int n = min(f_per, limit - f_sub);
    if (lane == 0) {
      const int ntok = min(f_ntok - f_sub * f_subtok, n * f_subtok);
      sts128(descs + 16 * k, f_code | (n << 16), ntok, f_seg, 0);
      mbar_expect_tx(bars + 8 * k, (uint32_t)(n * f_sb1));
      bulk_g2s(ring + k * SLOT, f_base + (size_t)f_sub * f_sb1, (uint32_t)(n * f_sb1), bars + 8 * k);
    }
    f_sub += n;
    bool moved = false;
    if (f_sub == f_nsub) {
      f_sub = 0;
      ++f_u;
      moved = true;
      if (f_u == f_uend) {
        ++f_seg;
        if (++f_lh == p.LH) {
          f_lh = 0;
          ++f_b;
          f_ubeg = f_u;
          if (f_seg < p.n_segs) f_uend = __ldg(p.ustart + f_b + 1);
        } else {
          f_u = f_ubeg;
        }
      }
    }
    if (f_seg == we.x && f_u == we.y && f_sub == we.z) f_on = false;
    else if (moved) unit_setup();
  };
#pragma unroll 1
  for (int k = 0; k < NS; ++k) fetch_one(k);
  __syncwarp();

  // ---- compute stream ----------------------------------------------------------------------------------------------------
  State<NKB, D> st;
  QRegs<NKB, D, PAIR> q;
  int cur_seg = -1, k_c = 0, slot_next = ws.w;
  uint32_t phase = 0u;
  while (true) {
    const uint4 dsc = lds128(descs + 16 * k_c);
    const int n = (int)(dsc.x >> 16);
    if (n == 0) break;
    const int seg = (int)dsc.z;
    if (seg != cur_seg) {
      if (cur_seg >= 0) {
        flush_partial<NKB, D, PAIR>(st, p, slot_next, lane);
        slot_next = __ldg(p.pstart + seg);     // a segment entered inside a slice is entered at its start: its first slot
      }
      state_reset<NKB, D>(st);
      segment_prologue<NKB, D, PAIR>(q, p, seg, lane);
      cur_seg = seg;
    }
    mbar_wait(bars + 8 * k_c, (phase >> k_c) & 1u);
    phase ^= 1u << k_c;
    const uint32_t sp = ring + k_c * SLOT;
    const int ntok = (int)dsc.y;
    switch (dsc.x & 0xffffu) {
      case 0x001: process_stage<1, false, NKB, D, PAIR>(st, sp, n, ntok, lane, q, p.cscale); break;
      case 0x101: process_stage<1, true, NKB, D, PAIR>(st, sp, n, ntok, lane, q, p.cscale); break;
      case 0x002: process_stage<2, false, NKB, D, PAIR>(st, sp, n, ntok, lane, q, p.cscale); break;
      case 0x102: process_stage<2, true, NKB, D, PAIR>(st, sp, n, ntok, lane, q, p.cscale); break;
      case 0x003: if constexpr (NKB >= 3) process_stage<3, false, NKB, D, PAIR>(st, sp, n, ntok, lane, q, p.cscale); break;
      case 0x103: if constexpr (NKB >= 3) process_stage<3, true, NKB, D, PAIR>(st, sp, n, ntok, lane, q, p.cscale); break;
      case 0x004: if constexpr (NKB >= 4) process_stage<4, false, NKB, D, PAIR>(st, sp, n, ntok, lane, q, p.cscale); break;
      case 0x104: if constexpr (NKB >= 4) process_stage<4, true, NKB, D, PAIR>(st, sp, n, ntok, lane, q, p.cscale); break;
      case 0x006: if constexpr (NKB >= 6) process_stage<6, false, NKB, D, PAIR>(st, sp, n, ntok, lane, q, p.cscale); break;
      case 0x106: if constexpr (NKB >= 6) process_stage<6, true, NKB, D, PAIR>(st, sp, n, ntok, lane, q, p.cscale); break;
      case 0x008: if constexpr (NKB >= 8) process_stage<8, false, NKB, D, PAIR>(st, sp, n, ntok, lane, q, p.cscale); break;
      case 0x108: if constexpr (NKB >= 8) process_stage<8, true, NKB, D, PAIR>(st, sp, n, ntok, lane, q, p.cscale); break;
      default: break;   // unsupported rank (the host refuses these configurations)
    }
    __syncwarp();
    fetch_one(k_c);      // refill the slot that was just consumed
    __syncwarp();
    k_c = (k_c + 1 == NS) ? 0 : k_c + 1;
  }
  if (cur_seg >= 0) flush_partial<NKB, D, PAIR>(st, p, slot_next, lane);
}

template <int NKB, int D, bool PAIR>
void launch_instance(const Scan3Params& p, int n_sms, cudaStream_t s) {
  const int smem = kWarps * kWarpSmem;
  static bool attr_set = false;
  if (!attr_set) {
    cudaFuncSetAttribute(scan3_kernel<NKB, D, PAIR>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    attr_set = true;
  }
  scan3_kernel<NKB, D, PAIR><<<n_sms, kWarps * 32, smem, s>>>(p);
}

template <int D, bool PAIR>
bool launch_by_rank(const Scan3Params& p, int n_sms, cudaStream_t s) {
  const int nkb = (p.r + 15) / 16 * 2;      // basis rank / 8 rounded up to even
  switch (nkb) {
    case 2: launch_instance<2, D, PAIR>(p, n_sms, s); return true;
    case 4: launch_instance<4, D, PAIR>(p, n_sms, s); return true;
    case 6: launch_instance<6, D, PAIR>(p, n_sms, s); return true;
    case 8: launch_instance<8, D, PAIR>(p, n_sms, s); return true;
  }
  return false;
}

}  // namespace s3
}  // namespace dwkv
