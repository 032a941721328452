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
// Split in two: the loads (one batch, issued as early as possible: under load a DRAM round trip costs several microseconds
// because it queues behind the chip's outstanding bulk copies) and the arithmetic.
template <int NKB, int D>
struct ProLoads {
  static constexpr int NKK = D / 16;
  static constexpr int JB = NKB < 4 ? NKB : 4;       // basis row chunks of the first load batch
  uint32_t qv[NKK][2], gv[NKK][2];
  uint32_t bw[JB][NKK][2];
};

struct SegPtrs {
  const __nv_bfloat16 *qhead, *gk, *Bk;               // first query head of the kv head, gate row, basis block
};
__device__ __forceinline__ SegPtrs seg_ptrs(const Scan3Params& p, const int seg, const int D) {
  const int b = seg / p.LH, lh = seg - b * p.LH;
  const int layer = p.layer0 + lh / p.H, h = lh % p.H;
  SegPtrs s;
  s.qhead = p.q + (((size_t)b * p.Lq + (p.Lq == 1 ? 0 : layer)) * (size_t)(p.H * p.G) + (size_t)h * p.G) * D;
  s.gk = p.gK + ((size_t)layer * p.H + h) * D;
  s.Bk = p.BK + ((size_t)(layer / p.w) * p.H + h) * (size_t)p.r * D;
  return s;
}

// L2 prefetch of everything the prologue of `seg` will read (q rows, gate row, basis block); called by the fetch cursor
// when it crosses into the segment, a few stages ahead of the compute side.
__device__ __forceinline__ void prefetch_segment(const Scan3Params& p, const int seg, const int D, const int lane) {
  const SegPtrs sp = seg_ptrs(p, seg, D);
  const int nq = (p.G * D * 2 + 127) / 128, ng = (D * 2 + 127) / 128, nb = (p.r * D * 2 + 127) / 128;
  for (int i = lane; i < nq + ng + nb; i += 32) {
    const char* a = i < nq ? (const char*)sp.qhead + 128 * i : i < nq + ng ? (const char*)sp.gk + 128 * (i - nq) : (const char*)sp.Bk + 128 * (i - nq - ng);
    asm volatile("prefetch.global.L2 [%0];" ::"l"(a));
  }
}

template <int NKB, int D, bool PAIR>
__device__ __forceinline__ void prologue_load(ProLoads<NKB, D>& pl, const Scan3Params& p, const int seg, const int lane) {
  constexpr int NKK = D / 16, JB = ProLoads<NKB, D>::JB;
  const int g = lane >> 2, t = lane & 3;
  const int hd = PAIR ? (g & 3) : g;
  const bool valid = hd < p.G;
  const SegPtrs sp = seg_ptrs(p, seg, D);
  const __nv_bfloat16* qrow = sp.qhead + (size_t)(valid ? hd : 0) * D;
#pragma unroll
  for (int kk = 0; kk < NKK; ++kk) {
    pl.qv[kk][0] = valid ? ldg32(qrow + 16 * kk + 2 * t) : 0u;
    pl.qv[kk][1] = valid ? ldg32(qrow + 16 * kk + 8 + 2 * t) : 0u;
    pl.gv[kk][0] = ldg32(sp.gk + 16 * kk + 2 * t);
    pl.gv[kk][1] = ldg32(sp.gk + 16 * kk + 8 + 2 * t);
  }
#pragma unroll
  for (int jb = 0; jb < JB; ++jb) {
    const int row = 8 * jb + g;
    const bool ok = row < p.r;
    const __nv_bfloat16* br = sp.Bk + (size_t)(ok ? row : 0) * D + 2 * t;
#pragma unroll
    for (int kk = 0; kk < NKK; ++kk) {
      pl.bw[jb][kk][0] = ok ? ldg32(br + 16 * kk) : 0u;
      pl.bw[jb][kk][1] = ok ? ldg32(br + 16 * kk + 8) : 0u;
    }
  }
}

template <int NKB, int D, bool PAIR, bool I8 = false>
__device__ __forceinline__ void prologue_compute(QRegs<NKB, D, PAIR>& q, const ProLoads<NKB, D>& pl, const Scan3Params& p, const int seg,
                                                 const int lane) {
  constexpr int NKK = D / 16, JB = ProLoads<NKB, D>::JB;
  const int g = lane >> 2, t = lane & 3;
  const uint32_t mA = (g < 4) ? 0xffffffffu : 0u;
  uint32_t af[NKK][4];
  float c[NKB][4];
#pragma unroll
  for (int jj = 0; jj < NKB; ++jj) c[jj][0] = c[jj][1] = c[jj][2] = c[jj][3] = 0.f;
#pragma unroll
  for (int kk = 0; kk < NKK; ++kk) {
    const float2 x0 = bf2(pl.qv[kk][0]), x2 = bf2(pl.qv[kk][1]), g0 = bf2(pl.gv[kk][0]), g2 = bf2(pl.gv[kk][1]);
    split_bf16x2(x0.x * g0.x, x0.y * g0.y, af[kk][0], af[kk][1]);
    split_bf16x2(x2.x * g2.x, x2.y * g2.y, af[kk][2], af[kk][3]);
    if constexpr (PAIR) {
      q.qr[kk][0] = pl.qv[kk][0] & mA; q.qr[kk][1] = pl.qv[kk][0] & ~mA; q.qr[kk][2] = pl.qv[kk][1] & mA; q.qr[kk][3] = pl.qv[kk][1] & ~mA;
    } else {
      q.qr[kk >> 1][kk & 1] = pl.qv[kk][0]; q.qr[kk >> 1][2 + (kk & 1)] = pl.qv[kk][1];
    }
    float sum = (x0.x + x0.y) + (x2.x + x2.y);
    sum += __shfl_xor_sync(kFull, sum, 1);
    sum += __shfl_xor_sync(kFull, sum, 2);
    q.qbias[kk] = -136.f * sum;
  }
#pragma unroll
  for (int jb = 0; jb < JB; ++jb) {
#pragma unroll
    for (int kk = 0; kk < NKK; ++kk) mma16(c[jb], af[kk][0], af[kk][1], af[kk][2], af[kk][3], pl.bw[jb][kk][0], pl.bw[jb][kk][1]);
  }
  if constexpr (NKB > JB) {      // remaining basis row chunks (basis rank > 32): a second load batch
    const SegPtrs sp = seg_ptrs(p, seg, D);
    uint32_t bw2[NKB - JB][NKK][2];
#pragma unroll
    for (int jb = 0; jb < NKB - JB; ++jb) {
      const int row = 8 * (JB + jb) + g;
      const bool ok = row < p.r;
      const __nv_bfloat16* br = sp.Bk + (size_t)(ok ? row : 0) * D + 2 * t;
#pragma unroll
      for (int kk = 0; kk < NKK; ++kk) {
        bw2[jb][kk][0] = ok ? ldg32(br + 16 * kk) : 0u;
        bw2[jb][kk][1] = ok ? ldg32(br + 16 * kk + 8) : 0u;
      }
    }
#pragma unroll
    for (int jb = 0; jb < NKB - JB; ++jb) {
#pragma unroll
      for (int kk = 0; kk < NKK; ++kk) mma16(c[JB + jb], af[kk][0], af[kk][1], af[kk][2], af[kk][3], bw2[jb][kk][0], bw2[jb][kk][1]);
    }
  }
#pragma unroll
  for (int jj = 0; jj < NKB; ++jj) {
    uint32_t hi, lo;
    if constexpr (I8) split_f16x2((c[jj][0] + c[jj][2]) * p.cscale, (c[jj][1] + c[jj][3]) * p.cscale, hi, lo);   // f16 score MMAs
    else split_bf16x2((c[jj][0] + c[jj][2]) * p.cscale, (c[jj][1] + c[jj][3]) * p.cscale, hi, lo);
    if constexpr (PAIR) {
      q.qa[jj][0] = hi & mA; q.qa[jj][1] = lo & mA; q.qa[jj][2] = hi & ~mA; q.qa[jj][3] = lo & ~mA;
    } else {
      q.qa[jj][0] = hi; q.qa[jj][1] = lo;
    }
  }
}

template <int NKB, int D>
__device__ __forceinline__ void state_reset(State<NKB, D>& st, const float zero) {
  st.m = -INFINITY; st.thr = -INFINITY; st.l = 0.f;
  // (zero comes from a kernel parameter: a value the compiler cannot fold, so the quad stays in four registers of its own instead of
  //  being rebuilt before every MMA chain)
  st.cq[0] = st.cq[1] = st.cq[2] = st.cq[3] = zero;
#pragma unroll
  for (int i = 0; i < NKB; ++i) st.acc[i][0] = st.acc[i][1] = st.acc[i][2] = st.acc[i][3] = 0.f;
#pragma unroll
  for (int c = 0; c < D / 16; ++c) st.eacc[c][0] = st.eacc[c][1] = st.eacc[c][2] = st.eacc[c][3] = 0.f;
}

// Write this warp's partial of a segment: per query head (m, l, a[r], e[d]) fp32. PAIR: the tile-A and tile-B rows of a
// head are merged by log-sum-exp first.
template <int NKB, int D, bool PAIR>
__device__ __forceinline__ void flush_partial(const State<NKB, D>& st, const Scan3Params& p, float* rec, const int lane) {
  constexpr int NG = D / 16;
  const int g = lane >> 2, t = lane & 3;
  const int PR = 2 + p.r + D;
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

template <int NK, bool RESID, int NKB, int D, bool PAIR, bool I8>
__device__ __forceinline__ void process_stage(State<NKB, D>& st, const uint32_t sp, const int n, const int ntok, const int lane,
                                              const QRegs<NKB, D, PAIR>& q, const float cscale) {
  constexpr int SUBTOK = RESID ? 16 : 32;
  constexpr int NBK = (NK + 3) / 4;      // 8-bit planes: exponent bytes per slot and 32-column block
  constexpr int SB1 = I8 ? (RESID ? 2 * (NK * 128 + NBK * 16) + 20 * D : 2 * (NK * 256 + NBK * 32)) : (RESID ? NK * 512 + 20 * D : NK * 1024);
  // only the last sub-block of a stage can be ragged (the end of a unit): the full ones run without the per-score slot checks
  const int nfull = (ntok >= n * SUBTOK) ? n : n - 1;
  if constexpr (RESID || NK > 2) {
#pragma unroll 1
    for (int sb = 0; sb < nfull; ++sb) process_sub<NK, RESID, NKB, D, PAIR, I8, false>(st, sp + sb * SB1, SUBTOK, lane, q, cscale);
  } else {   // two independent sub-blocks per iteration: more instruction-level parallelism for the 2 warps per scheduler
    int sb = 0;
#pragma unroll 1
    for (; sb + 2 <= nfull; sb += 2) {
      process_sub<NK, RESID, NKB, D, PAIR, I8, false>(st, sp + sb * SB1, SUBTOK, lane, q, cscale);
      process_sub<NK, RESID, NKB, D, PAIR, I8, false>(st, sp + (sb + 1) * SB1, SUBTOK, lane, q, cscale);
    }
    if (sb < nfull) process_sub<NK, RESID, NKB, D, PAIR, I8, false>(st, sp + sb * SB1, SUBTOK, lane, q, cscale);
  }
  if (nfull < n) process_sub<NK, RESID, NKB, D, PAIR, I8, true>(st, sp + nfull * SB1, ntok - nfull * SUBTOK, lane, q, cscale);
}

template <int NKB, int D, bool PAIR, bool I8>
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
  // Consecutive slices go to different SMs. With equal-length sequences slice k and slice k + grid sit at the same phase of their
  // segment / sequence, so an SM runs eight slices of the same class mix: good for the instruction cache, and measured faster on
  // every batched shape than a rotated numbering. The one exception the host selects (p.rot = 53): all layers of a single sequence
  // with interleaved classes, where all slices look alike and the rotation evens out the SMs (170.5 -> 164.3 us at 64K).
  const int gw = warp * (int)gridDim.x + (int)(((int)blockIdx.x + p.rot * warp) % (int)gridDim.x);
  int4 ws = make_int4(0, 0, 0, 0), we = ws;
  bool active = gw < p.n_slices;
  if (active) {
    ws = __ldg(p.wentry + gw); we = __ldg(p.wentry + gw + 1);
    active = !(ws.x == we.x && ws.y == we.y && ws.z == we.z);
  }
  if (!active) { cudaGridDependencySynchronize(); return; }

  State<NKB, D> st;
  int cur_seg = -1, slot_next = 0, n_entered = 0;
  const int PRG = p.G * (2 + p.r + D);
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
    f_sb1 = I8 ? (fl ? 2 * (nk * 128 + ((nk + 3) >> 2) * 16) + 20 * D : 2 * (nk * 256 + ((nk + 3) >> 2) * 32)) : (fl ? nk * 512 + 20 * D : nk * 1024);
    f_subtok = fl ? 16 : 32;
    f_ntok = un.ntok;
    f_nsub = (un.ntok + f_subtok - 1) / f_subtok;
    f_per = SLOT / f_sb1;
    if (!fl && nk <= 2) f_per &= ~1;  // even stages: the unflagged low-rank classes are processed two sub-blocks at a time
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
        if (f_seg < p.n_segs) prefetch_segment(p, f_seg, D, lane);
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
  QRegs<NKB, D, PAIR> q;
  {   // first segment: loads ahead of the ring fills in the memory queues, arithmetic while the ring fills land.
      // (Issuing the fills before the grid dependency resolves -- they read the plan and cache pages only -- was measured: neutral for
      //  all-layer calls, 1-3 % slower for per-layer calls, because q then queues behind 32 MB of bulk copies)
    ProLoads<NKB, D> pl;
    cudaGridDependencySynchronize();
    prologue_load<NKB, D, PAIR>(pl, p, ws.x, lane);
#pragma unroll 1
    for (int k = 0; k < NS; ++k) fetch_one(k);
    __syncwarp();
    prologue_compute<NKB, D, PAIR, I8>(q, pl, p, ws.x, lane);
    state_reset<NKB, D>(st, p.zero);
  }

  // ---- compute stream ----------------------------------------------------------------------------------------------------
  int k_c = 0;
  cur_seg = ws.x; slot_next = ws.w; n_entered = 1;
  uint32_t phase = 0u;
  while (true) {
    const uint4 dsc = lds128(descs + 16 * k_c);
    const int n = (int)(dsc.x >> 16);
    if (n == 0) break;
    const int seg = (int)dsc.z;
    if (seg != cur_seg) {
      ProLoads<NKB, D> pl;
      prologue_load<NKB, D, PAIR>(pl, p, seg, lane);       // L2 hits: the fetch cursor prefetched them when it crossed over
      float* rec = p.part + (size_t)slot_next * (size_t)PRG;
      flush_partial<NKB, D, PAIR>(st, p, rec, lane);
      slot_next = __ldg(p.pstart + seg);       // a segment entered inside a slice is entered at its start: its first slot
      prologue_compute<NKB, D, PAIR, I8>(q, pl, p, seg, lane);
      state_reset<NKB, D>(st, p.zero);
      cur_seg = seg;
      ++n_entered;
    }
    mbar_wait(bars + 8 * k_c, (phase >> k_c) & 1u);
    phase ^= 1u << k_c;
    const uint32_t sp = ring + k_c * SLOT;
    const int ntok = (int)dsc.y;
    switch (dsc.x & 0xffffu) {
      case 0x001: process_stage<1, false, NKB, D, PAIR, I8>(st, sp, n, ntok, lane, q, p.cscale); break;
      case 0x101: process_stage<1, true, NKB, D, PAIR, I8>(st, sp, n, ntok, lane, q, p.cscale); break;
      case 0x002: process_stage<2, false, NKB, D, PAIR, I8>(st, sp, n, ntok, lane, q, p.cscale); break;
      case 0x102: process_stage<2, true, NKB, D, PAIR, I8>(st, sp, n, ntok, lane, q, p.cscale); break;
      case 0x003: if constexpr (NKB >= 3) process_stage<3, false, NKB, D, PAIR, I8>(st, sp, n, ntok, lane, q, p.cscale); break;
      case 0x103: if constexpr (NKB >= 3) process_stage<3, true, NKB, D, PAIR, I8>(st, sp, n, ntok, lane, q, p.cscale); break;
      case 0x004: if constexpr (NKB >= 4) process_stage<4, false, NKB, D, PAIR, I8>(st, sp, n, ntok, lane, q, p.cscale); break;
      case 0x104: if constexpr (NKB >= 4) process_stage<4, true, NKB, D, PAIR, I8>(st, sp, n, ntok, lane, q, p.cscale); break;
      case 0x006: if constexpr (NKB >= 6) process_stage<6, false, NKB, D, PAIR, I8>(st, sp, n, ntok, lane, q, p.cscale); break;
      case 0x106: if constexpr (NKB >= 6) process_stage<6, true, NKB, D, PAIR, I8>(st, sp, n, ntok, lane, q, p.cscale); break;
      case 0x008: if constexpr (NKB >= 8) process_stage<8, false, NKB, D, PAIR, I8>(st, sp, n, ntok, lane, q, p.cscale); break;
      case 0x108: if constexpr (NKB >= 8) process_stage<8, true, NKB, D, PAIR, I8>(st, sp, n, ntok, lane, q, p.cscale); break;
      default: break;   // unsupported rank (the host refuses these configurations)
    }
    __syncwarp();
    fetch_one(k_c);      // refill the slot that was just consumed
    __syncwarp();
    k_c = (k_c + 1 == NS) ? 0 : k_c + 1;
  }
  flush_partial<NKB, D, PAIR>(st, p, p.part + (size_t)slot_next * (size_t)PRG, lane);
  if (p.stamps && lane == 0) {       // measurement aid: when did this warp finish (planner cost-model fits)
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    p.stamps[gw] = t;
    p.stamps[p.n_slices + gw] = (unsigned long long)n_entered;     // segments this slice touched
  }
}

// cudaFuncSetAttribute is per device: remember which devices this instance has been prepared on
template <int NKB, int D, bool PAIR, bool I8>
cudaError_t launch_instance(const Scan3Params& p, int n_sms, cudaStream_t s) {
  const int smem = kWarps * kWarpSmem;
  static bool attr_set[64] = {};
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= 64 || !attr_set[dev]) {
    e = cudaFuncSetAttribute(scan3_kernel<NKB, D, PAIR, I8>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    if (dev >= 0 && dev < 64) attr_set[dev] = true;
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(n_sms);
  cfg.blockDim = dim3(kWarps * 32);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = s;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, scan3_kernel<NKB, D, PAIR, I8>, p);
}

// returns false if no instance exists for the basis rank; *err receives the launch status otherwise
template <int D, bool PAIR>
bool launch_by_rank(const Scan3Params& p, int n_sms, cudaStream_t s, cudaError_t* err) {
  const int nkb = (p.r + 15) / 16 * 2;      // basis rank / 8 rounded up to even
  switch (nkb) {
    case 2: *err = launch_instance<2, D, PAIR, false>(p, n_sms, s); return true;
    case 4: *err = launch_instance<4, D, PAIR, false>(p, n_sms, s); return true;
    case 6: *err = launch_instance<6, D, PAIR, false>(p, n_sms, s); return true;
    case 8: *err = launch_instance<8, D, PAIR, false>(p, n_sms, s); return true;
  }
  return false;
}
// 8-bit coefficient planes (one exponent byte per 32-column block of a token vector)
template <int D, bool PAIR>
bool launch_by_rank_i8(const Scan3Params& p, int n_sms, cudaStream_t s, cudaError_t* err) {
  const int nkb = (p.r + 15) / 16 * 2;
  switch (nkb) {
    case 2: *err = launch_instance<2, D, PAIR, true>(p, n_sms, s); return true;
    case 4: *err = launch_instance<4, D, PAIR, true>(p, n_sms, s); return true;
    case 6: *err = launch_instance<6, D, PAIR, true>(p, n_sms, s); return true;
    case 8: *err = launch_instance<8, D, PAIR, true>(p, n_sms, s); return true;
  }
  return false;
}

}  // namespace s3
}  // namespace dwkv
