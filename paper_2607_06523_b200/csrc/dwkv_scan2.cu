// dwkv_scan2.cu -- split-T scan, persistent form.
//
// One launch covers every class of the step. The grid is one CTA of 16 warps per SM; every WARP owns a contiguous,
// byte-balanced slice of the item list (item = (unit, layer, kv head), host-planned in `wstart`) and streams it
// through a private shared-memory ring filled by cp.async.bulk (TMA engine, 1-D, no tensor map) with one mbarrier
// per stage: registers hold no prefetched data, so the bytes in flight per SM are set by the ring (13.5 KB x 16 warps)
// and not by occupancy. A stage is one sub-block (32 slots, or 16 slots of a flagged class) in fragment-native order
// (dwkv_layout.cuh), read back with conflict-free vector LDS straight into mma.sync operand registers.
// Softmax uses a lazily updated reference m_ref: the score MMA starts from C = -m_ref, so p = 2^(s - m_ref) needs no
// subtraction, and accumulators are rescaled only when a score exceeds m_ref by more than 2^8.
#include "dwkv_internal.h"
#include "dwkv_mma.cuh"

namespace dwkv {
namespace {
using namespace dwkv::dev;

constexpr int kWarps = 16;
constexpr int kRing = 13824;       // ring bytes per warp (3 stages of the 4.5 KB flagged r=32 sub-block)
constexpr int kMaxStages = 8;
constexpr float kLazy = 8.0f;      // rescale when a score exceeds the reference by more than this (log2 units)

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
               "l"(src), "r"(bytes), "r"(bar)
               : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  do {
    asm volatile(
        "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
  } while (!ok);
}

__device__ __forceinline__ uint4 lds128(uint32_t a) {
  uint4 r;
  asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "r"(a));
  return r;
}
__device__ __forceinline__ uint2 lds64(uint32_t a) {
  uint2 r;
  asm volatile("ld.shared.v2.u32 {%0,%1}, [%2];" : "=r"(r.x), "=r"(r.y) : "r"(a));
  return r;
}
// full-quad forms: the A operand carries explicit zero registers for rows 8..15 and the accumulator keeps its (always
// zero) rows 8..15, so no scratch outputs and no per-call zero materialisation are needed.
__device__ __forceinline__ void mma16816q(float (&d)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  asm("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
      : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
      : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}

__device__ __forceinline__ Unit load_unit(const Unit* u) {
  const uint4 a = __ldg(reinterpret_cast<const uint4*>(u));
  const uint4 b = __ldg(reinterpret_cast<const uint4*>(u) + 1);
  Unit r;
  r.page_off = (int64_t)(((uint64_t)a.y << 32) | a.x);
  r.blk0 = (int32_t)a.z; r.nblk = (int32_t)a.w;
  r.ntok = (int32_t)b.x; r.cls = (int16_t)(b.y & 0xffff); r.b = (int16_t)(b.y >> 16);
  r.epart = (int32_t)b.z; r.rk = (int32_t)b.w;
  return r;
}

template <int NK, bool RESID, int D>
struct Geo {
  static constexpr int TB = RESID ? 2 : 4;
  static constexpr int SUBTOK = 8 * TB;
  static constexpr int COEF = NK * 128 * TB;                      // bytes of [K coef] (= [V coef])
  static constexpr int SB = 2 * COEF + (RESID ? 20 * D : 0);      // stage bytes = one sub-block
  static constexpr int NS = (kRing / SB) < kMaxStages ? ((kRing / SB) < 1 ? 1 : (kRing / SB)) : kMaxStages;
  static constexpr int NG = D / 16;
  static constexpr int NE = RESID ? D / 8 : 1;
};

template <int NK, bool RESID, int D>
struct State {
  float m, l;
  float acc[NK][4];                                  // rows 8..15 (acc[i][2..3]) stay zero
  float eacc[Geo<NK, RESID, D>::NE][2];
};

// Query-side operands of one item, in MMA A-fragment order (rows 8..15 explicit zeros).
template <int NK, bool RESID, int D>
struct QFrag {
  static constexpr int NP = (NK + 1) / 2;            // k16 steps over the rank columns
  uint32_t hi[NP][4];                                // NK == 1: the single quad is [hi | lo]
  uint32_t lo[NP][4];                                // odd NK: last hi quad is [hi_last | lo_last], last lo quad unused
  uint32_t qa[RESID ? D / 16 : 1][2];
  float qbias[RESID ? D / 16 : 1];
};

// One stage (sub-block) from shared memory (32-bit shared address sp).
template <int NK, bool RESID, int D>
__device__ __forceinline__ void process_stage(State<NK, RESID, D>& st, const uint32_t sp, const int nv, const int lane,
                                              const bool first, const QFrag<NK, RESID, D>& qf, const float cscale) {
  using G = Geo<NK, RESID, D>;
  constexpr int TB = G::TB, NG = G::NG, NP = QFrag<NK, RESID, D>::NP;
  const int t = lane & 3;
  uint32_t kw[NK][TB], vw[NK][TB];
#pragma unroll
  for (int i = 0; i < NK; ++i) {
    if constexpr (TB == 4) {
      const uint4 a = lds128(sp + i * 512 + lane * 16);
      const uint4 b = lds128(sp + G::COEF + i * 512 + lane * 16);
      kw[i][0] = a.x; kw[i][1] = a.y; kw[i][2] = a.z; kw[i][3] = a.w;
      vw[i][0] = b.x; vw[i][1] = b.y; vw[i][2] = b.z; vw[i][3] = b.w;
    } else {
      const uint2 a = lds64(sp + i * 256 + lane * 8);
      const uint2 b = lds64(sp + G::COEF + i * 256 + lane * 8);
      kw[i][0] = a.x; kw[i][1] = a.y;
      vw[i][0] = b.x; vw[i][1] = b.y;
    }
  }
  // ---- scores relative to the reference: s' = q~ . cK - m_ref ------------------------------------------------------
  const float cinit = first ? 0.f : -st.m;
  float s[TB][4];
#pragma unroll
  for (int j = 0; j < TB; ++j) {
    s[j][0] = cinit; s[j][1] = cinit; s[j][2] = 0.f; s[j][3] = 0.f;
#pragma unroll
    for (int pi = 0; pi < NP; ++pi) {
      const int i0 = 2 * pi, i1 = (2 * pi + 1 < NK) ? 2 * pi + 1 : 2 * pi;
      mma16816q(s[j], qf.hi[pi], kw[i0][j], kw[i1][j]);              // odd tail: A = [hi | lo], B = [cK | cK]
      if (2 * pi + 1 < NK) mma16816q(s[j], qf.lo[pi], kw[i0][j], kw[i1][j]);
    }
  }
  // ---- residual-K term: integer-code dot on the tensor cores, fp32 group scales afterwards -------------------------
  if constexpr (RESID) {
    const uint32_t codeK = sp + 2 * G::COEF;
    const uint32_t scaleK = codeK + 8 * D;
#pragma unroll
    for (int j = 0; j < TB; ++j) {
      uint32_t w[D / 32], sc[NG];
      if constexpr (D == 128) {
        const uint4 c4 = lds128(codeK + j * 4 * D + lane * 16);
        w[0] = c4.x; w[1] = c4.y; w[2] = c4.z; w[3] = c4.w;
        const uint4 s0 = lds128(scaleK + j * D + t * 32);
        const uint4 s1 = lds128(scaleK + j * D + t * 32 + 16);
        sc[0] = s0.x; sc[1] = s0.y; sc[2] = s0.z; sc[3] = s0.w; sc[4] = s1.x; sc[5] = s1.y; sc[6] = s1.z; sc[7] = s1.w;
      } else {
        const uint2 c2 = lds64(codeK + j * 4 * D + lane * 8);
        w[0] = c2.x; w[1] = c2.y;
        const uint4 s0 = lds128(scaleK + j * D + t * 16);
        sc[0] = s0.x; sc[1] = s0.y; sc[2] = s0.z; sc[3] = s0.w;
      }
      float sr0 = 0.f, sr1 = 0.f;
#pragma unroll
      for (int grp = 0; grp < NG; ++grp) {
        float c0 = qf.qbias[grp], c1 = qf.qbias[grp];  // -136 * sum_i q_i cancels the offset of the biased codes
        const int q = 2 * grp;
        mma16816(c0, c1, qf.qa[grp][0], qf.qa[grp][1], nib_to_bf16x2_biased(w[q >> 2], q & 3),
                 nib_to_bf16x2_biased(w[q >> 2], (q & 3) + 1));
        const float2 f = h2f2(sc[grp]);
        sr0 = fmaf(c0, f.x, sr0);
        sr1 = fmaf(c1, f.y, sr1);
      }
      s[j][0] = fmaf(cscale, sr0, s[j][0]);
      s[j][1] = fmaf(cscale, sr1, s[j][1]);
    }
  }
  if (nv < G::SUBTOK) {   // ragged tail
#pragma unroll
    for (int j = 0; j < TB; ++j) {
      if (8 * j + 2 * t >= nv) s[j][0] = -INFINITY;
      if (8 * j + 2 * t + 1 >= nv) s[j][1] = -INFINITY;
    }
  }
  // ---- lazy online softmax ------------------------------------------------------------------------------------------
  float mx = fmaxf(s[0][0], s[0][1]);
#pragma unroll
  for (int j = 1; j < TB; ++j) mx = fmaxf(mx, fmaxf(s[j][0], s[j][1]));
  if (first || __any_sync(kFull, mx > kLazy)) {
    mx = fmaxf(mx, __shfl_xor_sync(kFull, mx, 1));
    mx = fmaxf(mx, __shfl_xor_sync(kFull, mx, 2));
    const float up = first ? mx : fmaxf(mx, 0.f);      // new reference = old reference + up (never lowered later)
    const float corr = first ? 1.f : ex2(-up);         // nothing accumulated yet on the first stage
    st.m = (first ? 0.f : st.m) + up;
    st.l *= corr;
#pragma unroll
    for (int i = 0; i < NK; ++i) { st.acc[i][0] *= corr; st.acc[i][1] *= corr; }
    if constexpr (RESID) {
#pragma unroll
      for (int c = 0; c < G::NE; ++c) { st.eacc[c][0] *= corr; st.eacc[c][1] *= corr; }
    }
#pragma unroll
    for (int j = 0; j < TB; ++j) { s[j][0] -= up; s[j][1] -= up; }
  }
  float pr[TB][2];
#pragma unroll
  for (int j = 0; j < TB; ++j) {
    pr[j][0] = ex2(s[j][0]);
    pr[j][1] = ex2(s[j][1]);
    st.l += pr[j][0] + pr[j][1];
  }
  // ---- a += P . cV ----------------------------------------------------------------------------------------------------
#pragma unroll
  for (int ks = 0; ks < TB / 2; ++ks) {
    uint32_t pa[4];
    pa[0] = pack_bf16x2(pr[2 * ks][0], pr[2 * ks][1]);
    pa[1] = 0u;
    pa[2] = pack_bf16x2(pr[2 * ks + 1][0], pr[2 * ks + 1][1]);
    pa[3] = 0u;
#pragma unroll
    for (int i = 0; i < NK; ++i) mma16816q(st.acc[i], pa, vw[i][2 * ks], vw[i][2 * ks + 1]);
  }
  // ---- e += (P * scaleV) . codeV ----------------------------------------------------------------------------------------
  if constexpr (RESID) {
    const uint32_t codeV = sp + 2 * G::COEF + 10 * D;
    const uint32_t scaleV = codeV + 8 * D;
    uint32_t w[D / 16], sc0[NG], sc1[NG];
    if constexpr (D == 128) {
      const uint4 c0 = lds128(codeV + lane * 32);
      const uint4 c1 = lds128(codeV + lane * 32 + 16);
      w[0] = c0.x; w[1] = c0.y; w[2] = c0.z; w[3] = c0.w; w[4] = c1.x; w[5] = c1.y; w[6] = c1.z; w[7] = c1.w;
      const uint32_t spv = scaleV + t * 32;
      const uint4 x0 = lds128(spv), x1 = lds128(spv + 16), y0 = lds128(spv + D), y1 = lds128(spv + D + 16);
      sc0[0] = x0.x; sc0[1] = x0.y; sc0[2] = x0.z; sc0[3] = x0.w; sc0[4] = x1.x; sc0[5] = x1.y; sc0[6] = x1.z; sc0[7] = x1.w;
      sc1[0] = y0.x; sc1[1] = y0.y; sc1[2] = y0.z; sc1[3] = y0.w; sc1[4] = y1.x; sc1[5] = y1.y; sc1[6] = y1.z; sc1[7] = y1.w;
    } else {
      const uint4 c0 = lds128(codeV + lane * 16);
      w[0] = c0.x; w[1] = c0.y; w[2] = c0.z; w[3] = c0.w;
      const uint32_t spv = scaleV + t * 16;
      const uint4 x0 = lds128(spv), y0 = lds128(spv + D);
      sc0[0] = x0.x; sc0[1] = x0.y; sc0[2] = x0.z; sc0[3] = x0.w;
      sc1[0] = y0.x; sc1[1] = y0.y; sc1[2] = y0.z; sc1[3] = y0.w;
    }
#pragma unroll
    for (int grp = 0; grp < NG; ++grp) {
      const float2 f0 = h2f2(sc0[grp]);
      const float2 f1 = h2f2(sc1[grp]);
      const uint32_t a0 = pack_bf16x2(pr[0][0] * f0.x, pr[0][1] * f0.y);
      const uint32_t a2 = pack_bf16x2(pr[1][0] * f1.x, pr[1][1] * f1.y);
#pragma unroll
      for (int cc = 0; cc < 2; ++cc) {
        const int c = 2 * grp + cc, q = 2 * c;
        mma16816(st.eacc[c][0], st.eacc[c][1], a0, a2, nib_to_bf16x2(w[q >> 2], q & 3), nib_to_bf16x2(w[q >> 2], (q & 3) + 1));
      }
    }
  }
}

struct WarpCtx {          // per-warp streaming state, all in registers (everything below is force-inlined)
  uint32_t ring_s;        // shared address of this warp's ring
  uint32_t bar0;          // shared address of this warp's first mbarrier
  uint32_t phase;         // per-slot parity bits
  int lane;
};

// Process the run of consecutive items of one class starting at (u, lh); `n_items` items remain in the warp's slice.
// Returns the number of items consumed; (u, lh, un) are advanced past the run.
template <int NK, bool RESID, int D>
__device__ __forceinline__ int run_class(const Scan2Params& p, WarpCtx& cx, int& u, int& lh, Unit& un, const int n_items) {
  using G = Geo<NK, RESID, D>;
  using QF = QFrag<NK, RESID, D>;
  constexpr int SB = G::SB, NS = G::NS, NG = G::NG;
  constexpr int kBlockBytes = SB * (kBlockTok / G::SUBTOK);
  const int lane = cx.lane, g = lane >> 2, t = lane & 3;
  const int cls = un.cls;
  auto nstages = [](const Unit& x) { return RESID ? (x.ntok + 15) >> 4 : x.nblk; };
  auto item_base = [&](const Unit& x, int lhx) {
    return p.arena + x.page_off + (size_t)(p.layer0 * p.H + lhx) * kPageLhBytes + (size_t)x.blk0 * kBlockBytes;
  };

  // ---- fetch stream (runs up to NS stages ahead of the compute stream) --------------------------------------------------
  int u_f = u, lh_f = lh, st_f = 0, k_f = 0, left_f = n_items;
  Unit un_f = un;
  int nst_f = nstages(un_f);
  const uint8_t* src_f = item_base(un_f, lh_f);
  bool f_on = true;
  auto fetch_one = [&]() {
    if (!f_on) return;
    if (lane == 0) {
      const uint32_t bar = cx.bar0 + 8 * k_f;
      mbar_expect_tx(bar, SB);
      bulk_g2s(cx.ring_s + k_f * SB, src_f, SB, bar);
    }
    src_f += SB;
    k_f = (k_f + 1 == NS) ? 0 : k_f + 1;
    if (++st_f == nst_f) {
      st_f = 0;
      if (--left_f == 0) {
        f_on = false;
      } else {
        if (++lh_f == p.LH) {
          lh_f = 0;
          un_f = load_unit(p.units + (++u_f));
          nst_f = nstages(un_f);
          if (un_f.cls != cls) f_on = false;
        }
        src_f = item_base(un_f, lh_f);
      }
    }
  };
#pragma unroll 1
  for (int i = 0; i < NS; ++i) fetch_one();

  // ---- compute stream --------------------------------------------------------------------------------------------------
  int k_c = 0, done = 0;
  while (true) {
    const int layer = p.layer0 + lh / p.H, h = lh % p.H;
    QF qf;
    {
      const size_t qoff = ((size_t)un.b * p.LH + lh) * 8 * p.r + (size_t)g * p.r + 2 * t;
      uint32_t qh[NK], ql[NK];
#pragma unroll
      for (int i = 0; i < NK; ++i) {
        qh[i] = *reinterpret_cast<const uint32_t*>(p.qt_hi + qoff + 8 * i);
        ql[i] = *reinterpret_cast<const uint32_t*>(p.qt_lo + qoff + 8 * i);
      }
#pragma unroll
      for (int pi = 0; pi < QF::NP; ++pi) {
        const bool pair = 2 * pi + 1 < NK;
        qf.hi[pi][0] = qh[2 * pi]; qf.hi[pi][1] = 0u; qf.hi[pi][2] = pair ? qh[2 * pi + 1] : ql[2 * pi]; qf.hi[pi][3] = 0u;
        qf.lo[pi][0] = ql[2 * pi]; qf.lo[pi][1] = 0u; qf.lo[pi][2] = pair ? ql[2 * pi + 1] : 0u; qf.lo[pi][3] = 0u;
      }
    }
    if constexpr (RESID) {
      const __nv_bfloat16* q = p.q + (((size_t)un.b * p.Lq + (p.Lq == 1 ? 0 : layer)) * (p.H * p.G) + (size_t)h * p.G + g) * D;
#pragma unroll
      for (int grp = 0; grp < NG; ++grp) {
        qf.qa[grp][0] = (g < p.G) ? *reinterpret_cast<const uint32_t*>(q + 16 * grp + 2 * t) : 0u;
        qf.qa[grp][1] = (g < p.G) ? *reinterpret_cast<const uint32_t*>(q + 16 * grp + 8 + 2 * t) : 0u;
        const float2 x = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&qf.qa[grp][0]));
        const float2 y = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&qf.qa[grp][1]));
        float sum = (x.x + x.y) + (y.x + y.y);
        sum += __shfl_xor_sync(kFull, sum, 1);
        sum += __shfl_xor_sync(kFull, sum, 2);
        qf.qbias[grp] = -136.f * sum;
      }
    } else {
      qf.qa[0][0] = qf.qa[0][1] = 0u;
      qf.qbias[0] = 0.f;
    }
    State<NK, RESID, D> st;
    st.m = 0.f;
    st.l = 0.f;
#pragma unroll
    for (int i = 0; i < NK; ++i) st.acc[i][0] = st.acc[i][1] = st.acc[i][2] = st.acc[i][3] = 0.f;
#pragma unroll
    for (int c = 0; c < G::NE; ++c) st.eacc[c][0] = st.eacc[c][1] = 0.f;

    const int nst = nstages(un);
    int nv_left = un.ntok;
#pragma unroll 1
    for (int sidx = 0; sidx < nst; ++sidx) {
      mbar_wait(cx.bar0 + 8 * k_c, (cx.phase >> k_c) & 1u);
      cx.phase ^= 1u << k_c;
      process_stage<NK, RESID, D>(st, cx.ring_s + k_c * SB, nv_left, lane, sidx == 0, qf, p.cscale);
      nv_left -= G::SUBTOK;
      k_c = (k_c + 1 == NS) ? 0 : k_c + 1;
      __syncwarp();
      fetch_one();     // refill the slot that was just consumed
    }
    // ---- partial of this item: (m_ref, l, a[R]) (+ e[D]) per query head ------------------------------------------------
    st.l += __shfl_xor_sync(kFull, st.l, 1);
    st.l += __shfl_xor_sync(kFull, st.l, 2);
    if (g < p.G) {
      const int PR = 2 + p.r;
      float* prec = p.part + ((size_t)lh * p.n_units_total + u) * (size_t)(p.G * PR) + g * PR;
      if (t == 0) *reinterpret_cast<float2*>(prec) = make_float2(st.m, st.l);
#pragma unroll
      for (int i = 0; i < NK; ++i) *reinterpret_cast<float2*>(prec + 2 + 8 * i + 2 * t) = make_float2(st.acc[i][0], st.acc[i][1]);
      if constexpr (RESID) {
        float* erec = p.epart + ((size_t)lh * p.n_eunits_total + un.epart) * (size_t)(p.G * D) + g * D;
#pragma unroll
        for (int c = 0; c < G::NE; ++c) *reinterpret_cast<float2*>(erec + 8 * c + 2 * t) = make_float2(st.eacc[c][0], st.eacc[c][1]);
      }
    }
    ++done;
    if (++lh == p.LH) {
      lh = 0;
      ++u;
      if (done < n_items) un = load_unit(p.units + u);
    }
    if (done == n_items || un.cls != cls) break;
  }
  return done;
}

template <int D>
__global__ void __launch_bounds__(kWarps * 32, 1) scan2_kernel(const __grid_constant__ Scan2Params p) {
  extern __shared__ __align__(128) uint8_t smem[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t bars = smem_u32(smem + kWarps * kRing) + warp * kMaxStages * 8;
  if (lane == 0) {
    for (int s = 0; s < kMaxStages; ++s) mbar_init(bars + 8 * s, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  __syncwarp();
  const int gw = warp * gridDim.x + blockIdx.x;        // consecutive slices of the item list go to different SMs
  const int pos0 = p.wstart[gw];
  int left = p.wstart[gw + 1] - pos0;
  if (left <= 0) return;
  int u = pos0 / p.LH, lh = pos0 % p.LH;
  Unit un = load_unit(p.units + u);
  WarpCtx cx{smem_u32(smem) + warp * kRing, bars, 0u, lane};
  while (left > 0) {
    const int key = (un.rk >> 3) * 2 + (un.cls & 1);
    int n = left;
    switch (key) {
      case 2: n = run_class<1, false, D>(p, cx, u, lh, un, left); break;
      case 4: n = run_class<2, false, D>(p, cx, u, lh, un, left); break;
      case 6: n = run_class<3, false, D>(p, cx, u, lh, un, left); break;
      case 8: n = run_class<4, false, D>(p, cx, u, lh, un, left); break;
      case 12: n = run_class<6, false, D>(p, cx, u, lh, un, left); break;
      case 16: n = run_class<8, false, D>(p, cx, u, lh, un, left); break;
      case 3: n = run_class<1, true, D>(p, cx, u, lh, un, left); break;
      case 5: n = run_class<2, true, D>(p, cx, u, lh, un, left); break;
      case 7: n = run_class<3, true, D>(p, cx, u, lh, un, left); break;
      case 9: n = run_class<4, true, D>(p, cx, u, lh, un, left); break;
      case 13: n = run_class<6, true, D>(p, cx, u, lh, un, left); break;
      case 17: n = run_class<8, true, D>(p, cx, u, lh, un, left); break;
      default: break;   // unsupported rank (the host refuses these configurations)
    }
    left -= n;
  }
}

}  // namespace

int scan2_num_warps(int n_sms) { return n_sms * kWarps; }

int launch_scan2(const Scan2Params& p, int n_sms, cudaStream_t s) {
  const int smem = kWarps * kRing + kWarps * kMaxStages * 8;
  static bool attr_set[2] = {false, false};
  if (p.d == 128) {
    if (!attr_set[0]) { cudaFuncSetAttribute(scan2_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem); attr_set[0] = true; }
    scan2_kernel<128><<<n_sms, kWarps * 32, smem, s>>>(p);
  } else {
    if (!attr_set[1]) { cudaFuncSetAttribute(scan2_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem); attr_set[1] = true; }
    scan2_kernel<64><<<n_sms, kWarps * 32, smem, s>>>(p);
  }
  return 1;
}

}  // namespace dwkv
