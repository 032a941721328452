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

constexpr int kWarpsPlain = 16;    // unflagged classes: 16 warps x <= 128 registers
constexpr int kWarpsResid = 8;     // flagged classes: 8 warps x <= 255 registers (32 + 16 accumulators, 48 query registers)
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

__device__ __forceinline__ void mma1688q(float (&d)[4], uint32_t a0, uint32_t a1, uint32_t b0) {
  asm("mma.sync.aligned.m16n8k8.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5}, {%6}, {%0,%1,%2,%3};"
      : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
      : "r"(a0), "r"(a1), "r"(b0));
}
// D = A . B with C = 0: fresh outputs, rows 8..15 discarded by the caller
__device__ __forceinline__ void mma16816z(float (&d)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  asm("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%10,%10,%10,%10};"
      : "=f"(d[0]), "=f"(d[1]), "=f"(d[2]), "=f"(d[3])
      : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1), "f"(0.f));
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
  static constexpr int COEF = NK * 128 * TB;                      // bytes of [K coef] (= [V coef]) of a sub-block
  static constexpr int SB1 = 2 * COEF + (RESID ? 20 * D : 0);     // bytes of one sub-block
  static constexpr int BPS = (!RESID && NK == 1) ? 2 : 1;         // sub-blocks per stage (amortises the per-stage work)
  static constexpr int SB = SB1 * BPS;                            // stage bytes
  static constexpr int NS = (kRing / SB) < kMaxStages ? ((kRing / SB) < 1 ? 1 : (kRing / SB)) : kMaxStages;
  static constexpr int NG = D / 16;
};

template <int NK, bool RESID, int D>
struct State {
  float m, l;
  float acc[NK][4];                         // a[row g][8i + 2t + {0,1}]; rows 8..15 (acc[i][2..3]) stay zero
  float eacc[RESID ? D / 16 : 1][4];        // TRANSPOSED: e[head 2t+{0,1}][channel 16grp + g (+8)]
};

// Query-side operands of one item, in MMA A-fragment order.
template <int NK, bool RESID, int D>
struct QFrag {
  static constexpr int NP = NK / 2;                  // k16 steps over pairs of 8-column chunks; odd NK adds two k8 steps
  uint32_t hi[NP > 0 ? NP : 1][4];
  uint32_t lo[NP > 0 ? NP : 1][4];
  uint32_t hi_last, lo_last;                         // odd NK: last chunk, used with m16n8k8
  uint32_t qa[RESID ? D / 16 : 1][4];                // raw q, group grp: {k 0..7, 0, k 8..15, 0}
};

// One sub-block from shared memory (32-bit shared address sp).
template <int NK, bool RESID, int D>
__device__ __forceinline__ void process_sub(State<NK, RESID, D>& st, const uint32_t sp, const int nv, const int lane,
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
  // ---- scores relative to the reference: s' = q~ . cK - m_ref  (q~ = hi + lo) ----------------------------------------
  const float cinit = first ? 0.f : -st.m;
  float s[TB][4];
#pragma unroll
  for (int j = 0; j < TB; ++j) {
    s[j][0] = cinit; s[j][1] = cinit; s[j][2] = 0.f; s[j][3] = 0.f;
#pragma unroll
    for (int pi = 0; pi < NP; ++pi) {
      mma16816q(s[j], qf.hi[pi], kw[2 * pi][j], kw[2 * pi + 1][j]);
      mma16816q(s[j], qf.lo[pi], kw[2 * pi][j], kw[2 * pi + 1][j]);
    }
    if constexpr (NK & 1) {
      mma1688q(s[j], qf.hi_last, 0u, kw[NK - 1][j]);
      mma1688q(s[j], qf.lo_last, 0u, kw[NK - 1][j]);
    }
  }
  // ---- residual-K term: exact integer-code dot on the tensor cores, fp32 group scales afterwards -----------------------
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
        const int q = 2 * grp;
        float c[4];
        mma16816z(c, qf.qa[grp], nib_to_bf16x2(w[q >> 2], q & 3), nib_to_bf16x2(w[q >> 2], (q & 3) + 1));
        const float2 f = h2f2(sc[grp]);
        sr0 = fmaf(c[0], f.x, sr0);
        sr1 = fmaf(c[1], f.y, sr1);
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
    const float corr = first ? 1.f : ex2(-up);         // nothing accumulated yet on the first sub-block
    st.m = (first ? 0.f : st.m) + up;
    st.l *= corr;
#pragma unroll
    for (int i = 0; i < NK; ++i) { st.acc[i][0] *= corr; st.acc[i][1] *= corr; }
    if constexpr (RESID) {   // e is held transposed: this lane's entries belong to heads 2t and 2t+1
      const float c0 = __shfl_sync(kFull, corr, 8 * t), c1 = __shfl_sync(kFull, corr, 8 * t + 4);
#pragma unroll
      for (int grp = 0; grp < NG; ++grp) {
        st.eacc[grp][0] *= c0; st.eacc[grp][1] *= c1; st.eacc[grp][2] *= c0; st.eacc[grp][3] *= c1;
      }
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
  // ---- e^T += codeV^T . (P * scaleV): channels on the MMA m dimension, no padding rows ------------------------------------
  if constexpr (RESID) {
    const uint32_t codeV = sp + 2 * G::COEF + 10 * D;
    const uint32_t scaleV = codeV + 8 * D;
    uint32_t w[NG], sc0[NG], sc1[NG];
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
    const uint32_t neg136[4] = {0xC308C308u, 0xC308C308u, 0xC308C308u, 0xC308C308u};   // bf16 pairs of -136
#pragma unroll
    for (int grp = 0; grp < NG; ++grp) {
      const float2 f0 = h2f2(sc0[grp]);
      const float2 f1 = h2f2(sc1[grp]);
      const uint32_t b0 = pack_bf16x2(pr[0][0] * f0.x, pr[0][1] * f0.y);
      const uint32_t b1 = pack_bf16x2(pr[1][0] * f1.x, pr[1][1] * f1.y);
      uint32_t a[4];
#pragma unroll
      for (int x = 0; x < 4; ++x) a[x] = nib_to_bf16x2_biased(w[grp], x);     // 136 + code, exact
      mma16816q(st.eacc[grp], a, b0, b1);
      mma16816q(st.eacc[grp], neg136, b0, b1);                                // removes the 136 offset on the tensor pipe
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
  constexpr int SB1 = G::SB1, BPS = G::BPS, NS = G::NS, NG = G::NG;
  constexpr int kBlockBytes = SB1 * (kBlockTok / G::SUBTOK);
  const int lane = cx.lane, g = lane >> 2, t = lane & 3;
  const int cls = un.cls;
  auto nsubs = [](const Unit& x) { return RESID ? (x.ntok + 15) >> 4 : x.nblk; };
  auto item_base = [&](const Unit& x, int lhx) {
    return p.arena + x.page_off + (size_t)(p.layer0 * p.H + lhx) * kPageLhBytes + (size_t)x.blk0 * kBlockBytes;
  };

  // ---- fetch stream (runs up to NS stages ahead of the compute stream) --------------------------------------------------
  int u_f = u, lh_f = lh, k_f = 0, left_f = n_items;
  Unit un_f = un;
  int sub_left_f = nsubs(un_f);
  const uint8_t* src_f = item_base(un_f, lh_f);
  bool f_on = true;
  auto fetch_one = [&]() {
    if (!f_on) return;
    const int nb = (BPS == 1) ? 1 : min(BPS, sub_left_f);
    if (lane == 0) {
      const uint32_t bar = cx.bar0 + 8 * k_f;
      mbar_expect_tx(bar, nb * SB1);
      bulk_g2s(cx.ring_s + k_f * G::SB, src_f, nb * SB1, bar);
    }
    src_f += nb * SB1;
    k_f = (k_f + 1 == NS) ? 0 : k_f + 1;
    sub_left_f -= nb;
    if (sub_left_f == 0) {
      if (--left_f == 0) {
        f_on = false;
      } else {
        if (++lh_f == p.LH) {
          lh_f = 0;
          un_f = load_unit(p.units + (++u_f));
          if (un_f.cls != cls) f_on = false;
        }
        sub_left_f = nsubs(un_f);
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
        qf.hi[pi][0] = qh[2 * pi]; qf.hi[pi][1] = 0u; qf.hi[pi][2] = qh[2 * pi + 1]; qf.hi[pi][3] = 0u;
        qf.lo[pi][0] = ql[2 * pi]; qf.lo[pi][1] = 0u; qf.lo[pi][2] = ql[2 * pi + 1]; qf.lo[pi][3] = 0u;
      }
      qf.hi_last = qh[NK - 1];
      qf.lo_last = ql[NK - 1];
    }
    if constexpr (RESID) {
      const __nv_bfloat16* q = p.q + (((size_t)un.b * p.Lq + (p.Lq == 1 ? 0 : layer)) * (p.H * p.G) + (size_t)h * p.G + g) * D;
#pragma unroll
      for (int grp = 0; grp < NG; ++grp) {
        qf.qa[grp][0] = (g < p.G) ? *reinterpret_cast<const uint32_t*>(q + 16 * grp + 2 * t) : 0u;
        qf.qa[grp][1] = 0u;
        qf.qa[grp][2] = (g < p.G) ? *reinterpret_cast<const uint32_t*>(q + 16 * grp + 8 + 2 * t) : 0u;
        qf.qa[grp][3] = 0u;
      }
    } else {
      qf.qa[0][0] = qf.qa[0][1] = qf.qa[0][2] = qf.qa[0][3] = 0u;
    }
    State<NK, RESID, D> st;
    st.m = 0.f;
    st.l = 0.f;
#pragma unroll
    for (int i = 0; i < NK; ++i) st.acc[i][0] = st.acc[i][1] = st.acc[i][2] = st.acc[i][3] = 0.f;
#pragma unroll
    for (int c = 0; c < (RESID ? NG : 1); ++c) st.eacc[c][0] = st.eacc[c][1] = st.eacc[c][2] = st.eacc[c][3] = 0.f;

    int sub_left = nsubs(un);
    int nv_left = un.ntok;
    bool first = true;
#pragma unroll 1
    while (sub_left > 0) {
      mbar_wait(cx.bar0 + 8 * k_c, (cx.phase >> k_c) & 1u);
      cx.phase ^= 1u << k_c;
      const uint32_t sp = cx.ring_s + k_c * G::SB;
#pragma unroll
      for (int b = 0; b < BPS; ++b) {
        if (b == 0 || sub_left > b) {
          process_sub<NK, RESID, D>(st, sp + b * SB1, nv_left - b * G::SUBTOK, lane, first && b == 0, qf, p.cscale);
        }
      }
      first = false;
      nv_left -= BPS * G::SUBTOK;
      sub_left -= BPS;
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
    }
    if constexpr (RESID) {
      float* erec = p.epart + ((size_t)lh * p.n_eunits_total + un.epart) * (size_t)(p.G * D);
#pragma unroll
      for (int x = 0; x < 2; ++x) {
        const int head = 2 * t + x;
        if (head < p.G) {
#pragma unroll
          for (int grp = 0; grp < NG; ++grp) {
            erec[head * D + 16 * grp + g] = st.eacc[grp][x];
            erec[head * D + 16 * grp + 8 + g] = st.eacc[grp][2 + x];
          }
        }
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

template <int D, bool RESID>
__global__ void __launch_bounds__((RESID ? kWarpsResid : kWarpsPlain) * 32, 1) scan2_kernel(const __grid_constant__ Scan2Params p) {
  constexpr int WARPS = RESID ? kWarpsResid : kWarpsPlain;
  extern __shared__ __align__(128) uint8_t smem[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t bars = smem_u32(smem + WARPS * kRing) + warp * kMaxStages * 8;
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
    const int nk = un.rk >> 3;
    int n = left;
    switch (nk) {
      case 1: n = run_class<1, RESID, D>(p, cx, u, lh, un, left); break;
      case 2: n = run_class<2, RESID, D>(p, cx, u, lh, un, left); break;
      case 3: n = run_class<3, RESID, D>(p, cx, u, lh, un, left); break;
      case 4: n = run_class<4, RESID, D>(p, cx, u, lh, un, left); break;
      case 6: n = run_class<6, RESID, D>(p, cx, u, lh, un, left); break;
      case 8: n = run_class<8, RESID, D>(p, cx, u, lh, un, left); break;
      default: break;   // unsupported rank (the host refuses these configurations)
    }
    left -= n;
  }
}

template <int D, bool RESID>
void launch_one(const Scan2Params& p, int n_sms, cudaStream_t s) {
  constexpr int WARPS = RESID ? kWarpsResid : kWarpsPlain;
  const int smem = WARPS * kRing + WARPS * kMaxStages * 8;
  static bool attr_set = false;
  if (!attr_set) {
    cudaFuncSetAttribute(scan2_kernel<D, RESID>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    attr_set = true;
  }
  scan2_kernel<D, RESID><<<n_sms, WARPS * 32, smem, s>>>(p);
}

}  // namespace

int scan2_num_warps(int n_sms, int resid) { return n_sms * (resid ? kWarpsResid : kWarpsPlain); }

// `p.wstart` must be the slice table of the flagged (resid = 1) or unflagged (resid = 0) item range.
int launch_scan2(const Scan2Params& p, int resid, int n_sms, cudaStream_t s) {
  if (resid) {
    if (p.d == 128) launch_one<128, true>(p, n_sms, s); else launch_one<64, true>(p, n_sms, s);
  } else {
    launch_one<128, false>(p, n_sms, s);      // D is irrelevant for unflagged classes
  }
  return 1;
}

}  // namespace dwkv
