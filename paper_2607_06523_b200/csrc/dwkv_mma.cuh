// dwkv_mma.cuh -- small device helpers shared by the scan kernels: mma.sync wrappers, streaming loads, int4 unpack.
#pragma once
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <stdint.h>

namespace dwkv {
namespace dev {

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

// D(16x8) += A(16x16) . B(16x8), bf16 inputs, fp32 accumulate. Only rows 0..7 of A are populated (a1 = a3 = 0), so
// only d0,d1 (row g) are kept; d2,d3 (row g+8) are written to scratch registers.
__device__ __forceinline__ void mma16816(float& d0, float& d1, uint32_t a0, uint32_t a2, uint32_t b0, uint32_t b1) {
  float j2, j3;
  asm("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%5}, {%7,%8}, {%0,%1,%9,%9};"
      : "+f"(d0), "+f"(d1), "=f"(j2), "=f"(j3)
      : "r"(a0), "r"(0u), "r"(a2), "r"(b0), "r"(b1), "f"(0.f));
}
__device__ __forceinline__ void mma1688(float& d0, float& d1, uint32_t a0, uint32_t b0) {
  float j2, j3;
  asm("mma.sync.aligned.m16n8k8.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5}, {%6}, {%0,%1,%7,%7};"
      : "+f"(d0), "+f"(d1), "=f"(j2), "=f"(j3)
      : "r"(a0), "r"(0u), "r"(b0), "f"(0.f));
}

__device__ __forceinline__ uint32_t pack_bf16x2(float lo, float hi) {
  __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<uint32_t*>(&v);
}

// offset-binary nibble pair s of word w -> bf16x2 (code_lo, code_hi), exact small integers.
// (w >> 4s) & 0x000F000F | 0x43004300 is the bf16 pair (128 + u_lo, 128 + u_hi) = (136 + code).
__device__ __forceinline__ uint32_t nib_to_bf16x2_biased(uint32_t w, int s) {
  uint32_t r;   // one LOP3: (x & 0x000F000F) | 0x43004300, both constants in registers (0xEA = (a & b) | c)
  asm("lop3.b32 %0, %1, %2, %3, 0xEA;" : "=r"(r) : "r"(w >> (4 * s)), "r"(0x000F000Fu), "r"(0x43004300u));
  return r;
}
__device__ __forceinline__ uint32_t nib_to_bf16x2(uint32_t w, int s) {
  uint32_t x = nib_to_bf16x2_biased(w, s);
  const uint32_t c136 = 0x43084308u;
  __nv_bfloat162 r = __hsub2(*reinterpret_cast<__nv_bfloat162*>(&x), *reinterpret_cast<const __nv_bfloat162*>(&c136));
  return *reinterpret_cast<uint32_t*>(&r);
}

__device__ __forceinline__ uint32_t comp(const uint4& v, int j) {
  return j == 0 ? v.x : j == 1 ? v.y : j == 2 ? v.z : v.w;
}

__device__ __forceinline__ float2 h2f2(uint32_t w) {
  return __half22float2(*reinterpret_cast<__half2*>(&w));
}

// 8-bit blockwise coefficient quantiser (reading A27), block = 32 consecutive rank columns of the token's coefficient vector:
// e = smallest integer with amax <= 127 * 2^e, clamped to >= -126 (amax == 0 and subnormal amax land on the clamp);
// code = rint(c / 2^e) in [-127, 127]. Every step is exact in fp32. amax = m * 2^x, m in [0.5, 1): e = x - 7 if m <= 127/128 else x - 6.
__device__ __forceinline__ int coef8_exponent(float amax) {
  const uint32_t b = __float_as_uint(amax);
  const int x = (int)((b >> 23) & 0xffu) - 126;
  const int e = ((b & 0x7fffffu) <= 0x7e0000u) ? x - 7 : x - 6;
  return max(e, -126);
}
__device__ __forceinline__ int coef8_code(float c, int e) {
  const float q = rintf(c * __uint_as_float((uint32_t)(127 - e) << 23));     // c / 2^e, exact
  return (int)fminf(fmaxf(q, -127.f), 127.f);
}

}  // namespace dev
}  // namespace dwkv
