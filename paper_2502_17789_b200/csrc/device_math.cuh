// Small device helpers shared by the gridder epilogue and the degridder prologue.
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

namespace idg {

__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
  return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}
// a * conj(b)
__device__ __forceinline__ float2 cmulc(float2 a, float2 b) {
  return make_float2(fmaf(a.x, b.x, a.y * b.y), fmaf(a.y, b.x, -a.x * b.y));
}
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }

// Z = t * Mp * X * Mq^H for 2x2 row-major complex matrices (PAPER.md :156, §3.3 :251-257, R5).
// mp0 = (Mp00, Mp01), mp1 = (Mp10, Mp11) as float4 (re, im, re, im); likewise mq0, mq1.
__device__ __forceinline__ void sandwich(const float2 x[4], float4 mp0, float4 mp1, float4 mq0, float4 mq1,
                                         float t, float2 z[4]) {
  const float2 a = make_float2(mp0.x, mp0.y), b = make_float2(mp0.z, mp0.w);
  const float2 c = make_float2(mp1.x, mp1.y), d = make_float2(mp1.z, mp1.w);
  const float2 q00 = make_float2(mq0.x, mq0.y), q01 = make_float2(mq0.z, mq0.w);
  const float2 q10 = make_float2(mq1.x, mq1.y), q11 = make_float2(mq1.z, mq1.w);
  const float2 y00 = cadd(cmul(a, x[0]), cmul(b, x[2]));
  const float2 y01 = cadd(cmul(a, x[1]), cmul(b, x[3]));
  const float2 y10 = cadd(cmul(c, x[0]), cmul(d, x[2]));
  const float2 y11 = cadd(cmul(c, x[1]), cmul(d, x[3]));
  float2 r;
  r = cadd(cmulc(y00, q00), cmulc(y01, q01)); z[0] = make_float2(t * r.x, t * r.y);
  r = cadd(cmulc(y00, q10), cmulc(y01, q11)); z[1] = make_float2(t * r.x, t * r.y);
  r = cadd(cmulc(y10, q00), cmulc(y11, q01)); z[2] = make_float2(t * r.x, t * r.y);
  r = cadd(cmulc(y10, q10), cmulc(y11, q11)); z[3] = make_float2(t * r.x, t * r.y);
}

// 1 / || Mp Mq^H ||_F of row-major 2x2 complex matrices (section 3.3, R22): the power
// normalisation of the imaging sandwich.  IEEE sqrt and division (no fast-math approximations).
__device__ __forceinline__ float frobenius_inv(float4 mp0, float4 mp1, float4 mq0, float4 mq1) {
  const float2 a = make_float2(mp0.x, mp0.y), b = make_float2(mp0.z, mp0.w);
  const float2 c = make_float2(mp1.x, mp1.y), d = make_float2(mp1.z, mp1.w);
  const float2 q00 = make_float2(mq0.x, mq0.y), q01 = make_float2(mq0.z, mq0.w);
  const float2 q10 = make_float2(mq1.x, mq1.y), q11 = make_float2(mq1.z, mq1.w);
  // (Mp Mq^H)[i][j] = sum_k Mp[i][k] conj(Mq[j][k])
  const float2 p00 = cadd(cmulc(a, q00), cmulc(b, q01)), p01 = cadd(cmulc(a, q10), cmulc(b, q11));
  const float2 p10 = cadd(cmulc(c, q00), cmulc(d, q01)), p11 = cadd(cmulc(c, q10), cmulc(d, q11));
  const float n2 = (p00.x * p00.x + p00.y * p00.y) + (p01.x * p01.x + p01.y * p01.y) +
                   (p10.x * p10.x + p10.y * p10.y) + (p11.x * p11.x + p11.y * p11.y);
  return __fdiv_rn(1.f, __fsqrt_rn(n2));
}

// a * x + b * y modulo 2^32, as the signed value in [-2^31, 2^31): the fixed-point phase in cycles * 2^32, which is
// MEANT to wrap (exact modulo one cycle).  The arithmetic is unsigned because signed overflow is undefined
// behaviour in C++: a compiler may assume it never happens and widen or reorder the products.
__device__ __forceinline__ int32_t wrap_dot2(int32_t a, int32_t x, int32_t b, int32_t y) {
  return static_cast<int32_t>(static_cast<uint32_t>(a) * static_cast<uint32_t>(x) +
                              static_cast<uint32_t>(b) * static_cast<uint32_t>(y));
}

__device__ __forceinline__ float2 ffma2(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ float2 neg2(float2 a) { return make_float2(-a.x, -a.y); }

}  // namespace idg
