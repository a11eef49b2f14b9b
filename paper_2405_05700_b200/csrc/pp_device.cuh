// Device-side building blocks of the photon propagator (sm_100a).  Product code: shares nothing
// with oracle/.  Each function cites the step of DESIGN.md section 2 it implements.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "pp_types.h"

namespace pp {

// ---------------------------------------------------------------------------------------------
// R-3: Philox4x32-10 with precomputed round keys; counter = (photon, source, event, flight).
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void philox4x32_10(uint32_t& c0, uint32_t& c1, uint32_t& c2, uint32_t& c3,
                                              const uint32_t (&rk)[10][2]) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const unsigned long long p0 = (unsigned long long)0xD2511F53u * c0;
    const unsigned long long p1 = (unsigned long long)0xCD9E8D57u * c2;
    const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ rk[r][0];
    const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ rk[r][1];
    c1 = (uint32_t)p1;
    c3 = (uint32_t)p0;
    c0 = n0;
    c2 = n2;
  }
}

// u = (x >> 9) * 2^-23 + 2^-24, exactly (R-3): build 1.m from the top 23 bits with one funnel
// shift, then subtract (1 - 2^-24); both steps are exact in fp32.
__device__ __forceinline__ float uniform_from_word(uint32_t x) {
  return __uint_as_float(__funnelshift_r(x, 0x7fu, 9)) - 0.99999994f;
}

#ifdef PP_EXACT_MUFU  // diagnosis only: IEEE-rounded reciprocal / square roots instead of the MUFU approximations
__device__ __forceinline__ float fast_rcp(float x) { return __frcp_rn(x); }
__device__ __forceinline__ float fast_rsqrt(float x) { return __frcp_rn(__fsqrt_rn(x)); }
__device__ __forceinline__ float fast_sqrt(float x) { return __fsqrt_rn(x); }
#else
__device__ __forceinline__ float fast_rcp(float x) {
  float r;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}
__device__ __forceinline__ float fast_rsqrt(float x) {
  float r;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}
__device__ __forceinline__ float fast_sqrt(float x) {
  float r;
  asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}
#endif

// (a == b) ? x : y as one compare and one select whose operands are evaluated unconditionally
__device__ __forceinline__ float select_eq(int a, int b, float x, float y) {
  float r;
  asm("{ .reg .pred p; setp.eq.s32 p, %1, %2; selp.f32 %0, %3, %4, p; }" : "=f"(r) : "r"(a), "r"(b), "f"(x), "f"(y));
  return r;
}

// Step 9a: Henyey-Greenstein, returned as m = 1 - cos(theta) in the cancellation-free form
//   m = (1-g)(1-u)(q + 1 - g)/(1 - g + 2 g u),  q = (1-g^2)/(1 - g + 2 g u)        (R-1)
__device__ __forceinline__ float hg_one_minus_cos(float u, float one_minus_g, float two_g, float one_minus_g2) {
  const float inv = fast_rcp(fmaf(two_g, u, one_minus_g));
  const float q = one_minus_g2 * inv;
  return one_minus_g * (1.0f - u) * (q + one_minus_g) * inv;
}

// -ln(u) for both optical-depth budgets: one MUFU.LG2 and one multiply.  lg2.approx has an absolute error <= 2^-22 on
// [1/2, 2) and <= 2 ulp elsewhere, i.e. <= 1.7e-7 in optical depth: the scatter point moves along the ray by
// <= 1.7e-7 lambda_s (4e-6 m at 25 m) and the absorption point by <= 1.7e-7 lambda_abs.  Measured effect on the
// per-hit time parity against a degree-8 polynomial with relative error 1e-7: profiles/r02_parity.md.
// u is a normal number (R-3): no denormal handling is needed.
__device__ __forceinline__ float neg_log_fast(float u) {
  float l;
  asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(l) : "f"(u));
  return l * -0.693147182464599609375f;
}

// (sin, cos) of 2 pi u for u in (0, 1): j = rint(4u) picks the quadrant, f = 4u - j in [-1/2, 1/2] is exact,
// sin and cos of f pi/2 from degree-7/8 minimax fits (errors 2.4e-8 / 1e-8, fitted for this file), then the
// quadrant swap and signs from the two low bits of j.
__device__ __forceinline__ void sincos_2pi(float u, float& sn, float& cs) {
  const float t = fmaf(u, 4.0f, 12582912.0f);  // 1.5 * 2^23: the low mantissa bits now hold j
  const float jf = t - 12582912.0f;
  const float f = fmaf(u, 4.0f, -jf);
  const float f2 = f * f;
  float s = -0.004602177068591118f;
  s = fmaf(s, f2, 0.07968022674322128f);
  s = fmaf(s, f2, -0.6459634900093079f);
  s = fmaf(s, f2, 1.5707963705062866f);
  s *= f;
  float c = 0.0009095630957745016f;
  c = fmaf(c, f2, -0.020862672477960587f);
  c = fmaf(c, f2, 0.25366953015327454f);
  c = fmaf(c, f2, -1.2337005138397217f);
  c = fmaf(c, f2, 1.0f);
  const uint32_t j = __float_as_uint(t);
  const bool swap = (j & 1u) != 0u;
  const float a = swap ? c : s, b = swap ? s : c;
  sn = __uint_as_float(__float_as_uint(a) ^ ((j << 30) & 0x80000000u));
  cs = __uint_as_float(__float_as_uint(b) ^ (((j + 1u) << 30) & 0x80000000u));
}

// Step 2 / 9b: rotate d by polar angle (m = 1 - cos) and azimuth 2*pi*u_az about itself (R-9),
// then renormalise with one Newton step (|n|^2 is within ~1e-6 of 1).
__device__ __forceinline__ void rotate(float& dx, float& dy, float& dz, float m, float u_az) {
  const float cos_t = 1.0f - m;
  const float sin_t = fast_sqrt(fmaxf(m * (2.0f - m), 0.0f));
  float sp, cp;
  sincos_2pi(u_az, sp, cp);
  const float rho2 = fmaf(dx, dx, dy * dy);
  float nx, ny, nz;
  if (rho2 > kPoleRho2) {
    const float inv_rho = fast_rsqrt(rho2);
    const float a = sin_t * inv_rho;
    const float dzc = dz * cp;
    nx = fmaf(a, fmaf(dx, dzc, -dy * sp), dx * cos_t);
    ny = fmaf(a, fmaf(dy, dzc, dx * sp), dy * cos_t);
    nz = fmaf(-sin_t * cp, rho2 * inv_rho, dz * cos_t);
  } else {
    nx = sin_t * cp;
    ny = sin_t * sp;
    nz = dz >= 0.0f ? cos_t : -cos_t;
  }
  const float n2 = fmaf(nx, nx, fmaf(ny, ny, nz * nz));
  const float f = fmaf(-0.5f, n2, 1.5f);
  dx = nx * f;
  dy = ny * f;
  dz = nz * f;
}

}  // namespace pp
