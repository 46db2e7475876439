// Device math helpers of the IRIS-SO CUDA path (sm_100a).  fp32 throughout; SFU (MUFU) for exp2 / rcp.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace iris {

#include "erfc_poly.inc"

__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

__device__ __forceinline__ float rcp_approx(float x) {
  float y;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

__device__ __forceinline__ float lg2_approx(float x) {
  float y;
  asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// x^p for x > 0 with the SFU: 2^(p log2 x).  MUFU.LG2 has an absolute error of 2^-22 on (0.5, 2) and a relative one of 2^-22
// elsewhere, so |log2 x| <= 10 and |p| <= 2 keep the result within 2e-6 relative.
__device__ __forceinline__ float pow_approx(float x, float p) { return ex2_approx(p * lg2_approx(x)); }

// exp(x) - 1 for x >= 0 to ~2e-7 relative: series through x^6 / 720 below 0.25 (truncation 5e-8), 2^(x log2 e) - 1 above
// (cancellation <= 6e-8 / 0.28, argument rounding 6e-8 x); both evaluated and selected.  12 instructions against ~35 of expm1f.
__device__ __forceinline__ float expm1_pos(float x) {
  const float big = ex2_approx(x * 1.4426950408889634f) - 1.0f;
  float p = fmaf(x, 1.0f / 720.0f, 1.0f / 120.0f);
  p = fmaf(p, x, 1.0f / 24.0f);
  p = fmaf(p, x, 1.0f / 6.0f);
  p = fmaf(p, x, 0.5f);
  p = fmaf(p, x, 1.0f);
  return x < 0.25f ? p * x : big;
}

// ---- packed fp32 pairs (sm_100: FFMA2 / FMUL2 / FADD2), carried in 64-bit registers
typedef unsigned long long f32x2;

__device__ __forceinline__ f32x2 pk(float lo, float hi) {
  f32x2 r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ f32x2 pk1(float v) { return pk(v, v); }
__device__ __forceinline__ void upk(f32x2 v, float& lo, float& hi) {
  asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) {
  f32x2 r;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
  return r;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) {
  f32x2 r;
  asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) {
  f32x2 r;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}

// "Signed complementary error function"  G(x) = sign(x) * erfc(|x|)   (so erf(x) = sign(x) - G(x)).
// erfc(t) = 2^(t Q(t)) with a degree-10 polynomial (erfc_poly.inc): absolute error ~5e-8 near the line
// centre and RELATIVE error ~2e-6 in the wings, which a plain erf cannot give in fp32 (erf -> 1).
// 10 FFMA + FMNMX + FMUL + MUFU.EX2 + LOP3.
__device__ __forceinline__ float signed_erfc(float x) {
  const float t = fminf(fabsf(x), IRIS_ERFC_TMAX);
  const float c[IRIS_ERFC_DEG + 1] = {IRIS_ERFC_Q_LIST};
  float q = c[IRIS_ERFC_DEG];
#pragma unroll
  for (int i = IRIS_ERFC_DEG - 1; i >= 0; --i) q = fmaf(q, t, c[i]);
  return copysignf(ex2_approx(q * t), x);
}

// Channel integral of the Gaussian profile between two edges x_lo < x_hi (in units of the Doppler
// width):  erf(x_hi) - erf(x_lo) = [sign(x_hi) - sign(x_lo)] - [G(x_hi) - G(x_lo)].
// The sign difference is exactly 0 or 2; G_hi - G_lo keeps the relative accuracy of the wings.
__device__ __forceinline__ float erf_diff(float x_lo, float G_lo, float x_hi, float G_hi) {
  const float sgn = (x_lo < 0.0f && x_hi >= 0.0f) ? 2.0f : 0.0f;
  return sgn - (G_hi - G_lo);
}

// m(tau) = 1 - exp(-tau), accurate to ~1e-6 relative for every tau (also tau < 0).
// Small |tau|: Taylor (the fp32 rounding of exp(-tau) near 1 would otherwise leave an absolute error
// of 6e-8, i.e. a relative error of 6e-8 / tau).  FMUL + MUFU.EX2 + FADD + 4 FFMA/FMUL + FSETP + FSEL.
__device__ __forceinline__ float one_minus_exp_neg(float tau) {
  const float big = 1.0f - ex2_approx(tau * -1.4426950408889634f);
  float p = fmaf(tau, -1.0f / 120.0f, 1.0f / 24.0f);
  p = fmaf(p, -tau, 1.0f / 6.0f);      // 1/6 - tau/24 + tau^2/120
  p = fmaf(p, -tau, 0.5f);             // 1/2 - tau/6 + ...
  p = fmaf(p, -tau, 1.0f);             // 1 - tau/2 + ...
  const float small = p * tau;
  return fabsf(tau) < 0.15f ? small : big;
}

// exp(-tau) with the SFU.
__device__ __forceinline__ float exp_neg(float tau) { return ex2_approx(tau * -1.4426950408889634f); }

// Philox4x32-10 (Salmon et al. 2011): counter-based generator used for the noise stage.
__device__ __forceinline__ void philox4x32_10(uint32_t k0, uint32_t k1, uint32_t c0, uint32_t c1, uint32_t c2,
                                              uint32_t c3, uint32_t out[4]) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
    c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

}  // namespace iris
