// Shared pieces of the LOS transfer kernels (K3 + fused K4 / K5).
//
// The march of Eq. 4.8.5-4.8.7 is carried in the DIFFERENCE form
//   D_k = I^[T]_k - I^[C]_k     (total minus continuum, Rayleigh-Jeans Kelvin),
// together with the scalar continuum march C_k = I^[C]_k (Eq. 3.1.3), which is algebraically the same
// recurrence as marching I^[T] and I^[C] separately and subtracting at the end (section 4.10), but has no
// cancellation: weak lines on a bright continuum keep their relative accuracy in fp32.
//
// One cell, one channel, with  tau_L = a_c dErf,  J_L = e_c dErf,  m = 1 - exp(-tau_L),
// E_d = exp(-tau_d),  m_d = 1 - E_d,  tau_T = tau_L + tau_d:
//   D' = E_d [ D - (D + C) m ] + [ J_L (m_d + E_d m) + S_d (tau_d E_d m - tau_L m_d) ] / tau_T
//   C' = C E_d + S_d m_d
// and without dust (tau_d = 0, C = I_bg constant):   D' = D + (S_L - C - D) m,  S_L = e_c / a_c.
#pragma once
#include "iris_math.cuh"

// Checked build (python -m paper_2607_01338_b200.build --checked -> libiris_so_checked.so, tests/test_sanitizers.py):
// every shared-memory access of the line-window kernels is tested against the region its warp owns and traps outside it
// (compute-sanitizer is closed on the GPU pool this library is developed on; this is the bounds check of our own).
#ifdef IRIS_SO_CHECKED
#include <cstdio>
#define IRIS_CHECK_SMEM(ptr, bytes, lo, hi)                                                                    \
  do {                                                                                                         \
    const char* p_ = reinterpret_cast<const char*>(ptr);                                                       \
    if (p_ < reinterpret_cast<const char*>(lo) || p_ + (bytes) > reinterpret_cast<const char*>(hi)) {          \
      printf("IRIS_SO_CHECKED: shared-memory access out of the warp's region at %s:%d\n", __FILE__, __LINE__);  \
      __trap();                                                                                                \
    }                                                                                                          \
  } while (0)
#else
#define IRIS_CHECK_SMEM(ptr, bytes, lo, hi) ((void)0)
#endif

namespace iris {

// The windowed kernels store the spectrum multiplied by G = exp(dust optical depth so far) and fold G back into it when
// it passes kFoldG.  A single cell's exp(+-tau_d) is taken at min(tau_d, kMaxTauDCell): exp(-50) = 2e-22 is nothing in
// fp32, and kFoldG exp(50) times any intensity in K stays inside the fp32 range (a cell with tau_d ~ 100 would overflow).
constexpr float kMaxTauDCell = 50.0f;
constexpr float kFoldG = 1.0e10f;

// coefficient plane order written by K2
enum { Q_E = 0, Q_A = 1, Q_CLOS = 2, Q_S = 3, Q_TAUD = 4, Q_SD = 5 };

// output conversion (K5): what to write for a voxel with difference D and continuum C (both in K_RJ)
enum OutMode {
  OUT_TRJ_SUB = 0,     // D
  OUT_TRJ_TOT = 1,     // D + C
  OUT_I_SUB = 2,       // D / K_RJ
  OUT_I_TOT = 3,       // (D + C) / K_RJ
  OUT_TB_OF_SUB = 4,   // T_B(D / K_RJ)              (odd extension for negative values)
  OUT_TB_OF_TOT = 5,   // T_B((D + C) / K_RJ)
  OUT_TB_SUB = 6       // T_B(total) - T_B(continuum)  (Planck-space subtraction, section 4.10)
};

struct MarchConsts {
  float T_bg;       // K_RJ B_nu0(T_cmb): background in Rayleigh-Jeans Kelvin
  float hnu_k;      // h nu0 / k
  float inv_KRJ;    // 2 k nu0^2 / c^2  (Kelvin -> CGS intensity)
  int out_mode;
  int fine_m;       // fine velocity grid of the series kernel's MODE 3: intervals per channel (f + 1); 0 elsewhere
  int ray_simpson;  // series kernel MODE 2 (optically thin): 1 = Simpson weights along the ray (Eq. 4.7.7), 0 = Eq. 4.7.6
  // dust_per_channel = 1 (dense kernel only): channel k is observed at nu_k = nu0 (1 - v_k / c)
  float v0_over_c, dv_over_c;   // v_k / c = v0_over_c + k dv_over_c
  float hnu_k_over_Tcmb;        // h nu0 / (k T_cmb); 0 = no background
  int sel_thin;     // smooth window kernel only: 1 = selectively thin mode (the line does not absorb itself, Eq. 4.8.13)
};

// Planck function at nu = r nu0 in the units of the march (Rayleigh-Jeans Kelvin AT nu0: I c^2 / (2 k nu0^2)), for
// x0 = h nu0 / (k T):  (h nu0 / k) r^3 / (exp(x0 r) - 1)
__device__ __forceinline__ float planck_krj_at(float hnu_k, float x0, float r) {
  return x0 > 0.0f ? hnu_k * r * r * r * rcp_approx(expm1f(x0 * r)) : 0.0f;
}

// K5 at the channel's own frequency nu_k = r nu0: D, C in Rayleigh-Jeans Kelvin at nu0 (intensity = D inv_KRJ).
__device__ __forceinline__ float planck_tb_at(float t, float hnu_k, float r) {
  if (t == 0.0f) return 0.0f;
  const float tb = hnu_k * r / log1pf(hnu_k * r * r * r / fabsf(t));
  return copysignf(tb, t);
}

// Planck brightness temperature of a Rayleigh-Jeans temperature (Eq. 4.9.1 with I = T_rj / K_RJ):
// T_B = (h nu / k) / ln(1 + (h nu / k) / T_rj); odd extension, T_B(0) = 0.
__device__ __forceinline__ float planck_tb_of_trj(float t, float hnu_k) {
  if (t == 0.0f) return 0.0f;
  const float tb = hnu_k / log1pf(hnu_k / fabsf(t));
  return copysignf(tb, t);
}

__device__ __forceinline__ float convert_out(float D, float C, const MarchConsts& mc) {
  switch (mc.out_mode) {
    case OUT_TRJ_SUB: return D;
    case OUT_TRJ_TOT: return D + C;
    case OUT_I_SUB: return D * mc.inv_KRJ;
    case OUT_I_TOT: return (D + C) * mc.inv_KRJ;
    case OUT_TB_OF_SUB: return planck_tb_of_trj(D, mc.hnu_k);
    case OUT_TB_OF_TOT: return planck_tb_of_trj(D + C, mc.hnu_k);
    default: return planck_tb_of_trj(D + C, mc.hnu_k) - planck_tb_of_trj(C, mc.hnu_k);
  }
}

__device__ __forceinline__ float convert_out_at(float D, float C, const MarchConsts& mc, float r) {
  const float q = 1.0f / (r * r);                       // T_RJ at nu_k = T_RJ at nu0 * (nu0 / nu_k)^2
  switch (mc.out_mode) {
    case OUT_TRJ_SUB: return D * q;
    case OUT_TRJ_TOT: return (D + C) * q;
    case OUT_I_SUB: return D * mc.inv_KRJ;
    case OUT_I_TOT: return (D + C) * mc.inv_KRJ;
    case OUT_TB_OF_SUB: return planck_tb_at(D, mc.hnu_k, r);
    case OUT_TB_OF_TOT: return planck_tb_at(D + C, mc.hnu_k, r);
    default: return planck_tb_at(D + C, mc.hnu_k, r) - planck_tb_at(C, mc.hnu_k, r);
  }
}

// Per-(pixel, cell) scalars of the dust / continuum part.
struct DustStep {
  float tau_d, S_d, E_d, m_d, C;   // C = continuum BEFORE the cell
};

// One heavy update with dust.  dErf = erf difference of the channel in this cell.
__device__ __forceinline__ float update_dust(float D, float dErf, float e_c, float a_c, const DustStep& d) {
  const float tau_L = a_c * dErf;
  const float J_L = e_c * dErf;
  const float m = one_minus_exp_neg(tau_L);
  const float tau_T = tau_L + d.tau_d;
  const float r = rcp_approx(fabsf(tau_T) < 1.0e-30f ? 1.0f : tau_T);   // also keeps denormal tau_T away from rcp.ftz
  const float Em = d.E_d * m;
  const float t1 = d.m_d + Em;
  const float t2 = fmaf(d.tau_d, Em, -tau_L * d.m_d);
  const float num = fmaf(J_L, t1, d.S_d * t2);
  const float inner = fmaf(-(D + d.C), m, D);
  return fmaf(d.E_d, inner, r * num);
}

// One heavy update without dust: sc = S_L - C (per cell), D' = D + (sc - D) m.
__device__ __forceinline__ float update_nodust(float D, float dErf, float a_c, float sc) {
  const float m = one_minus_exp_neg(a_c * dErf);
  return fmaf(sc - D, m, D);
}

}  // namespace iris
