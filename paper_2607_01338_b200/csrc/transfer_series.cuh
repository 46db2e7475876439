// K3 (line-window formulation, narrow channels): the production LOS transfer kernel.
//
// Same recurrence and the same line window as transfer_window.cuh (difference form D = I^[T] - I^[C],
// Dt = D * exp(sum tau_d), updates only inside |x| <= X_w), with two changes that remove most of the
// instructions of that kernel:
//
// 1. Profile.  When a channel is narrower than ~half a Doppler width (s = dv / b <= kSeriesMaxS), the channel
//    integral of the Gaussian profile (Eq. 4.6.3) is evaluated from the channel CENTRE x by
//    the Taylor expansion of the integrand about the centre,
//      erf(x + s/2) - erf(x - s/2) = (2 s / sqrt(pi)) exp(-x^2) [1 + (s^2/24) H_2(x) + (s^4/1920) H_4(x)
//                                     + (s^6/322560) H_6(x) + (s^8/92897280) H_8(x)],   H_n = Hermite polynomials,
//    i.e. exp(-x^2) times a degree-4 polynomial in x^2 whose five coefficients depend on the cell only.
//    Truncation error at s = 0.55: <= 2e-7 relative for |x| <= 3, <= 2e-9 absolute everywhere (the error is
//    relative to a value that is itself < 1e-9 beyond |x| = 4.4).  One MUFU.EX2 + 7 FP32 instructions per
//    channel, no edge sharing between lanes, no sign handling.
// 2. Per-cell work is done ONCE per cell, not once per lane: the march is cut into chunks of LPP cells; in
//    phase A lane (g, i) of a warp turns the six coefficients of cell z0 + i of pixel g into a 16-float
//    "march record" (window, scaled coordinates, polynomial, dust factors) in shared memory; in phase B the
//    LPP lanes of pixel g walk the LPP cells, reading each record with four broadcast LDS.128.
//
// Mapping as in transfer_window.cuh: a warp owns 32/LPP adjacent pixels, LPP lanes per pixel; the spectrum
// Dt[nv] of each pixel lives in shared memory for the whole march, bank-interleaved (channel c of pixel g at
// word (c / LPP) * 32 + g * LPP + c % LPP: the lanes of a warp always hit 32 distinct banks).
#pragma once
#include "transfer_common.cuh"
#include "transfer_window.cuh"

namespace iris {

constexpr float kSeriesMaxS = 0.55f;   // largest dv / b the centre expansion is used for

// March record of one cell (16 floats, four float4):
//   r0 = { As, tau_d | sc, x0, xs }     As = a_c 2 s / sqrt(pi)  (tau_L = As g);  x0, xs: scaled centre of channel
//                                       klo and scaled step, x' = x sqrt(log2 e) so that exp(-x^2) = 2^(-x'^2)
//   r1 = { P, Q, R, bits(klo | khi << 16) }     num = g P + m (Q g + R)   (dust);  klo > khi: empty window
//   r2 = { p0, p1, p2, p3 }             polynomial in u' = x'^2
//   r3 = { p4, E_d, S_d m_d, exp(tau_d) }
struct SeriesRecord { float4 r0, r1, r2, r3; };

// Phase A: coefficients of one cell -> march record.
template <bool DUST>
__device__ __forceinline__ SeriesRecord make_series_record(float e_c, float a_c, float c_los, float s, float tau_d,
                                                           float S_d, float T_bg, int nv) {
  SeriesRecord r;
  int klo, khi;
  const int W = line_window(e_c, a_c, c_los, s, nv, klo, khi);
  if (W <= 0) { klo = 1; khi = 0; }
  const float sp = 1.1283791670955126f * s;                 // 2 s / sqrt(pi)
  const float a_safe = (a_c == 0.0f) ? 1.0e-30f : a_c;      // keeps e_c / a_c finite; tau_L stays ~0
  const float As = a_safe * sp, Es = e_c * sp;
  const float xs = 1.2011224087864498f * s;                 // s sqrt(log2 e)
  r.r0.x = As;
  r.r0.z = ((float)klo + 0.5f - c_los) * xs;
  r.r0.w = xs;
  // polynomial in u = x^2, then rescaled to u' = u log2(e):  p'_k = p_k ln(2)^k
  const float s2 = s * s, s4 = s2 * s2, s6 = s4 * s2, s8 = s4 * s4;
  const float p0 = 1.0f - s2 * (1.0f / 12.0f) + s4 * (1.0f / 160.0f) - s6 * (1.0f / 2688.0f) + s8 * (1.0f / 55296.0f);
  const float p1 = s2 * (1.0f / 6.0f) - s4 * (1.0f / 40.0f) + s6 * (1.0f / 448.0f) - s8 * (1.0f / 6912.0f);
  const float p2 = s4 * (1.0f / 120.0f) - s6 * (1.0f / 672.0f) + s8 * (1.0f / 6912.0f);
  const float p3 = s6 * (1.0f / 5040.0f) - s8 * (1.0f / 25920.0f);
  const float p4 = s8 * (1.0f / 362880.0f);
  constexpr float L1 = 0.6931471805599453f, L2 = L1 * L1, L3 = L2 * L1, L4 = L2 * L2;
  r.r2 = make_float4(p0, p1 * L1, p2 * L2, p3 * L3);
  r.r3.x = p4 * L4;
  r.r1.w = __int_as_float(klo | (khi << 16));
  if (DUST) {
    const float E_d = exp_neg(tau_d);
    const float m_d = one_minus_exp_neg(tau_d);
    r.r0.y = tau_d;
    r.r1.x = m_d * fmaf(-S_d, As, Es);
    r.r1.y = E_d * Es;
    r.r1.z = E_d * S_d * tau_d;
    r.r3.y = E_d;
    r.r3.z = S_d * m_d;
    r.r3.w = ex2_approx(tau_d * 1.4426950408889634f);
  } else {
    r.r0.y = Es / As - T_bg;      // sc = S_L - C, C = T_bg throughout
    r.r1.x = r.r1.y = r.r1.z = 0.0f;
    r.r3.y = 1.0f; r.r3.z = 0.0f; r.r3.w = 1.0f;
  }
  return r;
}

template <int LPP, bool DUST>
__global__ void __launch_bounds__(128)
transfer_series_kernel(MarchConsts mc, const float* __restrict__ coef, int64_t ncell, int npix, int nz, int nv,
                       int nvp, float* __restrict__ out, float* __restrict__ out_cont) {
  extern __shared__ float4 smem4[];
  constexpr int PPW = 32 / LPP;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, wpc = blockDim.x >> 5;
  const int g = lane / LPP, i = lane % LPP;
  const int pix = (blockIdx.x * wpc + warp) * PPW + g;
  const bool valid = pix < npix;
  const int pl = valid ? pix : npix - 1;
  // shared memory: records [wpc][LPP cells][PPW pixels][4 float4], then spectra [wpc][nvp / LPP rows][32]
  float4* rec = smem4 + (size_t)warp * (LPP * PPW * 4);
  float* spec = reinterpret_cast<float*>(smem4 + (size_t)wpc * (LPP * PPW * 4));
  float* sp = spec + (size_t)warp * nvp * PPW + g * LPP;
  for (int c = i; c < nvp; c += LPP) sp[(c / LPP) * 32 + i] = 0.0f;

  float C = mc.T_bg;      // continuum before the current cell
  float G = 1.0f;         // exp(dust optical depth accumulated so far), since the last rescale

  // phase-A operands of the first chunk: lane (g, i) <-> cell z = i of pixel g
  const float* p = coef + pl + (int64_t)i * npix;
  float l_e = 0.0f, l_a = 0.0f, l_c = 0.0f, l_s = 1.0f, l_td = 0.0f, l_sd = 0.0f;
  if (i < nz) {
    l_e = p[0]; l_a = p[ncell]; l_c = p[2 * ncell]; l_s = p[3 * ncell];
    if (DUST) { l_td = p[4 * ncell]; l_sd = p[5 * ncell]; }
  }

  for (int z0 = 0; z0 < nz; z0 += LPP) {
    // ---- phase A: one record per lane
    {
      const SeriesRecord r = make_series_record<DUST>(l_e, l_a, l_c, l_s, l_td, l_sd, mc.T_bg, nv);
      __syncwarp();                      // phase B of the previous chunk is done with the records
      float4* q = rec + (i * PPW + g) * 4;
      q[0] = r.r0; q[1] = r.r1; q[2] = r.r2; q[3] = r.r3;
      // prefetch the next chunk's coefficients
      const int zn = z0 + LPP + i;
      l_e = 0.0f; l_a = 0.0f; l_td = 0.0f;
      if (zn < nz) {
        p += (int64_t)LPP * npix;
        l_e = p[0]; l_a = p[ncell]; l_c = p[2 * ncell]; l_s = p[3 * ncell];
        if (DUST) { l_td = p[4 * ncell]; l_sd = p[5 * ncell]; }
      }
      __syncwarp();
    }
    // ---- phase B: the LPP lanes of a pixel walk the cells of the chunk
    const int ncz = min(LPP, nz - z0);
    for (int j = 0; j < ncz; ++j) {
      const float4* q = rec + (j * PPW + g) * 4;
      const float4 r0 = q[0], r1 = q[1], r2 = q[2], r3 = q[3];
      const int kk = __float_as_int(r1.w);
      const int klo = kk & 0xffff, khi = (int)((unsigned)kk >> 16);
      const int npass = __reduce_max_sync(0xffffffffu, (khi - klo + LPP) / LPP);   // 0 for an empty window
      float CG = 0.0f, Pn = 0.0f, Qn = 0.0f, Rn = 0.0f;
      if (DUST) {
        const float Gn = G * r3.w;
        CG = C * G;
        C = fmaf(C, r3.y, r3.z);
        Pn = r1.x * Gn; Qn = r1.y * Gn; Rn = r1.z * Gn;
        G = Gn;
      }
      if (npass > 0) {
        int c = klo + i;
        float x = fmaf((float)i, r0.w, r0.z);
        const float step = (float)LPP * r0.w;
        float* d = sp + (c / LPP) * 32 + (c % LPP);
#pragma unroll 2
        for (int ps = 0; ps < npass; ++ps) {
          const float u = x * x;
          float pol = fmaf(r3.x, u, r2.w);
          pol = fmaf(pol, u, r2.z);
          pol = fmaf(pol, u, r2.y);
          pol = fmaf(pol, u, r2.x);
          const float gpr = ex2_approx(-u) * pol;           // dErf / (2 s / sqrt(pi))
          const float tau_L = r0.x * gpr;
          const float m = one_minus_exp_neg(tau_L);
          if (c <= khi) {
            float Dt = *d;
            if (DUST) {
              const float tau_T = tau_L + r0.y;
              const float rr = rcp_approx(tau_T == 0.0f ? 1.0f : tau_T);
              const float num = fmaf(m, fmaf(Qn, gpr, Rn), gpr * Pn);
              Dt = fmaf(-(Dt + CG), m, Dt);
              Dt = fmaf(rr, num, Dt);
            } else {
              Dt = fmaf(r0.y - Dt, m, Dt);
            }
            *d = Dt;
          }
          x += step; c += LPP; d += 32;
        }
      }
      if (DUST && G > 1.0e18f) {   // rare: fold the accumulated dust attenuation into the stored spectrum
        const float inv = 1.0f / G;
        __syncwarp(__activemask());
        for (int cc = i; cc < nvp; cc += LPP) sp[(cc / LPP) * 32 + i] *= inv;
        G = 1.0f;
      }
    }
  }
  __syncwarp();

  const float invG = 1.0f / G;
  if (valid) {
    if (out != nullptr) {
      float* o = out + (int64_t)pix * nv;
      for (int c = i; c < nv; c += LPP) o[c] = convert_out(sp[(c / LPP) * 32 + i] * invG, C, mc);
    }
    if (out_cont != nullptr && i == 0) out_cont[pix] = C * mc.inv_KRJ;
  }
}

template <int LPP>
inline cudaError_t launch_transfer_series_lpp(const MarchConsts& mc, const float* coef, int64_t ncell, int npix, int nz,
                                              int nv, bool dust, float* out, float* out_cont, cudaStream_t st) {
  constexpr int PPW = 32 / LPP;
  const int nvp = (nv + LPP - 1) / LPP * LPP;
  const size_t rec_per_warp = (size_t)LPP * PPW * 4 * sizeof(float4);
  const size_t spec_per_warp = (size_t)PPW * nvp * sizeof(float);
  int wpc = 4;
  while (wpc > 1 && wpc * (rec_per_warp + spec_per_warp) > 200 * 1024) wpc >>= 1;
  const size_t smem = wpc * (rec_per_warp + spec_per_warp);
  if (smem > 227 * 1024) return cudaErrorInvalidConfiguration;
  const int ppc = wpc * PPW;
  const unsigned grid = (unsigned)((npix + ppc - 1) / ppc);
  cudaError_t e;
  if (dust) {
    e = cudaFuncSetAttribute(transfer_series_kernel<LPP, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    transfer_series_kernel<LPP, true><<<grid, wpc * 32, smem, st>>>(mc, coef, ncell, npix, nz, nv, nvp, out, out_cont);
  } else {
    e = cudaFuncSetAttribute(transfer_series_kernel<LPP, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    transfer_series_kernel<LPP, false><<<grid, wpc * 32, smem, st>>>(mc, coef, ncell, npix, nz, nv, nvp, out, out_cont);
  }
  return cudaGetLastError();
}

inline cudaError_t launch_transfer_series(const MarchConsts& mc, const float* coef, int64_t ncell, int npix, int nz, int nv,
                                          bool dust, float* out, float* out_cont, cudaStream_t st) {
  return launch_transfer_series_lpp<8>(mc, coef, ncell, npix, nz, nv, dust, out, out_cont, st);
}

}  // namespace iris
