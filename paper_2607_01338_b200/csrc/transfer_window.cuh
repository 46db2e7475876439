// K3 (line-window formulation): LOS transfer that touches only the channels a cell can change.
//
// In a cell the erf-averaged profile (Eq. 4.6.3) is non-zero only within a few Doppler
// widths of v_los; everywhere else the step of Eq. 4.8.5 is the dust-only step, which is the same for the
// total and the continuum cube.  Marching the DIFFERENCE D = I^[T] - I^[C] (transfer_common.cuh) turns
// that step into a pure attenuation  D' = D E_d,  and storing  Dt = D * G_k,  G_k = exp(sum_{k'<k} tau_d)
// makes it the identity: channels outside the window need NO work, with or without dust.  The result is
// the same recurrence as the dense kernel, evaluated only where it differs from the identity.
//
// Window of a cell: |x| <= X_w with  exp(-X_w^2) * max(|a_c|, e_c) = 1e-8  (X_w <= 5.5): the profile mass
// dropped per cell is < 2e-9 in optical depth and in Kelvin.
//
// Mapping: a warp owns 32/LPP adjacent pixels, LPP lanes per pixel.  The spectrum Dt[nv] of each pixel
// lives in shared memory (bank-interleaved so that the lanes of a pixel always hit distinct banks and the
// pixels of a warp disjoint bank ranges).  Per cell, the LPP lanes sweep the window in passes of LPP
// channels; the erfc at a channel's upper edge comes from the neighbouring lane by one shuffle, so one
// erfc is evaluated per channel.  The continuum march (K4) and the running G are per-pixel scalars; the
// subtraction / unit conversion (K5) is the epilogue, written as 32-byte segments per pixel.
#pragma once
#include "transfer_common.cuh"

namespace iris {

// Channel window [klo, khi] of one cell (empty if the returned width is 0).
__device__ __forceinline__ int line_window(float e_c, float a_c, float c_los, float s, int nv, int& klo, int& khi) {
  const float sig = fmaxf(fabsf(a_c), e_c);
  const float Xw2 = __logf(sig) + 18.420681f;                  // ln(sig / 1e-8)
  const float Xw = fminf(sqrtf(fmaxf(Xw2, 0.0f)), IRIS_ERFC_TMAX);
  const float hw = Xw * rcp_approx(s);
  klo = max(0, (int)floorf(c_los - hw));
  khi = min(nv - 1, (int)floorf(c_los + hw));
  return (Xw2 > 0.0f) ? max(khi - klo + 1, 0) : 0;
}

// Sum of the window widths over all cells (work counter for roofline accounting).  fine_m > 0: the windows on the fine
// velocity grid of fine_m intervals per channel (points k / fine_m, as the series kernel's MODE 3 and the smooth window
// kernel see them).
__global__ void __launch_bounds__(256) window_work_kernel(const float* __restrict__ coef, int64_t ncell, int nv, int fine_m,
                                                          unsigned long long* __restrict__ total) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  int w = 0;
  if (i < ncell) {
    int klo, khi;
    if (fine_m > 0)
      w = line_window(coef[i], coef[ncell + i], fmaf(coef[2 * ncell + i], (float)fine_m, 0.5f), coef[3 * ncell + i] / (float)fine_m,
                      nv * fine_m + 1, klo, khi);
    else
      w = line_window(coef[i], coef[ncell + i], coef[2 * ncell + i], coef[3 * ncell + i], nv, klo, khi);
  }
  w = __reduce_add_sync(0xffffffffu, w);
  if ((threadIdx.x & 31) == 0 && w) atomicAdd(total, (unsigned long long)w);
}

// Work of the smooth window kernel: per (pixel, cell) the points of the HULL of the windows of the last `keep` cells (the
// union of the first two windows for the trapezoidal step).  One thread per pixel.
__global__ void __launch_bounds__(128) hull_work_kernel(const float* __restrict__ coef, int64_t ncell, int npix, int nz, int nv,
                                                        int fine_m, int keep, unsigned long long* __restrict__ total) {
  const int pix = blockIdx.x * blockDim.x + threadIdx.x;
  unsigned long long cnt = 0ull;
  if (pix < npix) {
    int lo[16], hi[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) { lo[k] = 0x7fffffff; hi[k] = -1; }
    const int npts = fine_m > 0 ? nv * fine_m + 1 : nv;
    for (int z = 0; z < nz; ++z) {
      const int64_t c = (int64_t)z * npix + pix;
      int klo, khi;
      const float cl = fine_m > 0 ? fmaf(coef[2 * ncell + c], (float)fine_m, 0.5f) : coef[2 * ncell + c];
      const float s = fine_m > 0 ? coef[3 * ncell + c] / (float)fine_m : coef[3 * ncell + c];
      const int W = line_window(coef[c], coef[ncell + c], cl, s, npts, klo, khi);
      // shift the remembered windows (static indexing keeps them in registers)
#pragma unroll
      for (int k = 15; k > 0; --k) { lo[k] = lo[k - 1]; hi[k] = hi[k - 1]; }
      lo[0] = W > 0 ? klo : 0x7fffffff; hi[0] = W > 0 ? khi : -1;
      if (z == 0) continue;
      int elo = 0x7fffffff, ehi = -1;
#pragma unroll
      for (int k = 0; k < 16; ++k)
        if (k < keep) { elo = min(elo, lo[k]); ehi = max(ehi, hi[k]); }
      if (ehi >= elo) cnt += (unsigned long long)(ehi - elo + 1);
    }
  }
  cnt = __reduce_add_sync(0xffffffffu, (unsigned)min(cnt, 0xffffffffull));
  if ((threadIdx.x & 31) == 0 && cnt) atomicAdd(total, cnt);
}

template <int LPP, bool DUST>
__global__ void __launch_bounds__(128)
transfer_window_kernel(MarchConsts mc, const float* __restrict__ coef, int64_t ncell, int npix, int nz, int nv,
                       int nvp, float* __restrict__ out, float* __restrict__ out_cont) {
  extern __shared__ float spec[];
  constexpr int PPW = 32 / LPP;
  constexpr unsigned FULL = 0xffffffffu;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, wpc = blockDim.x >> 5;
  const int g = lane / LPP, i = lane % LPP;
  const int pix = (blockIdx.x * wpc + warp) * PPW + g;
  const bool valid = pix < npix;
  const int pl = valid ? pix : npix - 1;
  // spectrum of pixel g of this warp: channel c at sp[(c / LPP) * 32 + (c % LPP)]
  float* sp = spec + (size_t)warp * nvp * PPW + g * LPP;
  for (int c = i; c < nvp; c += LPP) sp[(c / LPP) * 32 + i] = 0.0f;
  __syncwarp();

  float C = mc.T_bg;      // continuum before the current cell
  float G = 1.0f;         // exp(dust optical depth accumulated so far), since the last rescale
  const int nxt_lane = (lane & ~(LPP - 1)) | ((i + 1) & (LPP - 1));

  const float* p = coef + pl;
  float n_e = p[0], n_a = p[ncell], n_c = p[2 * ncell], n_s = p[3 * ncell];
  float n_td = DUST ? p[4 * ncell] : 0.0f, n_sd = DUST ? p[5 * ncell] : 0.0f;

  for (int z = 0; z < nz; ++z) {
    const float e_c = n_e, a_c = n_a, c_los = n_c, s = n_s, tau_d = n_td, S_d = n_sd;
    if (z + 1 < nz) {
      p += npix;
      n_e = p[0]; n_a = p[ncell]; n_c = p[2 * ncell]; n_s = p[3 * ncell];
      if (DUST) { n_td = p[4 * ncell]; n_sd = p[5 * ncell]; }
    }
    // line window
    int klo, khi;
    const int W = line_window(e_c, a_c, c_los, s, nv, klo, khi);
    const int npass = __reduce_max_sync(FULL, (W + LPP - 1) / LPP);

    DustStep d;
    float CG = 0.0f, Gn = 1.0f, sc = 0.0f;
    if (DUST) {
      d.tau_d = tau_d; d.S_d = S_d; d.C = C;
      const float td_e = fminf(tau_d, kMaxTauDCell);
      d.E_d = exp_neg(td_e);
      d.m_d = one_minus_exp_neg(td_e);
      CG = C * G;
      Gn = G * ex2_approx(td_e * 1.4426950408889634f);           // G after this cell
      C = fmaf(C, d.E_d, S_d * d.m_d);
    } else {
      sc = (a_c != 0.0f ? e_c / a_c : 0.0f) - C;
    }

    if (npass > 0) {
      float x_lo = ((float)(klo + i) - c_los) * s;
      float G_cur = signed_erfc(x_lo);
      const float step = (float)LPP * s;
      int c = klo + i;
      for (int ps = 0; ps < npass; ++ps) {
        const float x_nx = x_lo + step;
        const float G_nx = signed_erfc(x_nx);
        const float G_hi = __shfl_sync(FULL, i == 0 ? G_nx : G_cur, nxt_lane);
        // the signs are taken from G itself (G carries the sign of the x it was evaluated at), so the edge
        // shared by two lanes is seen identically by both even when x = 0 rounds differently
        const float dErf = (copysignf(1.0f, G_hi) - copysignf(1.0f, G_cur)) - (G_hi - G_cur);
        if (c <= khi && W > 0) {
          float* q = sp + (c / LPP) * 32 + (c % LPP);
          float Dt = *q;
          if (DUST) {
            // Dt' = Dt - (Dt + C G) m + G' [J_L (m_d + E_d m) + S_d (tau_d E_d m - tau_L m_d)] / tau_T
            const float tau_L = a_c * dErf, J_L = e_c * dErf;
            const float m = one_minus_exp_neg(tau_L);
            const float tau_T = tau_L + tau_d;
            const float r = rcp_approx(tau_T == 0.0f ? 1.0f : tau_T);
            const float Em = d.E_d * m;
            const float t1 = d.m_d + Em;
            const float t2 = fmaf(tau_d, Em, -tau_L * d.m_d);
            const float num = fmaf(J_L, t1, S_d * t2);
            Dt = fmaf(-(Dt + CG), m, Dt);
            Dt = fmaf(Gn * r, num, Dt);
          } else {
            Dt = update_nodust(Dt, dErf, a_c, sc);
          }
          *q = Dt;
        }
        x_lo = x_nx; G_cur = G_nx; c += LPP;
      }
    }
    if (DUST) {
      G = Gn;
      if (G > kFoldG) {   // rare: fold the accumulated dust attenuation into the stored spectrum
        const float inv = 1.0f / G;
        __syncwarp(__activemask());
        for (int cc = i; cc < nvp; cc += LPP) sp[(cc / LPP) * 32 + i] *= inv;
        G = 1.0f;
      }
    }
    __syncwarp();
  }

  const float invG = 1.0f / G;
  if (valid) {
    if (out != nullptr) {
      float* o = out + (int64_t)pix * nv;
      for (int c = i; c < nv; c += LPP) o[c] = convert_out(sp[(c / LPP) * 32 + i] * invG, C, mc);
    }
    if (out_cont != nullptr && i == 0) out_cont[pix] = C * mc.inv_KRJ;
  }
}

// Picks lanes-per-pixel and CTA size from nv (shared memory per CTA = warps * (32/LPP) * nvp * 4 B).
inline cudaError_t launch_transfer_window(const MarchConsts& mc, const float* coef, int64_t ncell, int npix, int nz, int nv,
                                          bool dust, int sm_count, float* out, float* out_cont, cudaStream_t st) {
  constexpr int LPP = 8, PPW = 32 / LPP;
  const int nvp = (nv + LPP - 1) / LPP * LPP;
  int wpc = 4;
  while (wpc > 1 && (size_t)wpc * PPW * nvp * sizeof(float) > 200 * 1024) wpc >>= 1;
  const size_t smem = (size_t)wpc * PPW * nvp * sizeof(float);
  if (smem > 227 * 1024) return cudaErrorInvalidConfiguration;
  const int ppc = wpc * PPW;
  const unsigned grid = (unsigned)((npix + ppc - 1) / ppc);
  (void)sm_count;
  cudaError_t e;
  if (dust) {
    e = cudaFuncSetAttribute(transfer_window_kernel<LPP, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    transfer_window_kernel<LPP, true><<<grid, wpc * 32, smem, st>>>(mc, coef, ncell, npix, nz, nv, nvp, out, out_cont);
  } else {
    e = cudaFuncSetAttribute(transfer_window_kernel<LPP, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    transfer_window_kernel<LPP, false><<<grid, wpc * 32, smem, st>>>(mc, coef, ncell, npix, nz, nv, nvp, out, out_cont);
  }
  return cudaGetLastError();
}

}  // namespace iris
