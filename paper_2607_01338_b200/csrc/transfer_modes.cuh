// K3 in the paper's OTHER transfer / integration modes (PAPER.md sections 4.4 - 4.8); the hot path (optically thick,
// formal integration, channel-integrated profile) is transfer_series.cuh / transfer_window.cuh.
//
//   transfer mode   0 optically thick    Eq. 4.8.6 - 4.8.8  (line absorbs itself)
//                   1 selectively thin   Eq. 4.8.13 - 4.8.15 (line absorbs only the continuum, dust absorbs the line)
//                   2 optically thin     Eq. 4.7.3 - 4.7.5  (no absorption)
//   integration     0 formal             Eq. 4.8.5 (exponential step) / Eq. 4.7.6 (midpoint sum)
//                   1 smooth             Eq. 4.8.12 (trapezoidal first step) + Eq. 4.8.10 (BDF2), ReLU after every step;
//                                        Eq. 4.7.7 (Simpson along the ray) in the thin mode
//   profile         channel-integrated   Eq. 4.6.3 (erf difference), one spectral point per channel
//                   fine grid            Eq. 3.3.3 at f + 2 points per channel, Simpson over frequency, Eq. 4.5.1
//                                        (thick mode, "subsampling factor" f odd)
//
// Everything is marched in the DIFFERENCE form D = I^[T] - I^[C] next to the scalar continuum C (Rayleigh-Jeans Kelvin),
// as in transfer_common.cuh.  With  E = e_c p  (= h j_L),  A = a_c p  (= h alpha_L),  t_d = tau_d,  J_d = tau_d S_d
// for the profile weight p of a spectral point in a cell, subtracting the continuum recurrence from the total one gives
//   thin, formal      D += E                                    C += J_d
//   thin, smooth      D += w_n E,  C += w_n J_d                 w_n: Simpson weights along the ray (reading S25)
//   sel. thin, formal D' = E_d D + (E - A C') w(t_d)            C' = E_d C + S_d m_d,  w = (1 - e^-t) / t
//   smooth, first     D_1 = [(E_0 - A_0 C_0) + (E_1 - A_1 C_1) + (2 - a_0) D_0] / (2 + a_1)      (TR, Eq. 4.8.12)
//   smooth, n >= 2    D_n = [2 (E_n - A_n C_n) + 4 D_n-1 - D_n-2] / (3 + 2 a_n)                   (BDF2, Eq. 4.8.10)
//                     a_n = A_n + t_d,n (thick) or t_d,n (selectively thin);  C_n by the same formulas with E = A = 0
// none of which cancels.  The ReLU acts on the true intensities: I^[T] = D + C >= 0, C >= 0 (reading S26).
//
// Mapping: a thread owns one pixel and NPT consecutive spectral points in registers (8 channels with their 9 shared
// erfc edges, or the 9 fine points of 8 / m channels, or one Simpson panel of 3 points at a time for finer grids); lanes
// run along pixels, so the six coefficient planes are read with 128-byte coalesced loads and the per-cell continuum /
// dust scalars are computed once per NPT points; a block of points farther than 5.5 Doppler widths from the line centre
// skips the profile evaluation (its weights are zero); each thread writes its channels as contiguous 16-byte stores.
#pragma once
#include "transfer_common.cuh"

namespace iris {

struct ModeConsts {
  int mode, smooth;      // transfer mode 0 / 1 / 2, integration 0 / 1
  int fine_m;            // 0: channel-integrated profile; else fine intervals per channel (f + 1, even)
  int nx;                // pixels per image row (npix = nx * rows)
  const int* gate;       // nullptr, or the device counter of the pixels transfer_smooth_window_kernel handed over
                         // (transfer_smooth.cuh): the kernel then recomputes those pixels only (none: it returns at once)
  const int* list;       // their pixel indices, gate[0] of them
};

// w(t) = (1 - exp(-t)) / t, w(0) = 1
__device__ __forceinline__ float w_of(float t) {
  return fabsf(t) < 1.0e-3f ? fmaf(t, fmaf(t, 1.0f / 6.0f, -0.5f), 1.0f) : one_minus_exp_neg(t) / t;
}

constexpr int kModesCh0 = 16;         // channels per thread with the channel-integrated profile (PROF 0)
constexpr float kModesXmax = 5.5f;     // profile weights beyond this many Doppler widths are dropped (< 1e-13 of the peak)

// PROF 0: channel-integrated profile, kModesCh0 channels per thread (NPT weights from NPT + 1 edges)
// PROF 1: fine grid with m = 4 or 8 intervals per channel: 9 points = 8 / m channels per thread
// PROF 3: fine grid with m = 2 (the paper's production mode, f = 1): 17 points = 8 channels per thread
// PROF 2: fine grid, any even m: one channel per thread, one Simpson panel (3 points) per march
template <int MODE, bool SMOOTH, int PROF>
__global__ void __launch_bounds__(128)
transfer_modes_kernel(MarchConsts mc, ModeConsts md, const float* __restrict__ coef, int64_t ncell, int npix, int nz,
                      int nv, float* __restrict__ out, float* __restrict__ out_cont) {
  constexpr int NPT = PROF == 0 ? kModesCh0 : (PROF == 1 ? 9 : (PROF == 3 ? 17 : 3));
  // a warp takes a tile of 8 x 4 pixels: whole 32-byte sectors of every plane, and a quarter of the spread in
  // line-of-sight velocity that 32 pixels along x have (the dust-only path is taken when NO pixel of the warp is near
  // the line, and rotation shifts the line by several channels per pixel along x)
  const int tiles_x = (md.nx + 7) >> 3;
  const int px = (blockIdx.x % tiles_x) * 8 + (threadIdx.x & 7), py = (blockIdx.x / tiles_x) * 4 + (threadIdx.x >> 3);
  int pix = px < md.nx ? py * md.nx + px : npix;
  if (md.gate != nullptr) {
    // hand-over launch: thread slot -> entry of the list of flagged pixels (the grid is sized for all pixels; the blocks
    // beyond the list return at once)
    const int slot = blockIdx.x * 32 + threadIdx.x;
    pix = slot < *md.gate ? md.list[slot] : npix;
  }
  const int blk = blockIdx.y * blockDim.y + threadIdx.y;      // channel block of this thread
  const int m = md.fine_m;
  const int cpb = PROF == 0 ? kModesCh0 : (PROF == 3 ? 8 : (PROF == 1 ? 8 / m : 1));    // channels per thread
  const int v0 = blk * cpb;
  if (pix >= npix || v0 >= nv) return;
  const int npanel = PROF == 2 ? m / 2 : 1;
  const float inv_m = PROF == 0 ? 1.0f : 1.0f / (float)m;
  const int Rs = (nz & 1) ? nz : nz - 1;                      // points covered by whole Simpson panels along the ray
  float Dacc = 0.0f, Cfin = mc.T_bg;
  float Dfin[NPT];

  for (int panel = 0; panel < npanel; ++panel) {
    float D[NPT], Dm[NPT];
#pragma unroll
    for (int k = 0; k < NPT; ++k) D[k] = Dm[k] = 0.0f;
    float C = mc.T_bg, Cm = mc.T_bg;
    // position (channel-edge index units) of point 0 and spacing of the points
    const float pos0 = PROF == 2 ? (float)v0 + (float)(2 * panel) * inv_m : (float)v0;
    const float dpos = PROF == 0 ? 1.0f : inv_m;
    const float* p = coef + pix;
    // the coefficients of the next cell are loaded one cell ahead (the march of a point is a dependent chain)
    float n_e = p[0], n_a = p[ncell], n_c = p[2 * ncell], n_s = p[3 * ncell], n_td = p[4 * ncell], n_sd = p[5 * ncell];
    // One cell.  Dc holds the points at grid index n - 1 and Dp those at n - 2; the new values are written over Dp, so
    // the caller alternates the two arrays instead of moving 2 NPT registers per cell (modes without a second-order
    // history pass the same array twice).
    auto step = [&](const int n, float (&Dc)[NPT], float (&Dp)[NPT]) {
      const float e_c = n_e, a_c = n_a, c_los = n_c, s = n_s, td = n_td, Sd = n_sd;
      if (n + 1 < nz) {
        p += npix;
        n_e = p[0]; n_a = p[ncell]; n_c = p[2 * ncell]; n_s = p[3 * ncell]; n_td = p[4 * ncell]; n_sd = p[5 * ncell];
      }
      // the trapezoidal first step also needs the coefficients of grid index 0
      float e_p = 0.0f, a_p = 0.0f, c_p = 0.0f, s_p = 1.0f, td_p = 0.0f, Jd_p = 0.0f;
      if (SMOOTH && MODE != 2 && n == 1) {
        const float* q = coef + pix;
        e_p = q[0]; a_p = q[ncell]; c_p = q[2 * ncell]; s_p = q[3 * ncell]; td_p = q[4 * ncell];
        Jd_p = td_p * q[5 * ncell];
      }
      const float Jd = td * Sd;
      float wn = 0.0f;
      if (MODE == 2 && SMOOTH) {
        if (Rs >= 3 && n < Rs) wn = (n == 0 || n == Rs - 1) ? (1.0f / 3.0f) : ((n & 1) ? (4.0f / 3.0f) : (2.0f / 3.0f));
        if (!(nz & 1) && nz >= 2 && n >= nz - 2) wn += 0.5f;
      }
      // ---- per-cell scalars: continuum step, dust factors
      float C_unc;
      if (MODE == 2) C_unc = SMOOTH ? fmaf(wn, Jd, C) : C + Jd;
      else if (!SMOOTH) C_unc = fmaf(C, exp_neg(td), Sd * one_minus_exp_neg(td));
      else if (n == 0) C_unc = C;
      else if (n == 1) C_unc = (Jd_p + Jd + (2.0f - td_p) * C) * rcp_approx(2.0f + td);
      else C_unc = (2.0f * Jd + 4.0f * C - Cm) * rcp_approx(fmaf(2.0f, td, 3.0f));
      const float Cn = (MODE != 2 && (SMOOTH || MODE == 1)) ? fmaxf(C_unc, 0.0f) : C_unc;
      // ReLU of the smooth integrator on D: D' = relu(Du + C_unc) - relu(C_unc) = max(Du + relu_add, relu_min) with
      // (0, -C_unc) where the continuum is not clamped and (C_unc, 0) where it is
      const float relu_add = C_unc >= 0.0f ? 0.0f : C_unc, relu_min = C_unc >= 0.0f ? -C_unc : 0.0f;
      float Ed = 1.0f, wd = 1.0f;
      DustStep ds;
      if (MODE == 1 && !SMOOTH) { Ed = exp_neg(td); wd = w_of(td); }
      if (MODE == 0 && !SMOOTH) {
        ds.tau_d = td; ds.S_d = Sd; ds.C = C;
        ds.E_d = exp_neg(td);
        ds.m_d = one_minus_exp_neg(td);
      }
      // ---- profile weights of the NPT points in this cell ("erf-difference" units); zero far from the line
      float pw[NPT], pwp[NPT];
      const float x0 = (pos0 - c_los) * s;
      const float x1 = x0 + (PROF == 0 ? (float)NPT : (float)(NPT - 1) * dpos) * s;
      const bool near = x0 < kModesXmax && x1 > -kModesXmax;
      if (near) {
        if (PROF == 0) {
          float G_lo = signed_erfc(x0), xl = x0;
#pragma unroll
          for (int k = 0; k < NPT; ++k) {
            const float xh = ((pos0 + (float)(k + 1)) - c_los) * s;
            const float G_hi = signed_erfc(xh);
            pw[k] = erf_diff(xl, G_lo, xh, G_hi);
            xl = xh; G_lo = G_hi;
          }
        } else {
#pragma unroll
          for (int k = 0; k < NPT; ++k) {
            const float x = ((pos0 + (float)k * dpos) - c_los) * s;
            pw[k] = fabsf(x) < kModesXmax ? 1.1283791670955126f * s * ex2_approx(-1.4426950408889634f * x * x) : 0.0f;
          }
        }
      } else {
#pragma unroll
        for (int k = 0; k < NPT; ++k) pw[k] = 0.0f;
      }
      if (SMOOTH && MODE != 2 && n == 1) {            // trapezoidal first step needs the weights of grid index 0 too
        if (PROF == 0) {
          float xl = (pos0 - c_p) * s_p, G_lo = signed_erfc(xl);
#pragma unroll
          for (int k = 0; k < NPT; ++k) {
            const float xh = ((pos0 + (float)(k + 1)) - c_p) * s_p;
            const float G_hi = signed_erfc(xh);
            pwp[k] = (fabsf(xl) < kModesXmax || fabsf(xh) < kModesXmax) ? erf_diff(xl, G_lo, xh, G_hi) : 0.0f;
            xl = xh; G_lo = G_hi;
          }
        } else {
#pragma unroll
          for (int k = 0; k < NPT; ++k) {
            const float x = ((pos0 + (float)k * dpos) - c_p) * s_p;
            pwp[k] = fabsf(x) < kModesXmax ? 1.1283791670955126f * s_p * ex2_approx(-1.4426950408889634f * x * x) : 0.0f;
          }
        }
      }
      // ---- far from the line every weight is zero: the step of every point is the dust-only step
      if (!near && !(SMOOTH && MODE != 2 && n == 1)) {
        if (MODE == 2) {
          // nothing is emitted into these points
        } else if (!SMOOTH) {
          const float att = MODE == 1 ? Ed : ds.E_d;
#pragma unroll
          for (int k = 0; k < NPT; ++k) {
            const float Dn = Dc[k] * att;
            Dp[k] = MODE == 1 ? fmaxf(Dn, -Cn) : Dn;
          }
        } else if (n >= 2) {
          const float r = rcp_approx(fmaf(2.0f, td, 3.0f));
#pragma unroll
          for (int k = 0; k < NPT; ++k) Dp[k] = fmaxf(fmaf(fmaf(4.0f, Dc[k], -Dp[k]), r, relu_add), relu_min);
        } else {
#pragma unroll
          for (int k = 0; k < NPT; ++k) Dp[k] = Dc[k];      // n = 0 of the smooth march: nothing happens yet
        }
        Cm = C; C = Cn;
        return;
      }
      // ---- the step of every point
#pragma unroll
      for (int k = 0; k < NPT; ++k) {
        const float E = e_c * pw[k], A = a_c * pw[k];
        const float Dk = Dc[k];
        float Dn;
        if (MODE == 2) {
          Dn = SMOOTH ? fmaf(wn, E, Dk) : Dk + E;
        } else if (!SMOOTH) {
          if (MODE == 1) Dn = fmaxf(fmaf(Dk, Ed, (E - A * Cn) * wd), -Cn);       // ReLU on I_T = D + C (C' >= 0 here)
          else Dn = update_dust(Dk, pw[k], e_c, a_c, ds);                       // Eq. 4.8.5 in difference form
        } else {
          const float Ccoef = MODE == 0 ? C_unc : Cn;    // continuum the line term is paired with (see header)
          float Du;
          if (n == 0) Du = 0.0f;
          else if (n == 1) {
            const float Ep = e_p * pwp[k], Ap = a_p * pwp[k];
            const float a0 = (MODE == 0 ? Ap : 0.0f) + td_p, a1 = (MODE == 0 ? A : 0.0f) + td;
            Du = ((Ep - Ap * C) + (E - A * Ccoef) + (2.0f - a0) * Dk) * rcp_approx(2.0f + a1);
          } else {
            const float an = (MODE == 0 ? A : 0.0f) + td;
            Du = (2.0f * (E - A * Ccoef) + 4.0f * Dk - Dp[k]) * rcp_approx(fmaf(2.0f, an, 3.0f));
          }
          // ReLU on the true intensities: I_T = relu(Du + C_unc), C = relu(C_unc)
          Dn = fmaxf(Du + relu_add, relu_min);
        }
        Dp[k] = Dn;
      }
      Cm = C; C = Cn;
    };
    bool in_Dm = false;                 // which array holds the final points
    if (SMOOTH && MODE != 2) {
      int n = 0;
      for (; n + 1 < nz; n += 2) { step(n, D, Dm); step(n + 1, Dm, D); }
      if (n < nz) { step(n, D, Dm); in_Dm = true; }
    } else {
      for (int n = 0; n < nz; ++n) step(n, D, D);
    }
    if (in_Dm) {
#pragma unroll
      for (int k = 0; k < NPT; ++k) D[k] = Dm[k];
    }
    Cfin = C;
    if (PROF == 2) Dacc += (D[0] + 4.0f * D[1] + D[2]) * (inv_m * (1.0f / 3.0f));
#pragma unroll
    for (int k = 0; k < NPT; ++k) Dfin[k] = D[k];
  }

  // ---- channel values of this thread -> convert and store
  // (modes with the ReLU keep I_T = D + C >= 0 point by point, hence for a Simpson average too; the clamp below only
  // removes the rounding of the average)
  constexpr bool RELU = MODE != 2 && (SMOOTH || MODE == 1);
  auto conv = [&](float D) { return convert_out(RELU ? fmaxf(D, -Cfin) : D, Cfin, mc); };
  constexpr int NRES = PROF == 0 ? kModesCh0 : 8;
  float res[NRES];
  int nch = min(cpb, nv - v0);
  if constexpr (PROF == 0) {
#pragma unroll
    for (int k = 0; k < NRES; ++k) res[k] = conv(Dfin[k]);
  } else if constexpr (PROF == 3) {
#pragma unroll
    for (int c = 0; c < 8; ++c)
      res[c] = conv((Dfin[2 * c] + 4.0f * Dfin[2 * c + 1] + Dfin[2 * c + 2]) * (1.0f / 6.0f));
  } else if constexpr (PROF == 1) {
#pragma unroll
    for (int c = 0; c < 4; ++c) {                     // at most 2 channels (m = 4)
      float acc = 0.0f;
#pragma unroll
      for (int j = 0; j < 8; j += 2) {                // panels of the channel: points c m + j .. c m + j + 2, j < m
        const int q = c * m + j;
        if (j < m && c < cpb) {
          float d0 = 0.0f, d1 = 0.0f, d2 = 0.0f;
#pragma unroll
          for (int k = 0; k < NPT; ++k) {             // static indexing keeps Dfin in registers
            if (k == q) d0 = Dfin[k];
            if (k == q + 1) d1 = Dfin[k];
            if (k == q + 2) d2 = Dfin[k];
          }
          acc += d0 + 4.0f * d1 + d2;
        }
      }
      res[c] = conv(acc * (inv_m * (1.0f / 3.0f)));
    }
  } else {
    res[0] = conv(Dacc);
  }
  if (out != nullptr) {
    float* o = out + (int64_t)pix * nv + v0;
    if ((PROF == 0 || PROF == 3) && nch == NRES && (((int64_t)pix * nv + v0) & 3) == 0) {
#pragma unroll
      for (int k = 0; k < NRES; k += 4)
        reinterpret_cast<float4*>(o)[k / 4] = make_float4(res[k], res[k + 1], res[k + 2], res[k + 3]);
    } else {
#pragma unroll
      for (int k = 0; k < NRES; ++k)
        if (k < nch) o[k] = res[k];
    }
  }
  if (out_cont != nullptr && blk == 0) out_cont[pix] = Cfin * mc.inv_KRJ;
}

template <int MODE, bool SMOOTH>
inline cudaError_t launch_transfer_modes_t(const MarchConsts& mc, const ModeConsts& md, const float* coef, int64_t ncell,
                                           int npix, int nz, int nv, float* out, float* out_cont, cudaStream_t st) {
  const int m = md.fine_m;
  const int prof = m == 0 ? 0 : (m == 2 ? 3 : ((m == 4 || m == 8) ? 1 : 2));
  const int cpb = prof == 0 ? kModesCh0 : (prof == 3 ? 8 : (prof == 1 ? 8 / m : 1));
  const int nblk = (nv + cpb - 1) / cpb;
  const int rows = npix / md.nx;
  dim3 block(32, 4), grid(md.gate != nullptr ? (npix + 31) / 32 : ((md.nx + 7) / 8) * ((rows + 3) / 4), (nblk + 3) / 4);
  if (prof == 0) transfer_modes_kernel<MODE, SMOOTH, 0><<<grid, block, 0, st>>>(mc, md, coef, ncell, npix, nz, nv, out, out_cont);
  else if (prof == 1) transfer_modes_kernel<MODE, SMOOTH, 1><<<grid, block, 0, st>>>(mc, md, coef, ncell, npix, nz, nv, out, out_cont);
  else if (prof == 3) transfer_modes_kernel<MODE, SMOOTH, 3><<<grid, block, 0, st>>>(mc, md, coef, ncell, npix, nz, nv, out, out_cont);
  else transfer_modes_kernel<MODE, SMOOTH, 2><<<grid, block, 0, st>>>(mc, md, coef, ncell, npix, nz, nv, out, out_cont);
  return cudaGetLastError();
}

inline cudaError_t launch_transfer_modes(const MarchConsts& mc, const ModeConsts& md, const float* coef, int64_t ncell,
                                         int npix, int nz, int nv, float* out, float* out_cont, cudaStream_t st) {
  switch (md.mode * 2 + (md.smooth ? 1 : 0)) {
    case 0: return launch_transfer_modes_t<0, false>(mc, md, coef, ncell, npix, nz, nv, out, out_cont, st);
    case 1: return launch_transfer_modes_t<0, true>(mc, md, coef, ncell, npix, nz, nv, out, out_cont, st);
    case 2: return launch_transfer_modes_t<1, false>(mc, md, coef, ncell, npix, nz, nv, out, out_cont, st);
    case 3: return launch_transfer_modes_t<1, true>(mc, md, coef, ncell, npix, nz, nv, out, out_cont, st);
    case 4: return launch_transfer_modes_t<2, false>(mc, md, coef, ncell, npix, nz, nv, out, out_cont, st);
    default: return launch_transfer_modes_t<2, true>(mc, md, coef, ncell, npix, nz, nv, out, out_cont, st);
  }
}

}  // namespace iris
