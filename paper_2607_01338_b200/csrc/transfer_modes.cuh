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
// Mapping: a CTA is 32 pixels x 8 channels; lanes run along pixels, so the six coefficient planes are read with
// 128-byte coalesced loads (every plane of a column is re-read once per 8 channels, from L2); the result tile is
// transposed through shared memory so that each pixel writes 32 contiguous bytes.
#pragma once
#include "transfer_common.cuh"

namespace iris {

struct ModeConsts {
  int mode, smooth;      // transfer mode 0 / 1 / 2, integration 0 / 1
  int fine_m;            // 0: channel-integrated profile; else fine intervals per channel (f + 1, even)
};

// State of one spectral point: D at the last two grid indices.
struct ModePoint { float D, Dm; };

// Continuum step at grid index n (n = 0: initial condition).  Returns the new continuum; *C_unc receives the value
// before the ReLU (the difference recurrences are derived from the unclamped relation).
__device__ __forceinline__ float continuum_step(const ModeConsts& md, int n, float C, float Cm, float td, float Jd,
                                                float Sd, float td_prev, float Jd_prev, float wn, float* C_unc) {
  float c;
  if (md.mode == 2) c = md.smooth ? fmaf(wn, Jd, C) : C + Jd;
  else if (!md.smooth) c = fmaf(C, exp_neg(td), Sd * one_minus_exp_neg(td));
  else if (n == 0) c = C;
  else if (n == 1) c = (Jd_prev + Jd + (2.0f - td_prev) * C) / (2.0f + td);
  else c = (2.0f * Jd + 4.0f * C - Cm) / fmaf(2.0f, td, 3.0f);
  *C_unc = c;
  return (md.mode != 2 && (md.smooth || md.mode == 1)) ? fmaxf(c, 0.0f) : c;
}

// w(t) = (1 - exp(-t)) / t, w(0) = 1
__device__ __forceinline__ float w_of(float t) {
  return fabsf(t) < 1.0e-3f ? fmaf(t, fmaf(t, 1.0f / 6.0f, -0.5f), 1.0f) : one_minus_exp_neg(t) / t;
}

template <int NP>
__global__ void __launch_bounds__(256)
transfer_modes_kernel(MarchConsts mc, ModeConsts md, const float* __restrict__ coef, int64_t ncell, int npix, int nz,
                      int nv, float* __restrict__ out, float* __restrict__ out_cont) {
  __shared__ float tile[8][33];
  const int lane = threadIdx.x, ty = threadIdx.y;
  const int pix = blockIdx.x * 32 + lane;
  const int v = blockIdx.y * 8 + ty;
  const bool active = pix < npix && v < nv;
  const int pl = min(pix, npix - 1);
  const int m = md.fine_m;
  const int npanel = m > 0 ? m / 2 : 1;
  const bool dust = true;      // tau_d = 0 planes when dust is off: the same formulas hold
  (void)dust;
  float Dacc = 0.0f, Cfin = mc.T_bg;

  for (int panel = 0; panel < npanel; ++panel) {
    ModePoint pt[NP];
#pragma unroll
    for (int k = 0; k < NP; ++k) pt[k].D = pt[k].Dm = 0.0f;
    float C = mc.T_bg, Cm = mc.T_bg;
    float e_p = 0.0f, a_p = 0.0f, c_p = 0.0f, s_p = 1.0f, td_p = 0.0f, Jd_p = 0.0f;   // coefficients of grid index n - 1
    const float* p = coef + pl;
    const int Rs = (nz & 1) ? nz : nz - 1;               // points covered by whole Simpson panels along the ray
    for (int n = 0; n < nz; ++n, p += npix) {
      const float e_c = p[0], a_c = p[ncell], c_los = p[2 * ncell], s = p[3 * ncell];
      const float td = p[4 * ncell], Sd = p[5 * ncell];
      const float Jd = td * Sd;
      float wn = 0.0f;
      if (md.mode == 2 && md.smooth) {
        if (Rs >= 3 && n < Rs) wn = (n == 0 || n == Rs - 1) ? (1.0f / 3.0f) : ((n & 1) ? (4.0f / 3.0f) : (2.0f / 3.0f));
        if (!(nz & 1) && nz >= 2 && n >= nz - 2) wn += 0.5f;
      }
      float C_unc;
      const float Cn = continuum_step(md, n, C, Cm, td, Jd, Sd, td_p, Jd_p, wn, &C_unc);
      const float Ed = (md.mode == 1 && !md.smooth) ? exp_neg(td) : 1.0f;
      const float wd = (md.mode == 1 && !md.smooth) ? w_of(td) : 1.0f;
      DustStep ds;
      if (md.mode == 0 && !md.smooth) {
        ds.tau_d = td; ds.S_d = Sd; ds.C = C;
        ds.E_d = exp_neg(td);
        ds.m_d = one_minus_exp_neg(td);
      }
#pragma unroll
      for (int k = 0; k < NP; ++k) {
        // profile weight of this point in this cell (in "erf-difference" units) and of the previous cell
        float pw, pw_prev = 0.0f;
        if (m == 0) {
          const float x_lo = ((float)v - c_los) * s, x_hi = ((float)(v + 1) - c_los) * s;
          pw = erf_diff(x_lo, signed_erfc(x_lo), x_hi, signed_erfc(x_hi));
          if (md.smooth && n == 1) {
            const float y_lo = ((float)v - c_p) * s_p, y_hi = ((float)(v + 1) - c_p) * s_p;
            pw_prev = erf_diff(y_lo, signed_erfc(y_lo), y_hi, signed_erfc(y_hi));
          }
        } else {
          const float pos = (float)v + (float)(2 * panel + k) / (float)m;      // channel-edge index units
          const float x = (pos - c_los) * s;
          pw = 1.1283791670955126f * s * ex2_approx(-1.4426950408889634f * x * x);
          if (md.smooth && n == 1) {
            const float y = (pos - c_p) * s_p;
            pw_prev = 1.1283791670955126f * s_p * ex2_approx(-1.4426950408889634f * y * y);
          }
        }
        const float E = e_c * pw, A = a_c * pw;
        float D = pt[k].D, Dn;
        if (md.mode == 2) {
          Dn = md.smooth ? fmaf(wn, E, D) : D + E;
        } else if (!md.smooth) {
          if (md.mode == 1) {
            Dn = fmaf(D, Ed, (E - A * Cn) * wd);
            Dn = fmaxf(Dn, -Cn);                           // ReLU on I_T = D + C (C' >= 0 here)
          } else {
            Dn = update_dust(D, pw, e_c, a_c, ds);         // Eq. 4.8.5 in difference form (transfer_common.cuh)
          }
        } else {
          const float Ccoef = md.mode == 0 ? C_unc : Cn;   // continuum the line term is paired with (see header)
          float Du;
          if (n == 0) Du = 0.0f;
          else if (n == 1) {
            const float Ep = e_p * pw_prev, Ap = a_p * pw_prev;
            const float a0 = (md.mode == 0 ? Ap : 0.0f) + td_p, a1 = (md.mode == 0 ? A : 0.0f) + td;
            Du = ((Ep - Ap * C) + (E - A * Ccoef) + (2.0f - a0) * D) / (2.0f + a1);
          } else {
            const float an = (md.mode == 0 ? A : 0.0f) + td;
            Du = (2.0f * (E - A * Ccoef) + 4.0f * D - pt[k].Dm) / fmaf(2.0f, an, 3.0f);
          }
          // ReLU on the true intensities: I_T = relu(Du + C_unc), C = relu(C_unc)
          Dn = (C_unc >= 0.0f) ? fmaxf(Du, -C_unc) : fmaxf(Du + C_unc, 0.0f);
        }
        pt[k].Dm = D;
        pt[k].D = Dn;
      }
      Cm = C; C = Cn;
      e_p = e_c; a_p = a_c; c_p = c_los; s_p = s; td_p = td; Jd_p = Jd;
    }
    Cfin = C;
    if (m == 0) Dacc = pt[0].D;
    else Dacc += (pt[0].D + 4.0f * pt[NP > 1 ? 1 : 0].D + pt[NP > 2 ? 2 : 0].D) / (3.0f * (float)m);
  }

  tile[ty][lane] = active ? convert_out(Dacc, Cfin, mc) : 0.0f;
  __syncthreads();
  if (out != nullptr) {
    const int t = ty * 32 + lane;
    const int pp = t >> 3, cc = t & 7;
    const int opix = blockIdx.x * 32 + pp, ov = blockIdx.y * 8 + cc;
    if (opix < npix && ov < nv) out[(int64_t)opix * nv + ov] = tile[cc][pp];
  }
  if (out_cont != nullptr && blockIdx.y == 0 && ty == 0 && pix < npix) out_cont[pix] = Cfin * mc.inv_KRJ;
}

inline cudaError_t launch_transfer_modes(const MarchConsts& mc, const ModeConsts& md, const float* coef, int64_t ncell,
                                         int npix, int nz, int nv, float* out, float* out_cont, cudaStream_t st) {
  dim3 block(32, 8), grid((npix + 31) / 32, (nv + 7) / 8);
  if (md.fine_m > 0) transfer_modes_kernel<3><<<grid, block, 0, st>>>(mc, md, coef, ncell, npix, nz, nv, out, out_cont);
  else transfer_modes_kernel<1><<<grid, block, 0, st>>>(mc, md, coef, ncell, npix, nz, nv, out, out_cont);
  return cudaGetLastError();
}

}  // namespace iris
