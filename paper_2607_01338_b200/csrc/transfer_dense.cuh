// K3 (dense formulation): LOS transfer with register-resident channel blocks.
//
// Thread <-> (pixel, block of CB consecutive channels).  A warp holds an 8 x 4 tile of pixels of the sky plane
// (whole 32-byte sectors of every plane; a quarter of the spread in line-of-sight velocity that 32 pixels
// along x have, so fewer warps have to evaluate a block that only some of their pixels need) and one channel
// block; the six planes are read once per z step and reused for the CB channels a thread keeps in registers.  The
// CB + 1 channel edges of a block share their erfc evaluations.  A block farther than the erfc fit range
// from the line centre only attenuates by the dust (D *= E_d) -- exact in fp32 because erfc underflows
// the fp32 sum there.  The continuum march (K4) is a scalar per thread; subtraction / unit conversion
// (K5) is the epilogue.  Output: CB consecutive floats per thread (float4 stores).
//
// PERCH (dust_per_channel = 1; "the Doppler-shifted Planck source function"): the dust source of a cell,
// the background and the unit conversion are evaluated at every channel's own frequency, nu_k = nu0 (1 - v_k / c),
// the dust of a cell moving with v_los emitting at nu' = nu_k (1 + v_los / c) in its own frame.  The continuum is then
// one value per channel (CB more registers), the dust temperature is recovered from S_d(nu0) of the coefficient plane,
// and every update costs one more exponential; this kernel, where a thread owns its channels, is the natural home.
#pragma once
#include "transfer_common.cuh"

namespace iris {

template <int CB, bool DUST, bool PERCH = false>
__global__ void __launch_bounds__(128)
transfer_dense_kernel(MarchConsts mc, const float* __restrict__ coef, int64_t ncell, int npix, int nx, int nz, int nv,
                      float* __restrict__ out, float* __restrict__ out_cont) {
  const int tiles_x = (nx + 7) >> 3;
  const int px = (blockIdx.x % tiles_x) * 8 + (threadIdx.x & 7), py = (blockIdx.x / tiles_x) * 4 + (threadIdx.x >> 3);
  const int pix = px < nx ? py * nx + px : npix;
  const int cb = blockIdx.y * blockDim.y + threadIdx.y;
  const int k0 = cb * CB;
  if (pix >= npix || k0 >= nv) return;

  float D[CB];
#pragma unroll
  for (int i = 0; i < CB; ++i) D[i] = 0.0f;
  float C = mc.T_bg;
  float Ck[PERCH ? CB : 1], rk[PERCH ? CB : 1];      // PERCH: continuum and nu_k / nu0 per channel
  if (PERCH) {
#pragma unroll
    for (int i = 0; i < CB; ++i) {
      rk[i] = 1.0f - fmaf((float)(k0 + i), mc.dv_over_c, mc.v0_over_c);
      Ck[i] = planck_krj_at(mc.hnu_k, mc.hnu_k_over_Tcmb, rk[i]);
    }
  }

  const float* p = coef + pix;
  // software prefetch of the next cell's coefficients
  float n_e = p[0], n_a = p[ncell], n_c = p[2 * ncell], n_s = p[3 * ncell];
  float n_td = DUST ? p[4 * ncell] : 0.0f, n_sd = DUST ? p[5 * ncell] : 0.0f;

  for (int z = 0; z < nz; ++z) {
    const float e_c = n_e, a_c = n_a, c_los = n_c, s = n_s, tau_d = n_td, S_d = n_sd;
    if (z + 1 < nz) {
      p += npix;
      n_e = p[0]; n_a = p[ncell]; n_c = p[2 * ncell]; n_s = p[3 * ncell];
      if (DUST) { n_td = p[4 * ncell]; n_sd = p[5 * ncell]; }
    }
    DustStep d;
    if (DUST) {
      d.tau_d = tau_d; d.S_d = S_d; d.C = C;
      d.E_d = exp_neg(tau_d);
      d.m_d = one_minus_exp_neg(tau_d);
      C = fmaf(C, d.E_d, S_d * d.m_d);
    }
    // PERCH: h nu0 / (k T_d) from S_d(nu0) = (h nu0 / k) / expm1(x_d), and 1 + v_los / c of the cell
    const float x_d = (PERCH && S_d > 0.0f) ? log1pf(mc.hnu_k / S_d) : 0.0f;
    const float r_cell = PERCH ? 1.0f + fmaf(c_los - 0.5f, mc.dv_over_c, mc.v0_over_c) : 1.0f;
    const float base = ((float)k0 - c_los) * s;          // x of the block's first edge
    const float top = fmaf((float)CB, s, base);          // x of its last edge
    if (top > -IRIS_ERFC_TMAX && base < IRIS_ERFC_TMAX && a_c != 0.0f) {
      const float sc = DUST ? 0.0f : e_c / a_c - C;
      float x_lo = base;
      float G_lo = signed_erfc(x_lo);
      float sg_lo = copysignf(1.0f, x_lo);
#pragma unroll
      for (int i = 0; i < CB; ++i) {
        const float x_hi = fmaf((float)(i + 1), s, base);
        const float G_hi = signed_erfc(x_hi);
        const float sg_hi = copysignf(1.0f, x_hi);
        const float dErf = (sg_hi - sg_lo) - (G_hi - G_lo);
        if (PERCH) {
          d.S_d = planck_krj_at(mc.hnu_k, x_d, rk[i] * r_cell);
          d.C = Ck[i];
          Ck[i] = fmaf(Ck[i], d.E_d, d.S_d * d.m_d);
        }
        D[i] = DUST ? update_dust(D[i], dErf, e_c, a_c, d) : update_nodust(D[i], dErf, a_c, sc);
        G_lo = G_hi; sg_lo = sg_hi;
      }
    } else if (DUST) {
#pragma unroll
      for (int i = 0; i < CB; ++i) {
        D[i] *= d.E_d;
        if (PERCH) Ck[i] = fmaf(Ck[i], d.E_d, planck_krj_at(mc.hnu_k, x_d, rk[i] * r_cell) * d.m_d);
      }
    }
  }

  float* o = out + (int64_t)pix * nv + k0;
  if (out != nullptr) {
    if ((nv & 3) == 0 && k0 + CB <= nv) {
#pragma unroll
      for (int i = 0; i < CB; i += 4) {
        float4 v;
        if (PERCH) {
          v.x = convert_out_at(D[i], Ck[i], mc, rk[i]); v.y = convert_out_at(D[i + 1], Ck[i + 1], mc, rk[i + 1]);
          v.z = convert_out_at(D[i + 2], Ck[i + 2], mc, rk[i + 2]); v.w = convert_out_at(D[i + 3], Ck[i + 3], mc, rk[i + 3]);
        } else {
          v.x = convert_out(D[i], C, mc); v.y = convert_out(D[i + 1], C, mc);
          v.z = convert_out(D[i + 2], C, mc); v.w = convert_out(D[i + 3], C, mc);
        }
        *reinterpret_cast<float4*>(o + i) = v;
      }
    } else {
#pragma unroll
      for (int i = 0; i < CB; ++i)
        if (k0 + i < nv) o[i] = PERCH ? convert_out_at(D[i], Ck[i], mc, rk[i]) : convert_out(D[i], C, mc);
    }
  }
  if (out_cont != nullptr && cb == 0) out_cont[pix] = C * mc.inv_KRJ;
}

}  // namespace iris
