// K3 with the SMOOTH integrator (trapezoidal first step Eq. 4.8.12, BDF2 Eq. 4.8.10, ReLU of PAPER.md:709) in the
// optically thick mode, as a LINE-WINDOW march: the windowed counterpart of transfer_modes_kernel<0, true, *>.
//
// Same difference form as transfer_modes.cuh (D = I^[T] - I^[C] next to the scalar continuum C):
//   n = 0     D_0 = 0
//   n = 1     D_1 = [(E_0 - A_0 C_0) + (E_1 - A_1 C_1) + (2 - a_0) D_0] / (2 + a_1)
//   n >= 2    D_n = [2 (E_n - A_n C_n) + 4 D_n-1 - D_n-2] / (3 + 2 a_n),     a_n = A_n + tau_d,n
// with E = e_c p, A = a_c p for the profile weight p of the point in the cell, and the ReLU on D + C and on C.
//
// Why a window works.  Where a cell has no line (p = 0) the step is the homogeneous recurrence
//   D_n = (4 D_n-1 - D_n-2) / (3 + 2 tau_d,n),
// the same for every spectral point of a pixel.  Its solutions are spanned by a dominant one, d_n, and a recessive one
// that loses a factor ~3 per cell against it, so a point that no line has come near for K cells is a d_n to 3^-K, with
// its own constant a.  The kernel stores U_n = D_n / d_n: such points are constants and are not touched.  A cell
// updates, explicitly and with the ReLU, the points of its own window and of the windows of the K - 1 cells before it
// (K = 12: 2e-6 of the last change of the point), taking D_n-1 = U d_n-1 and D_n-2 = V d_n-2 from the two stored
// spectra, which alternate roles.
//
// What the window cannot see is a ReLU that fires OUTSIDE it: a far point a d_n + C_n < 0, or the continuum itself
// clamped (C_n < 0 before the ReLU), or the dominant solution losing its sign (4 d_n-1 < d_n-2: a cell that turns
// opaque abruptly).  Each lane keeps the most negative U it has stored and tests these three conditions per cell; if
// one holds for a pixel, the kernel appends the pixel to a list (gate[0] counts its entries) and the caller's next
// launch, transfer_modes_kernel driven by that list, recomputes those pixels densely (exact in every case; the list
// stays empty or short for the paper's workloads).
//
// Fourth condition: "a factor ~3 per cell" holds for tau_d << 1 only.  The roots of the homogeneous step are
// [2 +- sqrt(1 - 2 tau_d)] / (3 + 2 tau_d): the recessive solution loses rho(tau_d) = [2 - sqrt(1 - 2 tau_d)] /
// [2 + sqrt(1 - 2 tau_d)] per cell against the dominant one (1/3 at tau_d = 0, 0.44 at 0.2, 0.63 at 0.4, 1 at 0.5; beyond
// 0.5 the roots are complex and there is no dominant solution at all).  A point released K cells ago is a d_n to the
// PRODUCT of rho over those K cells, so the kernel keeps rho of the last K cells (lane i remembers cell n = i mod K,
// like the windows) and hands over when their product exceeds kSmoothReleaseTol (3^-12 = 1.9e-6 without dust; the
// budget is reached at a sustained tau_d of 0.1 per cell).
//
// (The selectively thin mode is NOT run this way: its absorption saturates at I^[T] = 0, i.e. the ReLU keeps acting on
// points long after the line has left them, and the gate fires on every thick workload; measured: 3.5 + 5.8 ms against
// 5.8 ms for the dense kernel alone on the medium cube.)
//
// Mapping as in transfer_window.cuh: LPP = 16 lanes per pixel, 2 pixels per warp, both spectra of a pixel in shared
// memory, point k at word (k / LPP) * 32 + g * LPP + k % LPP of its array.  Profile: the point value of Eq. 3.3.3 on
// the fine grid (fine_m intervals per channel, Simpson's rule over a channel in the epilogue, Eq. 4.5.1), or the
// channel integral from the channel centre (fine_m = 0; needs dv <= 0.55 b, see transfer_series.cuh).
#pragma once
#include "transfer_common.cuh"
#include "transfer_window.cuh"
#include "transfer_series.cuh"       // packed f32x2 helpers

namespace iris {

constexpr int kSmoothLPP = 16;          // lanes per pixel
constexpr int kSmoothKeep = 12;         // cells a window stays active (K <= kSmoothLPP: lane i remembers cell n = i mod K)
constexpr float kSmoothReleaseTol = 1.0e-5f;   // largest recessive / dominant ratio a released point may carry

// profile weight ("erf-difference" units) of a point at x Doppler widths from the line centre, as a function of
// u = x^2 log2(e): (2 s / sqrt(pi)) 2^-u P(u); P = 1 for the point profile, the degree-4 polynomial of the channel
// integral from the channel centre (transfer_series.cuh) otherwise.  Zero beyond 5.5 Doppler widths (transfer_modes.cuh).
template <bool POINT>
struct SmoothProfile {
  float p0, p1, p2, p3, p4;
  __device__ __forceinline__ void set(float s_amp) {
    const float sp = 1.1283791670955126f * s_amp;               // 2 s / sqrt(pi)
    if (POINT) { p0 = sp; p1 = p2 = p3 = p4 = 0.0f; return; }
    constexpr float L1 = 0.6931471805599453f, L2 = L1 * L1, L3 = L2 * L1, L4 = L2 * L2;   // u = x^2 log2(e)
    const float s2 = s_amp * s_amp, s4 = s2 * s2, s6 = s4 * s2, s8 = s4 * s4;
    p0 = sp * (1.0f - s2 * (1.0f / 12.0f) + s4 * (1.0f / 160.0f) - s6 * (1.0f / 2688.0f) + s8 * (1.0f / 55296.0f));
    p1 = sp * L1 * (s2 * (1.0f / 6.0f) - s4 * (1.0f / 40.0f) + s6 * (1.0f / 448.0f) - s8 * (1.0f / 6912.0f));
    p2 = sp * L2 * (s4 * (1.0f / 120.0f) - s6 * (1.0f / 672.0f) + s8 * (1.0f / 6912.0f));
    p3 = sp * L3 * (s6 * (1.0f / 5040.0f) - s8 * (1.0f / 25920.0f));
    p4 = sp * L4 * (s8 * (1.0f / 362880.0f));
  }
  // xs = x sqrt(log2 e)
  __device__ __forceinline__ float at(float xs) const {
    const float u = xs * xs;
    float pol = p0;
    if (!POINT) {
      pol = fmaf(p4, u, p3);
      pol = fmaf(pol, u, p2);
      pol = fmaf(pol, u, p1);
      pol = fmaf(pol, u, p0);
    }
    const float v = pol * ex2_approx(-u);
    return u > 43.64f ? 0.0f : v;                               // 5.5^2 log2(e)
  }
};

template <bool POINT>
__global__ void __launch_bounds__(128)
transfer_smooth_window_kernel(MarchConsts mc, const float* __restrict__ coef, int64_t ncell, int npix, int nz, int nv,
                              int nvp /* padded points per spectrum */, float* __restrict__ out,
                              float* __restrict__ out_cont, int* __restrict__ gate, int* __restrict__ gate_list) {
  extern __shared__ float sm[];
  constexpr int LPP = kSmoothLPP, PPW = 32 / LPP;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, wpc = blockDim.x >> 5;
  const int g = lane / LPP, i = lane % LPP;
  const unsigned gmask = 0xffffu << (g * LPP);
  const int pix_raw = (blockIdx.x * wpc + warp) * PPW + g;
  const bool valid = pix_raw < npix;
  const int pix = valid ? pix_raw : npix - 1;                   // idle groups shadow the last pixel and write nothing
  const int m = mc.fine_m;
  constexpr bool point = POINT;           // fine grid with the point profile (m > 0) or channel integrals (m = 0)
  const int npts = point ? nv * m + 1 : nv;
  const size_t arr = (size_t)nvp * PPW;
  float* cur = sm + (size_t)warp * 2 * arr + g * LPP;           // U_n-1 = D_n-1 / d_n-1 when cell n is entered
  float* prv = cur + arr;                                       // V = D_n-2 / d_n-2; receives U_n
#define IDX(k) (((k) / LPP) * 32 + ((k) % LPP))
  for (int k = i; k < nvp; k += LPP) { cur[IDX(k)] = 0.0f; prv[IDX(k)] = 0.0f; }
  __syncwarp();

  // position of a point in the units line_window works in (point k is the "channel" [k, k + 1) of width 1 / m whose
  // centre it is), and its spacing in Doppler widths
  const float fm = point ? (float)m : 1.0f, inv_fm = 1.0f / fm;

  float C = mc.T_bg, Cm = mc.T_bg;          // continuum at n - 1 and n - 2 (after the ReLU)
  float d_c = 1.0f, d_m = 1.0f;             // dominant homogeneous solution at n - 1 and n - 2
  float u_min = 0.0f;                       // most negative U this lane has stored
  unsigned ring = 0u;                       // window of the cell this lane remembers (cell n with n % K == i)
  float rho_ring = i < kSmoothKeep ? (1.0f / 3.0f) : 1.0f;   // rho of that cell (lanes K .. LPP - 1 remember nothing)
  int slot = 0;                             // n % K
  bool risk = false;
  // cell 0, for the trapezoidal step
  float e_0 = 0.0f, a_0 = 0.0f, c_0 = 0.0f, s_0 = 1.0f, td_0 = 0.0f, Jd_0 = 0.0f;

  const float* p = coef + pix;
  float n_e = p[0], n_a = p[ncell], n_c = p[2 * ncell], n_s = p[3 * ncell], n_td = p[4 * ncell], n_sd = p[5 * ncell];
  for (int n = 0; n < nz; ++n) {
    const float e_c = n_e, a_c = n_a, s_ch = n_s, td = n_td, Sd = n_sd;
    const float c_los = point ? fmaf(n_c, fm, 0.5f) : n_c;      // in point units
    const float s = s_ch * inv_fm;                              // Doppler widths per point
    if (n + 1 < nz) {
      p += npix;
      n_e = p[0]; n_a = p[ncell]; n_c = p[2 * ncell]; n_s = p[3 * ncell]; n_td = p[4 * ncell]; n_sd = p[5 * ncell];
    }
    const float Jd = td * Sd;
    // ---- window of this cell, remembered for LPP cells; the points to update are the union of what is remembered
    int klo, khi;
    const int W = line_window(e_c, a_c, c_los, s, npts, klo, khi);
    // (remembered as one word, hi in the upper and 0xffff - lo in the lower half: the union of the LPP windows is a
    // halfword maximum, __vmaxu2, per exchange; an empty window is 0)
    if (i == slot) {
      ring = W > 0 ? (((unsigned)khi << 16) | (0xffffu - (unsigned)klo)) : 0u;
      const float sq = sqrtf(fmaxf(fmaf(-2.0f, td, 1.0f), 0.0f));
      rho_ring = __fdividef(2.0f - sq, 2.0f + sq);
    }
    slot = slot + 1 == kSmoothKeep ? 0 : slot + 1;
    unsigned un = ring;
    float rho_prod = rho_ring;
#pragma unroll
    for (int o = LPP / 2; o > 0; o >>= 1) {
      un = __vmaxu2(un, __shfl_xor_sync(gmask, un, o));
      rho_prod *= __shfl_xor_sync(gmask, rho_prod, o);
    }
    if (rho_prod > kSmoothReleaseTol) risk = true;              // released points would not be a d_n any more
    // no window at all: lo = 0xffff, hi = 0 (ehi < elo)
    const int elo = 0xffff - (int)(un & 0xffffu), ehi = (int)(un >> 16);
    if (n == 0) {                                               // D_0 = 0, C_0 = T_bg: nothing moves yet
      e_0 = e_c; a_0 = a_c; c_0 = c_los; s_0 = s; td_0 = td; Jd_0 = Jd;
      continue;
    }
    // ---- continuum and dominant solution of this cell
    float C_unc, d_n;
    if (n == 1) {
      const float r = rcp_approx(2.0f + td);
      C_unc = (Jd_0 + Jd + (2.0f - td_0) * C) * r;
      d_n = 1.0f;                                               // any positive start: every point is still 0
    } else {
      const float r = rcp_approx(fmaf(2.0f, td, 3.0f));
      C_unc = (2.0f * Jd + 4.0f * C - Cm) * r;
      d_n = fmaf(4.0f, d_c, -d_m) * r;
    }
    const float Cn = fmaxf(C_unc, 0.0f);
    const float relu_add = C_unc >= 0.0f ? 0.0f : C_unc, relu_min = C_unc >= 0.0f ? -C_unc : 0.0f;
    // a ReLU outside the window (see the header): recompute densely
    if (C_unc < 0.0f || !(d_n > 1.0e-6f * d_c) || fmaf(u_min, d_n, C_unc) < 0.0f) risk = true;
    const float inv_dn = rcp_approx(d_n);

    if (ehi >= elo) {
      constexpr float SQL2E = 1.2011224087864498f;              // sqrt(log2 e)
      SmoothProfile<POINT> prof;
      prof.set(s_ch);
      const float xstep = (float)LPP * s * SQL2E;
      float xs = ((float)(elo + i) + 0.5f - c_los) * (s * SQL2E);
      if (n == 1) {
        // trapezoidal step over the windows of cells 0 and 1 (D_0 = 0)
        SmoothProfile<POINT> prof0;
        prof0.set(s_0 * fm);
        for (int k = elo + i; k <= ehi; k += LPP, xs += xstep) {
          const float pw = prof.at(xs);
          const float pw0 = prof0.at(((float)k + 0.5f - c_0) * (s_0 * SQL2E));
          const float E = e_c * pw, A = a_c * pw, E0 = e_0 * pw0, A0 = a_0 * pw0;
          const float Du = ((E0 - A0 * C) + (E - A * C_unc)) * rcp_approx(2.0f + A + td);
          const float U = fmaxf(Du + relu_add, relu_min) * inv_dn;              // ReLU on D + C and on C
          IRIS_CHECK_SMEM(prv + IDX(k), 4, sm + (size_t)warp * 2 * arr, sm + (size_t)(warp + 1) * 2 * arr);
          prv[IDX(k)] = U;
          u_min = fminf(u_min, U);
        }
      } else {
        // BDF2: D_n = [2 p (e_c - a_c C_n) + 4 U d_n-1 - V d_n-2] / (3 + 2 tau_d + 2 a_c p), on even-aligned PAIRS of
        // points with packed arithmetic (fma / mul / add.rn.f32x2): a lane takes points k, k + 1, the LPP lanes of a
        // pixel 2 LPP consecutive points (two rows of its spectra) per pass.  A pair may reach one point beyond the
        // window on either side; the step is as valid there.
        const f32x2 g2 = pk1(2.0f * fmaf(-a_c, C_unc, e_c)), a2 = pk1(2.0f * a_c), den0 = pk1(fmaf(2.0f, td, 3.0f));
        const f32x2 c4 = pk1(4.0f * d_c), cm = pk1(-d_m), radd = pk1(relu_add), idn = pk1(inv_dn), pp0 = pk1(prof.p0);
        const f32x2 pp1 = pk1(prof.p1), pp2 = pk1(prof.p2), pp3 = pk1(prof.p3), pp4 = pk1(prof.p4);
        const int k0 = (elo & ~1) + 2 * i;
        const float xa = ((float)k0 + 0.5f - c_los) * (s * SQL2E), xb = s * SQL2E;
        f32x2 xx = pk(xa, xa + xb);
        const f32x2 xstep2 = pk1(2.0f * (float)LPP * xb);
        for (int k = k0; k <= ehi; k += 2 * LPP, xx = add2(xx, xstep2)) {
          const int w = IDX(k);
          IRIS_CHECK_SMEM(cur + w, 8, sm + (size_t)warp * 2 * arr, sm + (size_t)(warp + 1) * 2 * arr);
          IRIS_CHECK_SMEM(prv + w, 8, sm + (size_t)warp * 2 * arr, sm + (size_t)(warp + 1) * 2 * arr);
          const f32x2 u = mul2(xx, xx);
          float u0, u1;
          upk(u, u0, u1);
          f32x2 pw = pk(ex2_approx(-u0), ex2_approx(-u1));
          if (POINT) pw = mul2(pw, pp0);
          else pw = mul2(pw, fma2(fma2(fma2(fma2(pp4, u, pp3), u, pp2), u, pp1), u, pp0));
          const float2 Uo = *reinterpret_cast<const float2*>(cur + w), Vo = *reinterpret_cast<const float2*>(prv + w);
          const f32x2 lin = fma2(pk(Uo.x, Uo.y), c4, mul2(pk(Vo.x, Vo.y), cm));
          const f32x2 den = fma2(pw, a2, den0);
          float e0, e1;
          upk(den, e0, e1);
          const f32x2 Du = add2(mul2(fma2(pw, g2, lin), pk(rcp_approx(e0), rcp_approx(e1))), radd);
          float D0, D1;
          upk(Du, D0, D1);
          const f32x2 U = mul2(pk(fmaxf(D0, relu_min), fmaxf(D1, relu_min)), idn);      // ReLU on D + C and on C
          float2 Un;
          upk(U, Un.x, Un.y);
          if (k + 1 >= npts) Un.y = 0.0f;                                               // padding, not a point
          *reinterpret_cast<float2*>(prv + w) = Un;
          u_min = fminf(u_min, fminf(Un.x, Un.y));
        }
      }
    }
    __syncwarp();
    // ---- roles: what was written is now "n - 1"
    { float* t = cur; cur = prv; prv = t; }
    Cm = C; C = Cn;
    d_m = d_c; d_c = d_n;
    if (n == 1) d_m = 1.0f;
    // keep the dominant solution inside the fp32 range (dust attenuates it like exp(-tau_d)); rare
    if (d_c < 1.0e-12f) {
      const float f = d_c;
      for (int k = i; k < nvp; k += LPP) { cur[IDX(k)] *= f; prv[IDX(k)] *= f; }
      u_min *= f;
      d_m /= f; d_c = 1.0f;
      __syncwarp(gmask);                    // the condition is the same for the LPP lanes of a pixel
    }
  }
  __syncwarp();
  // hand the pixel over: gate[0] = pixels listed by this launch, gate[1] = pixels handed over since the public call began
  const bool group_risk = (__ballot_sync(0xffffffffu, risk && valid) & gmask) != 0u;
  if (group_risk && i == 0) { gate_list[atomicAdd(gate, 1)] = pix; atomicAdd(gate + 1, 1); }

  if (valid) {
    // the points are D = U d; nz = 1 leaves D = 0
    const float dfin = nz > 1 ? d_c : 0.0f;
    if (out != nullptr) {
      if (point) {
        const float wgt = dfin / (3.0f * (float)m);
        for (int c = i; c < nv; c += LPP) {
          float acc = 0.0f;
          for (int j = 0; j < m; j += 2) acc += cur[IDX(c * m + j)] + 4.0f * cur[IDX(c * m + j + 1)] + cur[IDX(c * m + j + 2)];
          out[(int64_t)pix * nv + c] = convert_out(acc * wgt, C, mc);
        }
      } else {
        for (int c = i; c < nv; c += LPP) out[(int64_t)pix * nv + c] = convert_out(cur[IDX(c)] * dfin, C, mc);
      }
    }
    if (out_cont != nullptr && i == 0) out_cont[pix] = C * mc.inv_KRJ;
  }
#undef IDX
}

// Shared memory the kernel needs for one warp (two spectra of two pixels).
inline size_t smooth_window_smem_per_warp(int nv, int fine_m) {
  const int npts = fine_m > 0 ? nv * fine_m + 1 : nv;
  const int nvp = (npts + kSmoothLPP - 1) / kSmoothLPP * kSmoothLPP;
  return (size_t)2 * (32 / kSmoothLPP) * nvp * sizeof(float);
}

inline cudaError_t launch_transfer_smooth_window(const MarchConsts& mc, const float* coef, int64_t ncell, int npix, int nz,
                                                 int nv, float* out, float* out_cont, int* gate, int* gate_list,
                                                 cudaStream_t st) {
  const int npts = mc.fine_m > 0 ? nv * mc.fine_m + 1 : nv;
  const int nvp = (npts + kSmoothLPP - 1) / kSmoothLPP * kSmoothLPP;
  const size_t per_warp = smooth_window_smem_per_warp(nv, mc.fine_m);
  int wpc = 1, best = 0;
  for (int w = 4; w >= 1; w >>= 1) {
    const size_t per_cta = w * per_warp + 1024;
    const int resident = per_cta <= 227 * 1024 ? (int)((227 * 1024) / per_cta) * w : 0;
    if (resident > best) { best = resident; wpc = w; }
  }
  if (best == 0) return cudaErrorInvalidConfiguration;
  const size_t smem = wpc * per_warp;
  const int ppc = wpc * (32 / kSmoothLPP);
  const unsigned grid = (unsigned)((npix + ppc - 1) / ppc);
  cudaError_t e;
  if (mc.fine_m > 0) {
    e = cudaFuncSetAttribute(transfer_smooth_window_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    transfer_smooth_window_kernel<true><<<grid, wpc * 32, smem, st>>>(mc, coef, ncell, npix, nz, nv, nvp, out, out_cont, gate, gate_list);
  } else {
    e = cudaFuncSetAttribute(transfer_smooth_window_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    transfer_smooth_window_kernel<false><<<grid, wpc * 32, smem, st>>>(mc, coef, ncell, npix, nz, nv, nvp, out, out_cont, gate, gate_list);
  }
  return cudaGetLastError();
}

}  // namespace iris
