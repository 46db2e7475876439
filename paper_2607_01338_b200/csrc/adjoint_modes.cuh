// K8 outside the hot-path mode: gradient of L = sum what * cube_raw with respect to the per-cell coefficients in the
// optically thick mode with the SMOOTH integrator (trapezoidal first step Eq. 4.8.12, BDF2 Eq. 4.8.10, ReLU of
// PAPER.md:709) and / or the FINE velocity grid with Simpson's rule over a channel (Eq. 4.5.1) -- the paper's production
// mode is thick + smooth + f = 1 and its pipeline is differentiable end to end.
//
// Reverse mode through the march of one spectral point, in the total-intensity form (Rayleigh-Jeans Kelvin; E = e_c p,
// A = a_c p for the profile weight p of the point in the cell, J_d = tau_d S_d):
//   smooth  y_0 = T_bg
//           y_1 = relu(N_1 / D_1),  N_1 = (E_0 + J_d0) + (E_1 + J_d1) + (2 - A_0 - tau_d0) y_0,  D_1 = 2 + A_1 + tau_d1
//           y_n = relu(N_n / D_n),  N_n = 2 (E_n + J_dn) + 4 y_n-1 - y_n-2,                     D_n = 3 + 2 (A_n + tau_dn)
//   reverse u = lambda_n / D_n where y_n > 0 (the ReLU passes nothing otherwise):
//           dL/dE_n = 2 u,  dL/dA_n = -2 u y_n,  dL/dtau_dn = 2 u (S_dn - y_n),  lambda_n-1 += 4 u,  lambda_n-2 -= u
//           (n = 1: dL/dE_0 = dL/dE_1 = u, dL/dA_1 = -u y_1, dL/dA_0 = -u y_0, dL/dtau_d likewise)
//   formal  I_n+1 = I_n e^-tau + (E + J_d) w(tau),  tau = A + tau_d:  lambda_n = lambda_n+1 e^-tau,
//           dL/dE = lambda w,  dL/dtau = lambda (-I_n e^-tau + (E + J_d) w'(tau)),  dL/dtau_d = dL/dtau + lambda S_d w
// and dL/de_c = sum over points of dL/dE p, dL/da_c = sum of dL/dA p.  The cube is scale (channel value - continuum)
// with the channel value the point itself (coarse grid) or the Simpson average of its m + 1 fine points, which fixes
// the seed lambda of every point; the continuum is the same march with p = 0 and seed -sum(scale what).
//
// The reverse sweep needs y_n of every cell: the forward sweep stores them in a scratch the size of the RESIDENT warps
// (cells x 256 floats per warp), not of the cube.  One warp owns one pixel and walks its points in blocks of 32 NPT
// (point q0 + 32 j + lane; NPT = 8, or 4 / 1 for what is left of the reach): forward sweep (states out), reverse
// sweep (states in, the row of the next cell requested before the arithmetic of the current one; three warp sums per cell
// into the pixel's per-cell accumulators in shared memory).  Measured on 128^3 cells x 256 channels, production mode: 2.2 ms
// without that prefetch, 1.5 ms with it at 16 resident warps per SM -- the state traffic (8.6 GB per gradient) at HBM rate.  The column's six coefficients are staged in shared memory once
// per pixel.  Points no line of the column reaches (outside the union of the cells' line windows) are never marched:
// such a point IS the continuum, so its seed is moved onto the continuum march (with continuum subtraction the two
// cancel and the point drops out altogether).  Inside the reach, a cell whose own line window misses the block of points
// in hand (most cells: a window is ~40 - 80 fine points of a reach of several hundred) takes the step without a line for
// the whole block: no profile, one reciprocal or exponential per cell instead of per point, only the dust accumulator.
//
// The chain to n_H2 (d e_c / dn, d a_c / dn from coef_grad_kernel, tau_d = c_d n) is applied per cell at the end.
#pragma once
#include <type_traits>
#include "adjoint_kernels.cuh"
#include "transfer_modes.cuh"

namespace iris {

constexpr int kAdjModesNPT = 8;            // points per lane in a full block
constexpr int kAdjModesWarps = 4;          // warps per CTA

__host__ __device__ inline size_t adjoint_modes_smem_per_warp(int nz) { return (size_t)11 * nz * sizeof(float); }
__host__ __device__ inline size_t adjoint_modes_scratch_per_warp(int nz) { return (size_t)nz * 32 * kAdjModesNPT * sizeof(float); }

// profile weight ("erf-difference" units, as in transfer_modes.cuh) of point q in a cell
template <bool FINE>
__device__ __forceinline__ float adj_modes_weight(int q, float inv_m, float c_los, float s) {
  if (FINE) {
    const float x = ((float)q * inv_m - c_los) * s;
    return fabsf(x) < kModesXmax ? 1.1283791670955126f * s * ex2_approx(-1.4426950408889634f * x * x) : 0.0f;
  }
  const float xl = ((float)q - c_los) * s, xh = ((float)(q + 1) - c_los) * s;
  if (!(xl < kModesXmax && xh > -kModesXmax)) return 0.0f;
  return erf_diff(xl, signed_erfc(xl), xh, signed_erfc(xh));
}

// seed dL / d(point value in Kelvin) of point q of a pixel: w = what of the pixel [nv]
template <bool FINE>
__device__ __forceinline__ float adj_modes_seed(const float* __restrict__ w, int q, int nv, int m, float scale) {
  if (!FINE) return scale * w[q];
  float s = 0.0f;
  const int v1 = q / m;
#pragma unroll
  for (int v = v1 - 1; v <= v1; ++v) {
    if (v < 0 || v >= nv) continue;
    const int jq = q - v * m;                                  // 0 .. m inside channel v
    if (jq > m) continue;
    const float simpson = (jq == 0 || jq == m) ? 1.0f : ((jq & 1) ? 4.0f : 2.0f);
    s = fmaf(w[v], simpson, s);
  }
  return s * scale / (3.0f * (float)m);
}

// One block of points of one pixel: forward sweep, reverse sweep.  cf: the column's coefficients [6][nz] (shared),
// G: the pixel's accumulators [3][nz] (shared; dL/de_c, dL/da_c, dL/dtau_d), ys: this warp's scratch [nz][32 NPT].
template <bool SMOOTH, bool FINE, int NPT>
__device__ __forceinline__ void adj_modes_block(float T_bg, int nz, int nv, int m, int npts, int q0, const float* cf, float* G,
                                                const int* win, float* __restrict__ ys, const float* __restrict__ w, float scale) {
  const int lane = threadIdx.x & 31;
  const float inv_m = FINE ? 1.0f / (float)m : 1.0f;
  const float *ce = cf, *ca = cf + nz, *cc = cf + 2 * nz, *cs = cf + 3 * nz, *ct = cf + 4 * nz, *cS = cf + 5 * nz;
  constexpr int STR = 32 * kAdjModesNPT;       // scratch row stride (the same for every NPT)
  // does the line window of cell n reach this block of points?  (warp-uniform.)  Where it does not, every point of the
  // block takes the step without a line: no profile, one reciprocal / exponential per cell instead of per point.
  // (checked build) every row of stored states lies inside this warp's slab of the scratch
  const float* ys_end = ys + (size_t)nz * STR;
  (void)ys_end;
  auto hit = [&](int n) {
    const int wv = win[n], klo = wv & 0xffff, khi = (int)((unsigned)wv >> 16);
    return khi >= klo && klo < q0 + 32 * NPT && khi >= q0;
  };
  float y1[NPT], y2[NPT];                      // smooth: y_n-1, y_n-2; formal: y1 = I
  bool live[NPT];
#pragma unroll
  for (int j = 0; j < NPT; ++j) { y1[j] = T_bg; y2[j] = T_bg; live[j] = q0 + 32 * j + lane < npts; }
  // ---- forward
  if (SMOOTH) {
    // cell 0 holds y_0 = T_bg; cell 1 is the trapezoidal step
    if (nz > 1) {
      const float td0 = ct[0], Jd0 = td0 * cS[0], td1 = ct[1], Jd1 = td1 * cS[1];
#pragma unroll
      for (int j = 0; j < NPT; ++j) {
        const int q = q0 + 32 * j + lane;
        const float p0 = adj_modes_weight<FINE>(q, inv_m, cc[0], cs[0]), p1 = adj_modes_weight<FINE>(q, inv_m, cc[1], cs[1]);
        const float N = fmaf(ce[0], p0, Jd0) + fmaf(ce[1], p1, Jd1) + (2.0f - fmaf(ca[0], p0, td0)) * T_bg;
        const float y = fmaxf(N * rcp_approx(2.0f + fmaf(ca[1], p1, td1)), 0.0f);
        y2[j] = T_bg; y1[j] = y;
        ys[STR + 32 * j + lane] = y;
      }
    }
    for (int n = 2; n < nz; ++n) {
      const float e = ce[n], a = ca[n], c = cc[n], s = cs[n], td = ct[n], Jd = td * cS[n];
      const float den0 = fmaf(2.0f, td, 3.0f);
      if (!hit(n)) {
        const float r = rcp_approx(den0), b = 2.0f * Jd;
#pragma unroll
        for (int j = 0; j < NPT; ++j) {
          const float y = fmaxf((fmaf(4.0f, y1[j], -y2[j]) + b) * r, 0.0f);
          y2[j] = y1[j]; y1[j] = y;
          ys[(size_t)n * STR + 32 * j + lane] = y;
        }
        continue;
      }
#pragma unroll
      for (int j = 0; j < NPT; ++j) {
        const int q = q0 + 32 * j + lane;
        const float p = adj_modes_weight<FINE>(q, inv_m, c, s);
        const float N = fmaf(2.0f, fmaf(e, p, Jd), fmaf(4.0f, y1[j], -y2[j]));
        const float y = fmaxf(N * rcp_approx(fmaf(2.0f * a, p, den0)), 0.0f);
        y2[j] = y1[j]; y1[j] = y;
        ys[(size_t)n * STR + 32 * j + lane] = y;
      }
    }
  } else {
    for (int n = 0; n < nz; ++n) {
      const float e = ce[n], a = ca[n], c = cc[n], s = cs[n], td = ct[n], Jd = td * cS[n];
      if (!hit(n)) {
        const float em = exp_neg(td), src = cS[n] * one_minus_exp_neg(td);
#pragma unroll
        for (int j = 0; j < NPT; ++j) {
          ys[(size_t)n * STR + 32 * j + lane] = y1[j];
          y1[j] = fmaf(y1[j], em, src);
        }
        continue;
      }
#pragma unroll
      for (int j = 0; j < NPT; ++j) {
        const int q = q0 + 32 * j + lane;
        ys[(size_t)n * STR + 32 * j + lane] = y1[j];            // the intensity BEFORE cell n
        const float p = adj_modes_weight<FINE>(q, inv_m, c, s);
        const float tau = fmaf(a, p, td), em = exp_neg(tau), mm = one_minus_exp_neg(tau);
        float wt, wp;
        w_and_wprime(tau, mm, em, rcp_approx(fabsf(tau) < 1.0e-30f ? 1.0f : tau), wt, wp);
        y1[j] = fmaf(y1[j], em, fmaf(e, p, Jd) * wt);
      }
    }
  }
  // ---- reverse
  float la[NPT], lb[NPT];                      // lambda_n (complete) and the part of lambda_n-1 known so far
#pragma unroll
  for (int j = 0; j < NPT; ++j) {
    const int q = q0 + 32 * j + lane;
    la[j] = live[j] ? adj_modes_seed<FINE>(w, q, nv, m, scale) : 0.0f;
    lb[j] = 0.0f;
  }
  auto reduce_into = [&](int n, float ge, float ga, float gt) {
    ge = warp_sum(ge); ga = warp_sum(ga); gt = warp_sum(gt);
    if (lane == 0) { G[n] += ge; G[nz + n] += ga; G[2 * nz + n] += gt; }
  };
  // the stored states come back from L2 / HBM: the row of the next cell of the sweep is requested before the arithmetic
  // of the current one (a warp would otherwise sit out the whole latency once per cell)
  float yc[NPT], yn[NPT];
  auto load_row = [&](int n, float (&dst)[NPT]) {
    IRIS_CHECK_SMEM(ys + (size_t)n * STR + lane, 4 * (32 * (NPT - 1) + 1), ys, ys_end);
#pragma unroll
    for (int j = 0; j < NPT; ++j) dst[j] = ys[(size_t)n * STR + 32 * j + lane];
  };
  if (SMOOTH) {
    if (nz > 1) load_row(nz - 1, yc);
    for (int n = nz - 1; n >= 2; --n) {
      load_row(n - 1, yn);
      const float e = ce[n], a = ca[n], c = cc[n], s = cs[n], td = ct[n], Sd = cS[n];
      const float den0 = fmaf(2.0f, td, 3.0f);
      float ge = 0.0f, ga = 0.0f, gt = 0.0f;
      (void)e;
      if (!hit(n)) {
        const float r = rcp_approx(den0);
#pragma unroll
        for (int j = 0; j < NPT; ++j) {
          const float y = yc[j];
          const float u = y > 0.0f ? la[j] * r : 0.0f;
          gt = fmaf(2.0f * u, Sd - y, gt);
          la[j] = fmaf(4.0f, u, lb[j]);
          lb[j] = -u;
        }
        gt = warp_sum(gt);
        if (lane == 0) G[2 * nz + n] += gt;
#pragma unroll
        for (int j = 0; j < NPT; ++j) yc[j] = yn[j];
        continue;
      }
#pragma unroll
      for (int j = 0; j < NPT; ++j) {
        const int q = q0 + 32 * j + lane;
        const float y = yc[j];
        const float p = adj_modes_weight<FINE>(q, inv_m, c, s);
        const float u = y > 0.0f ? la[j] * rcp_approx(fmaf(2.0f * a, p, den0)) : 0.0f;
        const float u2 = 2.0f * u;
        ge = fmaf(u2, p, ge);
        ga = fmaf(-u2 * y, p, ga);
        gt = fmaf(u2, Sd - y, gt);
        la[j] = fmaf(4.0f, u, lb[j]);
        lb[j] = -u;
        yc[j] = yn[j];
      }
      reduce_into(n, ge, ga, gt);
    }
    if (nz > 1) {
      const float td0 = ct[0], td1 = ct[1];
      float ge0 = 0.0f, ga0 = 0.0f, gt0 = 0.0f, ge1 = 0.0f, ga1 = 0.0f, gt1 = 0.0f;
#pragma unroll
      for (int j = 0; j < NPT; ++j) {
        const int q = q0 + 32 * j + lane;
        const float y = yc[j];
        const float p0 = adj_modes_weight<FINE>(q, inv_m, cc[0], cs[0]), p1 = adj_modes_weight<FINE>(q, inv_m, cc[1], cs[1]);
        const float u = y > 0.0f ? la[j] * rcp_approx(2.0f + fmaf(ca[1], p1, td1)) : 0.0f;
        ge0 = fmaf(u, p0, ge0); ga0 = fmaf(-u * T_bg, p0, ga0); gt0 = fmaf(u, cS[0] - T_bg, gt0);
        ge1 = fmaf(u, p1, ge1); ga1 = fmaf(-u * y, p1, ga1);    gt1 = fmaf(u, cS[1] - y, gt1);
      }
      (void)td0;
      reduce_into(0, ge0, ga0, gt0);
      reduce_into(1, ge1, ga1, gt1);
    }
  } else {
    load_row(nz - 1, yc);
    for (int n = nz - 1; n >= 0; --n) {
      if (n > 0) load_row(n - 1, yn);
      const float e = ce[n], a = ca[n], c = cc[n], s = cs[n], td = ct[n], Sd = cS[n], Jd = td * Sd;
      float ge = 0.0f, ga = 0.0f, gt = 0.0f;
      if (!hit(n)) {
        // d/dtau_d of  I e^-tau_d + S_d (1 - e^-tau_d)  is  e^-tau_d (S_d - I)
        const float em = exp_neg(td);
#pragma unroll
        for (int j = 0; j < NPT; ++j) {
          const float I = yc[j];
          gt = fmaf(la[j] * em, Sd - I, gt);
          la[j] *= em;
          yc[j] = yn[j];
        }
        gt = warp_sum(gt);
        if (lane == 0) G[2 * nz + n] += gt;
        continue;
      }
#pragma unroll
      for (int j = 0; j < NPT; ++j) {
        const int q = q0 + 32 * j + lane;
        const float I = yc[j];
        const float p = adj_modes_weight<FINE>(q, inv_m, c, s);
        const float tau = fmaf(a, p, td), em = exp_neg(tau), mm = one_minus_exp_neg(tau);
        float wt, wp;
        w_and_wprime(tau, mm, em, rcp_approx(fabsf(tau) < 1.0e-30f ? 1.0f : tau), wt, wp);
        const float dtau = la[j] * fmaf(-I, em, fmaf(e, p, Jd) * wp);
        const float dE = la[j] * wt;
        ge = fmaf(dE, p, ge);
        ga = fmaf(dtau, p, ga);
        gt += fmaf(dE, Sd, dtau);
        la[j] *= em;
        yc[j] = yn[j];
      }
      reduce_into(n, ge, ga, gt);
    }
  }
}

// One warp per pixel (persistent: warp g of the grid takes pixels g, g + warps, ...).  dc: d e_c / dn and d a_c / dn per
// cell [2][ncell] (or the planes e_c, a_c themselves for the abundance gradient), c_d = d tau_d / dn.
template <bool SMOOTH, bool FINE>
__global__ void __launch_bounds__(32 * kAdjModesWarps)
adjoint_modes_kernel(MarchConsts mc, AdjointConsts ac, const float* __restrict__ coef, const float* __restrict__ dc,
                     int64_t ncell, int npix, int nz, int nv, int m, const float* __restrict__ what,
                     float* __restrict__ scratch, float* __restrict__ grad) {
  extern __shared__ float sm_adjm[];
  constexpr unsigned FULL = 0xffffffffu;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int gwarp = blockIdx.x * kAdjModesWarps + warp, nwarps = gridDim.x * kAdjModesWarps;
  float* cf = sm_adjm + (size_t)warp * 11 * nz;        // [6][nz] coefficients
  float* G = cf + 6 * nz;                              // [3][nz] accumulators
  float* Cs = cf + 9 * nz;                             // [nz] continuum states
  int* win = reinterpret_cast<int*>(cf + 10 * nz);     // [nz] line window of the cell in points: klo | khi << 16 (empty: 1 | 0)
  float* ys = scratch + (size_t)gwarp * nz * 32 * kAdjModesNPT;
  const int npts = FINE ? nv * m + 1 : nv;
  const float fm = FINE ? (float)m : 1.0f;
  for (int pix = gwarp; pix < npix; pix += nwarps) {
    __syncwarp();
    // ---- the column's coefficients, its reach in points, zeroed accumulators
    int qlo = 0x3fffffff, qhi = -1;
    for (int n = lane; n < nz; n += 32) {
      const float* p = coef + (int64_t)n * npix + pix;
      const float e = p[0], a = p[ncell], c = p[2 * ncell], s = p[3 * ncell];
      cf[n] = e; cf[nz + n] = a; cf[2 * nz + n] = c; cf[3 * nz + n] = s;
      cf[4 * nz + n] = p[4 * ncell]; cf[5 * nz + n] = p[5 * ncell];
      G[n] = 0.0f; G[nz + n] = 0.0f; G[2 * nz + n] = 0.0f;
      int klo, khi;
      // (point q of the fine grid is the "channel" [q, q + 1) of width 1 / m whose centre it is, as in transfer_smooth.cuh)
      int wv = 1;
      if (line_window(e, a, FINE ? fmaf(c, fm, 0.5f) : c, s / fm, npts, klo, khi) > 0) {
        qlo = min(qlo, klo); qhi = max(qhi, khi);
        // (one point of margin: the bounds are floors of float positions)
        wv = max(klo - 1, 0) | (min(khi + 1, npts - 1) << 16);
      }
      win[n] = wv;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      qlo = min(qlo, __shfl_xor_sync(FULL, qlo, o));
      qhi = max(qhi, __shfl_xor_sync(FULL, qhi, o));
    }
    // one point of margin on either side: the window bounds are floors of float positions
    qlo = max(qlo - 1, 0); qhi = min(qhi + 1, npts - 1);
    __syncwarp();
    const float* w = what + (int64_t)pix * nv;
    // ---- seeds: all points, and the points that are marched
    float s_all = 0.0f, s_in = 0.0f;
    for (int q = lane; q < npts; q += 32) {
      const float sd = adj_modes_seed<FINE>(w, q, nv, m, ac.scale);
      s_all += sd;
      if (q >= qlo && q <= qhi) s_in += sd;
    }
    s_all = warp_sum(s_all); s_in = warp_sum(s_in);
    // ---- the marched points, block by block (a short last block runs with fewer points per lane)
    for (int q0 = qlo; q0 <= qhi;) {
      const int left = qhi - q0 + 1;
      // (the points of a block beyond qhi but inside the spectrum are marched with their own seeds: count them as "in")
      auto extra_in = [&](int cover) {
        float ex = 0.0f;
        for (int q = qhi + 1 + lane; q < min(q0 + cover, npts); q += 32) ex += adj_modes_seed<FINE>(w, q, nv, m, ac.scale);
        return warp_sum(ex);
      };
      // few, large blocks: a block costs a walk over all cells whatever its width (measured: blocks cut to fit the reach,
      // 8 / 4 / 2 / 1 points per lane, 2.05 ms against 1.51 ms for this rule on 128^3 x 256 channels)
      auto run = [&](auto npt_tag) {
        constexpr int NPT = decltype(npt_tag)::value;
        s_in += extra_in(32 * NPT);
        adj_modes_block<SMOOTH, FINE, NPT>(mc.T_bg, nz, nv, m, npts, q0, cf, G, win, ys, w, ac.scale);
        q0 += 32 * NPT;
      };
      if (left > 32 * 4) run(std::integral_constant<int, 8>{});
      else if (left > 32) run(std::integral_constant<int, 4>{});
      else run(std::integral_constant<int, 1>{});
      __syncwarp();
    }
    // ---- continuum: every point that was not marched is the continuum, and the subtraction takes sum(seeds) of it
    const float lamC = ac.subtract ? -s_in : s_all - s_in;
    if (lane == 0 && lamC != 0.0f) {
      const float *ct = cf + 4 * nz, *cS = cf + 5 * nz;
      if (SMOOTH) {
        if (nz > 1) {
          Cs[0] = mc.T_bg;
          Cs[1] = fmaxf((ct[0] * cS[0] + ct[1] * cS[1] + (2.0f - ct[0]) * mc.T_bg) / (2.0f + ct[1]), 0.0f);
          for (int n = 2; n < nz; ++n)
            Cs[n] = fmaxf((2.0f * ct[n] * cS[n] + 4.0f * Cs[n - 1] - Cs[n - 2]) / fmaf(2.0f, ct[n], 3.0f), 0.0f);
          float la = lamC, lb = 0.0f;
          for (int n = nz - 1; n >= 2; --n) {
            const float y = Cs[n];
            const float u = y > 0.0f ? la / fmaf(2.0f, ct[n], 3.0f) : 0.0f;
            G[2 * nz + n] += 2.0f * u * (cS[n] - y);
            la = fmaf(4.0f, u, lb);
            lb = -u;
          }
          const float u = Cs[1] > 0.0f ? la / (2.0f + ct[1]) : 0.0f;
          G[2 * nz] += u * (cS[0] - mc.T_bg);
          G[2 * nz + 1] += u * (cS[1] - Cs[1]);
        }
      } else {
        float I = mc.T_bg;
        for (int n = 0; n < nz; ++n) {
          Cs[n] = I;
          const float td = ct[n];
          I = fmaf(I, expf(-td), cS[n] * -expm1f(-td));
        }
        float la = lamC;
        for (int n = nz - 1; n >= 0; --n) {
          const float td = ct[n], em = expf(-td);
          // d/dtau_d of  I e^-tau + S_d (1 - e^-tau)
          G[2 * nz + n] += la * em * (cS[n] - Cs[n]);
          la *= em;
        }
      }
    }
    __syncwarp();
    // ---- chain to the density (or the abundance) and store
    for (int n = lane; n < nz; n += 32) {
      const int64_t cell = (int64_t)n * npix + pix;
      grad[cell] = fmaf(G[n], dc[cell], fmaf(G[nz + n], dc[ncell + cell], G[2 * nz + n] * ac.c_d));
    }
  }
}

// Launch: persistent grid of resident warps; scratch must hold adjoint_modes_scratch_per_warp(nz) * warps bytes.
inline int adjoint_modes_grid(int sm_count, int nz) {
  const size_t smem = kAdjModesWarps * adjoint_modes_smem_per_warp(nz);
  int ctas = (int)((200u * 1024u) / (smem + 1024));
  ctas = ctas < 1 ? 1 : (ctas > 4 ? 4 : ctas);
  return sm_count * ctas;
}

inline cudaError_t launch_adjoint_modes(const MarchConsts& mc, const AdjointConsts& ac, bool smooth, int fine_m,
                                        const float* coef, const float* dc, int64_t ncell, int npix, int nz, int nv,
                                        const float* what, float* scratch, float* grad, int grid, cudaStream_t st) {
  const size_t smem = kAdjModesWarps * adjoint_modes_smem_per_warp(nz);
  if (smem > 227u * 1024u) return cudaErrorInvalidConfiguration;
  cudaError_t e;
#define IRIS_LAUNCH_ADJM(S_, F_)                                                                                          \
  do {                                                                                                                    \
    e = cudaFuncSetAttribute(adjoint_modes_kernel<S_, F_>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);       \
    if (e != cudaSuccess) return e;                                                                                       \
    adjoint_modes_kernel<S_, F_><<<grid, 32 * kAdjModesWarps, smem, st>>>(mc, ac, coef, dc, ncell, npix, nz, nv, fine_m,  \
                                                                          what, scratch, grad);                           \
  } while (0)
  if (smooth) { if (fine_m > 0) IRIS_LAUNCH_ADJM(true, true); else IRIS_LAUNCH_ADJM(true, false); }
  else { if (fine_m > 0) IRIS_LAUNCH_ADJM(false, true); else IRIS_LAUNCH_ADJM(false, false); }
#undef IRIS_LAUNCH_ADJM
  return cudaGetLastError();
}

}  // namespace iris
