// K8 / K9: gradient of L = sum_{y,x,v} what * cube_raw with respect to n_H2 of every cell
// (what = beam-adjoint of the caller's weights; cube_raw = the noise-free cube before the beam).
//
// The paper obtains this gradient from PyTorch autograd through the whole observation.
// Here it is written out: the adjoint of the formal step (Eq. 4.8.5-4.8.7)
//   T' = T E_T + (J + S_d tau_d) w(tau_T),   tau_T = tau_L + tau_d,  E_T = exp(-tau_T),  w = (1 - E_T) / tau_T
// is  lambda_k = lambda_{k+1} E_T  with
//   dT'/dJ = w,   dT'/dtau_T = -T E_T + (J + S_d tau_d) w'(tau_T),   explicit dT'/dtau_d += S_d w.
// Instead of a reverse scan (which needs every intermediate intensity, or an unstable division by E_T),
// the adjoint variable is evaluated in closed form during a second FORWARD march:
//   lambda_{k+1}[v] = scale * what[v] * exp(-(totL[v] - cumL_k[v])) * exp(-(totD - cumD_k)),
// where totL[v] is the line optical depth of the whole ray in channel v (first march) and cumL_k its running
// sum: only sums of optical depths, stable for any tau.  One warp owns one pixel; its per-channel state
// (remaining line depth, attenuated weights, the scaled difference spectrum Dt of transfer_window.cuh) lives
// in shared memory; only the channels inside a cell's line window are touched, plus -- with dust -- one
// dense dot product per cell for the dust-attenuation term of the channels outside the window.
//
// Chain rule to n_H2 (K9): e_c = c_e n x_u, a_c = c_a n (x_l g_u/g_l - x_u), tau_d = c_d n, and
// y = n dx/dn solves  y Q = -x Q_C  (Q the generator of the level balance, Q_C its collisional part) with
// sum(y) = 0; it is obtained from the elimination factors the GTH solve of K1 leaves in registers.
#pragma once
#include "cell_kernels.cuh"
#include "transfer_common.cuh"
#include "transfer_window.cuh"
#include "transfer_series.cuh"      // packed f32x2 helpers

namespace iris {

struct AdjointConsts {
  float c_e, c_a, c_d, gr;
  int upper, lower;
  float T_inf;
  float scale;      // d(cube_raw) / d(D in Kelvin): 1 for T_RJ output, 1 / K_RJ for intensity output
  int subtract;     // 1: cube_raw = total - continuum
};

// Level fractions x and their logarithmic density derivative y = n dx/dn.  BW: bandwidth of the rate matrix
// (see level_fractions in cell_kernels.cuh).
template <int N, int BW, bool TABLE>
__device__ __forceinline__ void level_fractions_grad(const LevelConsts& lc, float n, float T, float (&x)[N],
                                                     float (&y)[N]) {
  const CollTable& tb = lc.tb;
  float R[N][N];
  float kf = n, wt = 0.0f;
  int t0 = 0;
  if (TABLE) locate_temperature(tb, T, t0, wt);
  else kf = n * pow_approx(T * lc.inv_Tref, lc.Texp);
  float q[N];
  boltzmann_adjacent<N>(lc, T, q);
  // collisional de-excitation rates of the band (per unit kf), and the same times g_u / g_l
  auto coll = [&](int u, int l, float& Kd, float& Kg) {
    const float4 pr = lc.pr[pair_index(u, l)];
    Kd = pr.x; Kg = pr.z;
    if (TABLE) {
      const float2 k0 = tb.K[t0 * kMaxPairs + pair_index(u, l)];
      const float2 k1 = tb.K[min(t0 + 1, tb.nT - 1) * kMaxPairs + pair_index(u, l)];
      Kd = fmaf(wt, k1.x - k0.x, k0.x);
      Kg = fmaf(wt, k1.y - k0.y, k0.y);
    }
  };
#pragma unroll
  for (int u = 1; u < N; ++u) {
    float bz = 1.0f;
#pragma unroll
    for (int l = u - 1; l >= 0; --l) {
      if (u - l > BW) continue;
      bz *= q[l + 1];
      const float4 pr = lc.pr[pair_index(u, l)];
      float Kd, Kg;
      coll(u, l, Kd, Kg);
      R[u][l] = fmaf(kf, Kd, pr.y);
      R[l][u] = fmaf(kf * bz, Kg, pr.w);
    }
  }
  float inv[N];
#pragma unroll
  for (int m = N - 1; m >= 1; --m) {
    const int lo = m - BW > 0 ? m - BW : 0;
    float s = 0.0f;
#pragma unroll
    for (int j = 0; j < m; ++j)
      if (j >= lo) s += R[m][j];
    inv[m] = rcp_approx(s);
#pragma unroll
    for (int i = 0; i < m; ++i)
      if (i >= lo) R[i][m] *= inv[m];
#pragma unroll
    for (int i = 0; i < m; ++i)
#pragma unroll
      for (int j = 0; j < m; ++j)
        if (i != j && i >= lo && j >= lo) R[i][j] = fmaf(R[i][m], R[m][j], R[i][j]);
  }
  x[0] = 1.0f;
  float tot = 1.0f;
#pragma unroll
  for (int j = 1; j < N; ++j) {
    float s = 0.0f;
#pragma unroll
    for (int i = 0; i < j; ++i)
      if (j - i <= BW) s = fmaf(x[i], R[i][j], s);
    x[j] = s;
    tot += s;
  }
  const float itot = rcp_approx(tot);
#pragma unroll
  for (int j = 0; j < N; ++j) x[j] *= itot;
  // right-hand side b = -x Q_C: net collisional outflow of every level (pairwise, so that sum(b) = 0)
  float b[N];
#pragma unroll
  for (int j = 0; j < N; ++j) b[j] = 0.0f;
#pragma unroll
  for (int u = 1; u < N; ++u) {
    float bz = 1.0f;
#pragma unroll
    for (int l = u - 1; l >= 0; --l) {
      if (u - l > BW) continue;
      bz *= q[l + 1];
      float Kd, Kg;
      coll(u, l, Kd, Kg);
      const float f = x[u] * (kf * Kd) - x[l] * (kf * bz * Kg);   // net flow u -> l
      b[u] += f;
      b[l] -= f;
    }
  }
  // the same eliminations applied to b, then back-substitution with y_0 = 0
#pragma unroll
  for (int m = N - 1; m >= 1; --m) {
    const float t = b[m] * inv[m];
#pragma unroll
    for (int j = 0; j < m; ++j)
      if (m - j <= BW) b[j] = fmaf(t, R[m][j], b[j]);
  }
  y[0] = 0.0f;
  float sy = 0.0f;
#pragma unroll
  for (int m = 1; m < N; ++m) {
    float s = -b[m] * inv[m];
#pragma unroll
    for (int i = 0; i < m; ++i)
      if (m - i <= BW) s = fmaf(y[i], R[i][m], s);
    y[m] = s;
    sy += s;
  }
#pragma unroll
  for (int j = 0; j < N; ++j) y[j] = fmaf(-sy, x[j], y[j]);     // project onto sum(y) = 0
}

// K9 (per cell): d e_c / d n and d a_c / d n  ->  dcoef[2][ncell]
template <int N, int BW, bool TABLE>
__global__ void __launch_bounds__(128) coef_grad_kernel(LevelConsts lc, AdjointConsts ac, int64_t ncell,
                                                        const float* __restrict__ nH2, const float* __restrict__ Tgas,
                                                        float* __restrict__ dcoef) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= ncell) return;
  const float n = nH2[i], T = Tgas[i];
  float x[N], y[N];
  level_fractions_grad<N, BW, TABLE>(lc, n, T, x, y);
  float xu = 0.0f, xl = 0.0f;
#pragma unroll
  for (int l = 0; l < N; ++l) {
    if (l == ac.upper) xu = x[l] + y[l];
    if (l == ac.lower) xl = x[l] + y[l];
  }
  float de = ac.c_e * xu, da = ac.c_a * fmaf(xl, ac.gr, -xu);
  if (T > ac.T_inf) { de = 0.0f; da = 0.0f; }
  dcoef[i] = de;
  dcoef[ncell + i] = da;
}

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// Sums of eight per-lane values over the warp in 17 shuffles instead of 40: three exchange steps halve the number of
// values a lane carries (lanes with the bit set keep the upper half), two more finish the one value that is left, and
// the eight totals (index j at lane 4 j) are broadcast back.
__device__ __forceinline__ void warp_sum8(float (&v)[8]) {
  const unsigned FULL = 0xffffffffu;
  const int lane = threadIdx.x & 31;
  const bool b4 = lane & 16, b3 = lane & 8, b2 = lane & 4;
  float a[4], b[2], r;
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    const float send = b4 ? v[j] : v[j + 4];
    a[j] = (b4 ? v[j + 4] : v[j]) + __shfl_xor_sync(FULL, send, 16);
  }
#pragma unroll
  for (int j = 0; j < 2; ++j) {
    const float send = b3 ? a[j] : a[j + 2];
    b[j] = (b3 ? a[j + 2] : a[j]) + __shfl_xor_sync(FULL, send, 8);
  }
  {
    const float send = b2 ? b[0] : b[1];
    r = (b2 ? b[1] : b[0]) + __shfl_xor_sync(FULL, send, 4);
  }
  r += __shfl_xor_sync(FULL, r, 2);
  r += __shfl_xor_sync(FULL, r, 1);
#pragma unroll
  for (int j = 0; j < 8; ++j) v[j] = __shfl_sync(FULL, r, 4 * j);
}

// Channel integral of the Gaussian profile from the channel CENTRE (dv / b <= 0.55; same expansion as
// transfer_series.cuh): erf(x + s/2) - erf(x - s/2) = (2 s / sqrt(pi)) exp(-x^2) P(x^2), P of degree 4 with
// coefficients that depend on the cell only.
struct CentreProfile {
  float p0, p1, p2, p3, p4;     // already multiplied by 2 s / sqrt(pi)
  __device__ __forceinline__ void set(float s) {
    const float sp = 1.1283791670955126f * s;
    const float s2 = s * s, s4 = s2 * s2, s6 = s4 * s2, s8 = s4 * s4;
    p0 = sp * (1.0f - s2 * (1.0f / 12.0f) + s4 * (1.0f / 160.0f) - s6 * (1.0f / 2688.0f) + s8 * (1.0f / 55296.0f));
    p1 = sp * (s2 * (1.0f / 6.0f) - s4 * (1.0f / 40.0f) + s6 * (1.0f / 448.0f) - s8 * (1.0f / 6912.0f));
    p2 = sp * (s4 * (1.0f / 120.0f) - s6 * (1.0f / 672.0f) + s8 * (1.0f / 6912.0f));
    p3 = sp * (s6 * (1.0f / 5040.0f) - s8 * (1.0f / 25920.0f));
    p4 = sp * (s8 * (1.0f / 362880.0f));
  }
  __device__ __forceinline__ float at(float x) const {
    const float u = x * x;
    float pol = fmaf(p4, u, p3);
    pol = fmaf(pol, u, p2);
    pol = fmaf(pol, u, p1);
    pol = fmaf(pol, u, p0);
    return pol * ex2_approx(-1.4426950408889634f * u);
  }
};

// ---- packed pairs (two adjacent channels per lane; f32x2 helpers of transfer_series.cuh)
// CentreProfile::at for the pair of channels at x and x + s
__device__ __forceinline__ f32x2 centre_profile_pair(const CentreProfile& p, float x, float s) {
  const f32x2 xx = pk(x, x + s);
  const f32x2 u = mul2(xx, xx);
  f32x2 pol = fma2(pk1(p.p4), u, pk1(p.p3));
  pol = fma2(pol, u, pk1(p.p2));
  pol = fma2(pol, u, pk1(p.p1));
  pol = fma2(pol, u, pk1(p.p0));
  float u0, u1;
  upk(u, u0, u1);
  return mul2(pol, pk(ex2_approx(-1.4426950408889634f * u0), ex2_approx(-1.4426950408889634f * u1)));
}

// w(tau) = (1 - exp(-tau)) / tau and w'(tau) = (exp(-tau)(1 + tau) - 1) / tau^2 from m = 1 - exp(-tau) and it = 1 / tau,
// accurate for every tau: the closed form of w' loses a factor 2 / tau of relative accuracy to cancellation, and the
// abundance gradient of a saturated line is itself a difference of an emission and an absorption term, so the series
// take over below |tau| = 0.25 (both forms are evaluated and selected: no divergent branch).
__device__ __forceinline__ void w_and_wprime(float tau, float m, float em /* exp(-tau) */, float it, float& w, float& wp) {
  float p = fmaf(tau, -1.0f / 5040.0f, 1.0f / 720.0f);
  p = fmaf(p, tau, -1.0f / 120.0f);
  p = fmaf(p, tau, 1.0f / 24.0f);
  p = fmaf(p, tau, -1.0f / 6.0f);
  p = fmaf(p, tau, 0.5f);
  const float ws = fmaf(-p, tau, 1.0f);                       // 1 - tau/2 + tau^2/6 - ...
  float r = fmaf(tau, -1.0f / 5760.0f, 1.0f / 840.0f);
  r = fmaf(r, tau, -1.0f / 144.0f);
  r = fmaf(r, tau, 1.0f / 30.0f);
  r = fmaf(r, tau, -0.125f);
  r = fmaf(r, tau, 1.0f / 3.0f);
  const float wps = fmaf(r, tau, -0.5f);                      // -1/2 + tau/3 - tau^2/8 + ...
  const float wb = m * it;
  const float wpb = fmaf(em, 1.0f + tau, -1.0f) * it * it;
  const bool small = fabsf(tau) < 0.25f;
  w = small ? ws : wb;
  wp = small ? wps : wpb;
}

// Channel erf difference of channel c in a cell (both edges evaluated by the calling lane).
__device__ __forceinline__ float channel_derf(int c, float c_los, float s) {
  const float x_lo = ((float)c - c_los) * s, x_hi = ((float)(c + 1) - c_los) * s;
  const float G_lo = signed_erfc(x_lo), G_hi = signed_erfc(x_hi);
  return (copysignf(1.0f, G_hi) - copysignf(1.0f, G_lo)) - (G_hi - G_lo);
}

// Sums over the LPP lanes of a pixel (aligned lane groups of a warp).
template <int LPP>
__device__ __forceinline__ float seg_sum(float v, unsigned gmask) {
#pragma unroll
  for (int o = LPP / 2; o > 0; o >>= 1) v += __shfl_xor_sync(gmask, v, o);
  return v;
}

// Eight sums over the LPP lanes of a pixel at once: three exchange steps halve the number of values a lane carries
// (lanes with the bit set keep the upper half), the remaining steps finish the one value that is left, and the eight
// totals (index j at lane (LPP / 8) j of the group) are broadcast back: 7 + log2(LPP / 8) + 8 shuffles instead of
// 8 log2(LPP).
template <int LPP>
__device__ __forceinline__ void seg_sum8(float (&v)[8], unsigned gmask, int gbase) {
  constexpr int H = LPP / 2;
  const int lane = threadIdx.x & 31;
  const bool b1 = lane & H, b2 = lane & (H / 2), b3 = lane & (H / 4);
  float a[4], b[2], r;
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    const float send = b1 ? v[j] : v[j + 4];
    a[j] = (b1 ? v[j + 4] : v[j]) + __shfl_xor_sync(gmask, send, H);
  }
#pragma unroll
  for (int j = 0; j < 2; ++j) {
    const float send = b2 ? a[j] : a[j + 2];
    b[j] = (b2 ? a[j + 2] : a[j]) + __shfl_xor_sync(gmask, send, H / 2);
  }
  {
    const float send = b3 ? b[0] : b[1];
    r = (b3 ? b[1] : b[0]) + __shfl_xor_sync(gmask, send, H / 4);
  }
#pragma unroll
  for (int o = H / 8; o > 0; o >>= 1) r += __shfl_xor_sync(gmask, r, o);
#pragma unroll
  for (int j = 0; j < 8; ++j) v[j] = __shfl_sync(gmask, r, gbase + (H / 4) * j);
}

__device__ __forceinline__ f32x2 sel2(bool c0, bool c1, f32x2 a, f32x2 b) {      // per half: c ? a : b
  float a0, a1, b0, b1;
  upk(a, a0, a1);
  upk(b, b0, b1);
  return pk(c0 ? a0 : b0, c1 ? a1 : b1);
}

// exp(-tau) and 1 - exp(-tau) of a pair, the latter accurate for every tau (Taylor below |tau| = 0.15, as one_minus_exp_neg)
__device__ __forceinline__ void exp_and_omen2(f32x2 tau, f32x2& e, f32x2& m) {
  float t0, t1;
  upk(tau, t0, t1);
  e = pk(ex2_approx(t0 * -1.4426950408889634f), ex2_approx(t1 * -1.4426950408889634f));
  const f32x2 big = fma2(e, pk1(-1.0f), pk1(1.0f));
  const f32x2 nt = mul2(tau, pk1(-1.0f));
  f32x2 p = fma2(tau, pk1(-1.0f / 120.0f), pk1(1.0f / 24.0f));
  p = fma2(p, nt, pk1(1.0f / 6.0f));
  p = fma2(p, nt, pk1(0.5f));
  p = fma2(p, nt, pk1(1.0f));
  m = sel2(fabsf(t0) < 0.15f, fabsf(t1) < 0.15f, mul2(p, tau), big);
}

// w(tau) and w'(tau) of a pair (see w_and_wprime)
__device__ __forceinline__ void w_and_wprime2(f32x2 tau, f32x2 m, f32x2 em, f32x2 it, f32x2& w, f32x2& wp) {
  f32x2 p = fma2(tau, pk1(-1.0f / 5040.0f), pk1(1.0f / 720.0f));
  p = fma2(p, tau, pk1(-1.0f / 120.0f));
  p = fma2(p, tau, pk1(1.0f / 24.0f));
  p = fma2(p, tau, pk1(-1.0f / 6.0f));
  p = fma2(p, tau, pk1(0.5f));
  const f32x2 ws = fma2(mul2(p, pk1(-1.0f)), tau, pk1(1.0f));
  f32x2 r = fma2(tau, pk1(-1.0f / 5760.0f), pk1(1.0f / 840.0f));
  r = fma2(r, tau, pk1(-1.0f / 144.0f));
  r = fma2(r, tau, pk1(1.0f / 30.0f));
  r = fma2(r, tau, pk1(-0.125f));
  r = fma2(r, tau, pk1(1.0f / 3.0f));
  const f32x2 wps = fma2(r, tau, pk1(-0.5f));
  const f32x2 wb = mul2(m, it);
  const f32x2 wpb = mul2(mul2(fma2(em, add2(tau, pk1(1.0f)), pk1(-1.0f)), it), it);
  float t0, t1;
  upk(tau, t0, t1);
  const bool s0 = fabsf(t0) < 0.25f, s1 = fabsf(t1) < 0.25f;
  w = sel2(s0, s1, ws, wb);
  wp = sel2(s0, s1, wps, wpb);
}

constexpr int kAdjRecFields = 6;      // float4 fields of a march record (adjoint_march_kernel)

// K8: LPP lanes per pixel, 32 / LPP pixels per warp (the launcher picks 16 or 32 from nv: five spectra per pixel live in
// shared memory).  Shared memory per warp: 5 arrays (xrem, P, Q, Dt, what) of nvp * PPW floats, channel c
// of pixel g at word (c / LPP) * 32 + g * LPP + c % LPP of its array (conflict-free for the lanes of a warp).  The
// per-cell scalars (window, dust factors, gradient assembly) are computed once per pixel group, so more pixels per warp
// means fewer instructions per (pixel, cell).
template <bool DUST, bool SERIES, int LPP>
__global__ void __launch_bounds__(128)
adjoint_march_kernel(MarchConsts mc, AdjointConsts ac, const float* __restrict__ coef, const float* __restrict__ dcoef,
                     int64_t ncell, int npix, int nz, int nv, int nvp, const float* __restrict__ what,
                     float* __restrict__ grad) {
  extern __shared__ float sm[];
  constexpr int PPW = 32 / LPP;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, wpc = blockDim.x >> 5;
  const int g = lane / LPP, i = lane % LPP, gbase = g * LPP;
  const unsigned gmask = LPP == 32 ? 0xffffffffu : (((1u << (LPP & 31)) - 1u) << gbase);
  const int pix_raw = (blockIdx.x * wpc + warp) * PPW + g;
  const bool valid = pix_raw < npix;
  const int pix = valid ? pix_raw : npix - 1;                // idle groups shadow the last pixel and write nothing
  const size_t arr = (size_t)nvp * PPW;
  float* xrem = sm + (size_t)warp * 5 * arr + gbase;         // line optical depth still ahead of the march
  float* P = xrem + arr;                                     // what * exp(-xrem)
  float* Q = P + arr;                                        // what * (1 - exp(-xrem))
  float* Dt = Q + arr;                                       // (I_total - I_cont) * G, as in transfer_window.cuh
  float* wh = Dt + arr;
#define IDX(c) (((c) / LPP) * 32 + ((c) % LPP))
  float Wtot = 0.0f;
  for (int c = i; c < nvp; c += LPP) {                         // (the padding channels carry no weight)
    const float w = c < nv ? what[(int64_t)pix * nv + c] : 0.0f;
    wh[IDX(c)] = w; xrem[IDX(c)] = 0.0f; Dt[IDX(c)] = 0.0f;
    Wtot += w;
  }
  Wtot = seg_sum<LPP>(Wtot, gmask);
  __syncwarp();

  // Both marches are cut into chunks of LPP cells.  Phase A: the lane (pixel g, cell j) works out, ONCE, what depends on
  // its cell only -- window, profile polynomial, dust factors, and the quantities that depend on the march so far (G,
  // the continuum C, the dust depth passed) as prefix scans over the lanes of the pixel -- and leaves a record in shared
  // memory.  Phase B: the LPP lanes of the pixel walk the cells, reading each record with broadcast LDS.128.
  float4* rec = reinterpret_cast<float4*>(sm + (size_t)(blockDim.x >> 5) * 5 * arr) + (size_t)warp * (kAdjRecFields * 32);
  const int rl0 = gbase;                                     // records of this pixel: rec[f * 32 + gbase + j]

  // ---- first march: total line optical depth per channel and total dust optical depth
  float totD = 0.0f;
  {
    const float* pc = coef + pix + (int64_t)i * npix;
    float l_e = 0.0f, l_a = 0.0f, l_c = 0.0f, l_s = 1.0f, l_td = 0.0f;
    if (i < nz) { l_e = pc[0]; l_a = pc[ncell]; l_c = pc[2 * ncell]; l_s = pc[3 * ncell]; if (DUST) l_td = pc[4 * ncell]; }
    for (int z0 = 0; z0 < nz; z0 += LPP) {
      const bool mine = z0 + i < nz;
      const float e_c = l_e, a_c = l_a, c_los = l_c, s = l_s;
      if (DUST && mine) totD += l_td;
      l_e = 0.0f; l_a = 0.0f;
      if (z0 + LPP + i < nz) {
        pc += (int64_t)LPP * npix;
        l_e = pc[0]; l_a = pc[ncell]; l_c = pc[2 * ncell]; l_s = pc[3 * ncell];
        if (DUST) l_td = pc[4 * ncell];
      }
      int klo = 0, khi = -1;
      const int W = mine ? line_window(e_c, a_c, c_los, s, nv, klo, khi) : 0;
      CentreProfile prof;
      prof.set(s);
      rec[lane] = make_float4(s, c_los, __int_as_float(W > 0 ? (klo | (khi << 16)) : 0x0000ffff), a_c);
      rec[32 + lane] = make_float4(a_c * prof.p0, a_c * prof.p1, a_c * prof.p2, a_c * prof.p3);
      rec[64 + lane] = make_float4(a_c * prof.p4, 0.0f, 0.0f, 0.0f);
      __syncwarp();
      const int ncz = min(LPP, nz - z0);
      for (int j = 0; j < ncz; ++j) {
        const float4 r0 = rec[rl0 + j];
        const int wb = __float_as_int(r0.z), lo = wb & 0xffff, hi = (int)((unsigned)wb >> 16);
        if (hi >= lo) {
          CentreProfile pa;
          if (SERIES) {
            const float4 r1 = rec[32 + rl0 + j];
            pa.p0 = r1.x; pa.p1 = r1.y; pa.p2 = r1.z; pa.p3 = r1.w; pa.p4 = rec[64 + rl0 + j].x;
          }
          // a lane takes the even-aligned PAIR of channels c, c + 1 (the window widened to pair boundaries: the extra
          // channel lies beyond |x| = X_w, both marches treat it alike)
          for (int c = (lo & ~1) + 2 * i; c <= hi; c += 2 * LPP) {
            float2* xp = reinterpret_cast<float2*>(xrem + IDX(c));
            f32x2 dd;
            if (SERIES) dd = centre_profile_pair(pa, ((float)c + 0.5f - r0.y) * r0.x, r0.x);      // (the polynomial carries a_c)
            else dd = pk(r0.w * channel_derf(c, r0.y, r0.x), r0.w * channel_derf(c + 1, r0.y, r0.x));
            float2 v = *xp;
            const f32x2 nv2 = add2(pk(v.x, v.y), dd);
            upk(nv2, v.x, v.y);
            *xp = v;
          }
        }
        __syncwarp();
      }
    }
    totD = seg_sum<LPP>(totD, gmask);
  }
  // SQ = sum_c Q[c] and SPD = sum_c P[c] Dt[c] over ALL channels are carried as running sums: a cell changes
  // them only through the channels of its window, so the sums over the channels OUTSIDE the window (which only
  // the dust of the cell acts on) are SQ - sum_window Q and SPD - sum_window P Dt -- no pass over all nv channels.
  float SQ = 0.0f, SPD = 0.0f;
  for (int c = i; c < nvp; c += LPP) {
    const float xr = xrem[IDX(c)], w = wh[IDX(c)];
    P[IDX(c)] = w * exp_neg(xr);
    const float q = w * one_minus_exp_neg(xr);
    Q[IDX(c)] = q;
    SQ += q;
  }
  SQ = seg_sum<LPP>(SQ, gmask);
  __syncwarp();

  // ---- second march: forward state and closed-form adjoint together
  float C_run = mc.T_bg, G_run = 1.0f, D_run = 0.0f;         // continuum, exp(dust depth) since the last fold, dust depth passed
  const float* pc = coef + pix + (int64_t)i * npix;
  const float* pd = dcoef + pix + (int64_t)i * npix;
  float l_e = 0.0f, l_a = 0.0f, l_c = 0.0f, l_s = 1.0f, l_td = 0.0f, l_sd = 0.0f, l_de = 0.0f, l_da = 0.0f;
  if (i < nz) {
    l_e = pc[0]; l_a = pc[ncell]; l_c = pc[2 * ncell]; l_s = pc[3 * ncell];
    if (DUST) { l_td = pc[4 * ncell]; l_sd = pc[5 * ncell]; }
    l_de = pd[0]; l_da = pd[ncell];
  }
  for (int z0 = 0; z0 < nz; z0 += LPP) {
    // a chunk whose dust could take G out of the fp32 range is marched one cell at a time (G is folded in between)
    float tsum = DUST ? fminf(l_td, kMaxTauDCell) : 0.0f;
    if (z0 + i >= nz) tsum = 0.0f;
    tsum = seg_sum<LPP>(tsum, gmask);
    const int step = __any_sync(0xffffffffu, tsum > 60.0f) ? 1 : LPP;
    for (int jlo = 0; jlo < LPP && z0 + jlo < nz; jlo += step) {
      const int jhi = jlo + step;
      const bool mine = i >= jlo && i < jhi && z0 + i < nz;
      // ---- phase A
      const float e_c = l_e, a_c = l_a, c_los = l_c, s = l_s;
      const float tau_d = (DUST && mine) ? l_td : 0.0f, S_d = DUST ? l_sd : 0.0f;
      int klo = 0, khi = -1;
      const int W = mine ? line_window(e_c, a_c, c_los, s, nv, klo, khi) : 0;
      float E_d = 1.0f, m_d = 0.0f, Eg = 1.0f;
      if (DUST && mine) {
        const float td_e = fminf(tau_d, kMaxTauDCell);
        E_d = exp_neg(td_e);
        m_d = one_minus_exp_neg(td_e);
        Eg = ex2_approx(td_e * 1.4426950408889634f);
      }
      // prefix scans over the cells of the pixel: G (product), C (affine map x -> E_d x + S_d m_d), dust depth (sum)
      float Pg = Eg, Ac = E_d, Bc = mine ? S_d * m_d : 0.0f, Ds = tau_d;
      if (DUST) {
#pragma unroll
        for (int o = 1; o < LPP; o <<= 1) {
          const float Pp = __shfl_up_sync(0xffffffffu, Pg, o), Ap = __shfl_up_sync(0xffffffffu, Ac, o),
                      Bp = __shfl_up_sync(0xffffffffu, Bc, o), Dp = __shfl_up_sync(0xffffffffu, Ds, o);
          if (i >= o) { Pg *= Pp; Bc = fmaf(Ac, Bp, Bc); Ac *= Ap; Ds += Dp; }
        }
      }
      float Pex = __shfl_up_sync(0xffffffffu, Pg, 1), Aex = __shfl_up_sync(0xffffffffu, Ac, 1), Bex = __shfl_up_sync(0xffffffffu, Bc, 1);
      if (i == 0) { Pex = 1.0f; Aex = 1.0f; Bex = 0.0f; }
      const float Gpre = G_run * Pex, Gn = Gpre * Eg, C = fmaf(C_run, Aex, Bex);
      const float Lam = DUST ? exp_neg(totD - (D_run + Ds)) : 1.0f;      // dust attenuation between this cell and the observer
      {
        const int last = gbase + LPP - 1;
        const float Pl = __shfl_sync(0xffffffffu, Pg, last), Al = __shfl_sync(0xffffffffu, Ac, last),
                    Bl = __shfl_sync(0xffffffffu, Bc, last), Dl = __shfl_sync(0xffffffffu, Ds, last);
        G_run *= Pl; C_run = fmaf(C_run, Al, Bl); D_run += Dl;
      }
      CentreProfile prof;
      prof.set(s);
      rec[lane] = make_float4(s, c_los, __int_as_float(W > 0 ? (klo | (khi << 16)) : 0x0000ffff), a_c);
      rec[32 + lane] = make_float4(prof.p0, prof.p1, prof.p2, prof.p3);
      rec[64 + lane] = make_float4(prof.p4, e_c, tau_d, S_d);
      rec[96 + lane] = make_float4(E_d, m_d, 1.0f / Gpre, C);
      rec[128 + lane] = make_float4(C * Gpre, Gn, DUST ? 0.0f : (a_c != 0.0f ? e_c / a_c : 0.0f) - C, ac.scale * Lam);
      rec[160 + lane] = make_float4(l_de, l_da, 0.0f, 0.0f);
      // the next chunk's coefficients, requested before the cells of this one are walked
      if (jhi >= LPP || z0 + jhi >= nz) {
        l_e = 0.0f; l_a = 0.0f; l_td = 0.0f;
        if (z0 + LPP + i < nz) {
          pc += (int64_t)LPP * npix; pd += (int64_t)LPP * npix;
          l_e = pc[0]; l_a = pc[ncell]; l_c = pc[2 * ncell]; l_s = pc[3 * ncell];
          if (DUST) { l_td = pc[4 * ncell]; l_sd = pc[5 * ncell]; }
          l_de = pd[0]; l_da = pd[ncell];
        }
      }
      __syncwarp();
      // ---- phase B
      const int jend = min(jhi, min(LPP, nz - z0));
      for (int j = jlo; j < jend; ++j) {
        const float4 r0 = rec[rl0 + j], r2 = rec[64 + rl0 + j], r3 = rec[96 + rl0 + j], r4 = rec[128 + rl0 + j];
        const float sj = r0.x, cl = r0.y, aj = r0.w, ej = r2.y, tdj = r2.z, Sdj = r2.w;
        const float Edj = r3.x, mdj = r3.y, invG = r3.z, Cj = r3.w, CGj = r4.x, Gnj = r4.y, scj = r4.z;
        const int wb = __float_as_int(r0.z), lo = wb & 0xffff, hi = (int)((unsigned)wb >> 16);
        float acc_e = 0.0f, acc_a = 0.0f, acc_d = 0.0f, accW = 0.0f, accQ = 0.0f, accPD = 0.0f;
        float winQ_old = 0.0f, winQ_new = 0.0f, winPD_old = 0.0f, winPD_new = 0.0f;
        if (hi >= lo) {
          CentreProfile prof;
          if (SERIES) {
            const float4 r1 = rec[32 + rl0 + j];
            prof.p0 = r1.x; prof.p1 = r1.y; prof.p2 = r1.z; prof.p3 = r1.w; prof.p4 = r2.x;
          }
          // pairs of channels with packed arithmetic (a window of ~20 channels is one pass of 16 lanes instead of two)
          f32x2 Ae = pk1(0.0f), Aa = pk1(0.0f), Ad = pk1(0.0f), AW = pk1(0.0f), AQo = pk1(0.0f), AQn = pk1(0.0f), APo = pk1(0.0f),
                APn = pk1(0.0f);
          const f32x2 ac2 = pk1(aj), ec2 = pk1(ej), td2 = pk1(tdj), Ed2 = pk1(Edj), md2 = pk1(mdj), Sd2 = pk1(Sdj);
          const f32x2 invG2 = pk1(invG), C2 = pk1(Cj), CG2 = pk1(CGj), Gn2 = pk1(Gnj), src0 = pk1(Sdj * tdj), sc2 = pk1(scj);
          for (int c = (lo & ~1) + 2 * i; c <= hi; c += 2 * LPP) {
            const int k = IDX(c);
            f32x2 dErf;
            if (SERIES) dErf = centre_profile_pair(prof, ((float)c + 0.5f - cl) * sj, sj);
            else dErf = pk(channel_derf(c, cl, sj), channel_derf(c + 1, cl, sj));
            const f32x2 tau_L = mul2(ac2, dErf), J_L = mul2(ec2, dErf), tau_T = add2(tau_L, td2);
            const float2 xo = *reinterpret_cast<const float2*>(xrem + k), wv = *reinterpret_cast<const float2*>(wh + k);
            const float2 Do = *reinterpret_cast<const float2*>(Dt + k);
            const f32x2 xr = fma2(tau_L, pk1(-1.0f), pk(xo.x, xo.y)), w = pk(wv.x, wv.y), Dto = pk(Do.x, Do.y);
            f32x2 ex, mx;
            exp_and_omen2(xr, ex, mx);
            const f32x2 Pn = mul2(w, ex), Qn = mul2(w, mx);
            if (DUST) {
              const float2 Qo = *reinterpret_cast<const float2*>(Q + k), Po = *reinterpret_cast<const float2*>(P + k);
              AQo = add2(AQo, pk(Qo.x, Qo.y)); AQn = add2(AQn, Qn);
              APo = fma2(pk(Po.x, Po.y), Dto, APo);
            }
            {
              float2 t;
              upk(xr, t.x, t.y); *reinterpret_cast<float2*>(xrem + k) = t;
              upk(Pn, t.x, t.y); *reinterpret_cast<float2*>(P + k) = t;
              upk(Qn, t.x, t.y); *reinterpret_cast<float2*>(Q + k) = t;
            }
            const f32x2 Tk = fma2(Dto, invG2, C2);
            // 1 - exp(-tau_T) = m_d + E_d m: no second exponential, and 1 / tau_T serves w, w' and the forward step
            f32x2 eL, m;
            exp_and_omen2(tau_L, eL, m);
            const f32x2 mT = fma2(Ed2, m, md2);
            const f32x2 eT = mul2(Ed2, fma2(m, pk1(-1.0f), pk1(1.0f)));      // exp(-tau_T) itself (1 - mT is rounding noise at large tau)
            float tt0, tt1;
            upk(tau_T, tt0, tt1);
            const f32x2 r = pk(rcp_approx(fabsf(tt0) < 1.0e-30f ? 1.0f : tt0), rcp_approx(fabsf(tt1) < 1.0e-30f ? 1.0f : tt1));
            f32x2 wT, wpT;
            w_and_wprime2(tau_T, mT, eT, r, wT, wpT);
            const f32x2 src = add2(src0, J_L);
            const f32x2 dIdtau = fma2(mul2(Tk, pk1(-1.0f)), eT, mul2(src, wpT));
            Ae = fma2(mul2(Pn, wT), dErf, Ae);
            Aa = fma2(mul2(Pn, dIdtau), dErf, Aa);
            Ad = fma2(Pn, fma2(Sd2, wT, dIdtau), Ad);
            AW = add2(AW, w);
            // forward step (same cancellation-free form as transfer_window_kernel)
            f32x2 Dn;
            if (DUST) {
              const f32x2 Em = mul2(Ed2, m);
              const f32x2 t1 = add2(md2, Em);
              const f32x2 t2 = fma2(td2, Em, mul2(mul2(tau_L, md2), pk1(-1.0f)));
              const f32x2 num = fma2(J_L, t1, mul2(Sd2, t2));
              Dn = fma2(mul2(add2(Dto, CG2), pk1(-1.0f)), m, Dto);
              Dn = fma2(mul2(Gn2, r), num, Dn);
            } else {
              Dn = fma2(add2(sc2, mul2(Dto, pk1(-1.0f))), m, Dto);      // D + (S_L - C - D) m
            }
            {
              float2 t;
              upk(Dn, t.x, t.y); *reinterpret_cast<float2*>(Dt + k) = t;
            }
            if (DUST) APn = fma2(Pn, Dn, APn);
          }
          {
            float lo, hi;
            upk(Ae, lo, hi); acc_e = lo + hi;  upk(Aa, lo, hi); acc_a = lo + hi;  upk(Ad, lo, hi); acc_d = lo + hi;
            upk(AW, lo, hi); accW = lo + hi;   upk(AQo, lo, hi); winQ_old = lo + hi;  upk(AQn, lo, hi); winQ_new = lo + hi;
            upk(APo, lo, hi); winPD_old = lo + hi;  upk(APn, lo, hi); winPD_new = lo + hi;
          }
        }
        if (!DUST) {
          acc_e = seg_sum<LPP>(acc_e, gmask); acc_a = seg_sum<LPP>(acc_a, gmask);
        } else {
          if (hi >= lo) {                                        // the same for the LPP lanes of the pixel
            float r8[8] = {acc_e, acc_a, acc_d, accW, winQ_old, winQ_new, winPD_old, winPD_new};
            seg_sum8<LPP>(r8, gmask, gbase);
            acc_e = r8[0]; acc_a = r8[1]; acc_d = r8[2]; accW = r8[3];
            winQ_old = r8[4]; winQ_new = r8[5]; winPD_old = r8[6]; winPD_new = r8[7];
          }
          // channels outside the window: only the dust of this cell acts on them
          accQ = SQ - winQ_old;
          accPD = SPD - winPD_old;
          SQ += winQ_new - winQ_old;
          SPD += winPD_new - winPD_old;
        }
        if (i == 0 && valid) {
          const float4 r5 = rec[160 + rl0 + j];
          const float pre = r4.w;
          float gr = pre * (acc_e * r5.x + acc_a * r5.y);
          if (DUST) {
            const float sub = ac.subtract ? 1.0f : 0.0f;
            const float dSC = Sdj - Cj;
            const float outside = fmaf(dSC, (1.0f - sub) * (Wtot - accW) - accQ, -invG * accPD);
            const float g_d = pre * (acc_d - sub * Edj * dSC * accW + Edj * outside);
            gr = fmaf(g_d, ac.c_d, gr);
          }
          grad[(int64_t)(z0 + j) * npix + pix] = gr;
        }
        __syncwarp();
      }
      // fold the accumulated dust attenuation into the stored forward state (keeps G inside the fp32 range); rare
      if (DUST && G_run > kFoldG) {                            // the same for the LPP lanes of the pixel
        const float inv = 1.0f / G_run;
        __syncwarp(gmask);
        for (int c = i; c < nvp; c += LPP) Dt[IDX(c)] *= inv;
        SPD *= inv;
        G_run = 1.0f;
      }
      __syncwarp();
    }
  }
#undef IDX
}

// band <= kBandNarrow selects the banded elimination (BW = kBandNarrow), anything wider the dense one.
template <int N>
inline void launch_coef_grad(const LevelConsts& lc, const AdjointConsts& ac, int band, int64_t ncell, const float* n,
                             const float* T, float* dcoef, cudaStream_t st) {
  const unsigned grid = (unsigned)((ncell + 127) / 128);
  constexpr int BN = kBandNarrow < N - 1 ? kBandNarrow : N - 1;
  const bool table = lc.tb.K != nullptr;
  if (band <= BN) {
    if (table) coef_grad_kernel<N, BN, true><<<grid, 128, 0, st>>>(lc, ac, ncell, n, T, dcoef);
    else coef_grad_kernel<N, BN, false><<<grid, 128, 0, st>>>(lc, ac, ncell, n, T, dcoef);
  } else {
    if (table) coef_grad_kernel<N, N - 1, true><<<grid, 128, 0, st>>>(lc, ac, ncell, n, T, dcoef);
    else coef_grad_kernel<N, N - 1, false><<<grid, 128, 0, st>>>(lc, ac, ncell, n, T, dcoef);
  }
}

// K9 for the configured number of levels
inline cudaError_t launch_coef_grad_levels(const LevelConsts& lc, const AdjointConsts& ac, int n_levels, int band, int64_t ncell,
                                           const float* nH2, const float* Tgas, float* dcoef, cudaStream_t st) {
  switch (n_levels) {
    case 2: launch_coef_grad<2>(lc, ac, band, ncell, nH2, Tgas, dcoef, st); break;
    case 3: launch_coef_grad<3>(lc, ac, band, ncell, nH2, Tgas, dcoef, st); break;
    case 4: launch_coef_grad<4>(lc, ac, band, ncell, nH2, Tgas, dcoef, st); break;
    case 5: launch_coef_grad<5>(lc, ac, band, ncell, nH2, Tgas, dcoef, st); break;
    case 6: launch_coef_grad<6>(lc, ac, band, ncell, nH2, Tgas, dcoef, st); break;
    case 7: launch_coef_grad<7>(lc, ac, band, ncell, nH2, Tgas, dcoef, st); break;
    case 8: launch_coef_grad<8>(lc, ac, band, ncell, nH2, Tgas, dcoef, st); break;
    case 9: launch_coef_grad<9>(lc, ac, band, ncell, nH2, Tgas, dcoef, st); break;
    default: launch_coef_grad<10>(lc, ac, band, ncell, nH2, Tgas, dcoef, st); break;
  }
  return cudaGetLastError();
}

// K9 then K8.  dcoef: scratch [2][ncell].  series: every cell has dv / b <= 0.55 (channel-centre profile expansion).  Returns the first CUDA error; *launches is advanced per kernel.
inline cudaError_t launch_adjoint(const MarchConsts& mc, const AdjointConsts& ac, const LevelConsts& lc, int n_levels,
                                  int band, const float* coef, float* dcoef, int64_t ncell, int npix, int nz, int nv,
                                  bool dust, bool series, const float* nH2, const float* Tgas, const float* what, float* grad,
                                  cudaStream_t st, uint64_t* launches, bool wrt_abundance = false) {
  // abundance-only gradient: e_c and a_c are linear in the tracer abundance, so d e_c / d ln X = e_c, d a_c / d ln X = a_c
  // (the first two coefficient planes take the place of dcoef) and the dust does not depend on it (ac.c_d = 0)
  if (!wrt_abundance) {
    cudaError_t e0 = launch_coef_grad_levels(lc, ac, n_levels, band, ncell, nH2, Tgas, dcoef, st);
    if (e0 != cudaSuccess) return e0;
    ++*launches;
  }
  cudaError_t e;
  const float* dc = wrt_abundance ? coef : dcoef;
  // lanes per pixel: 16 (two pixels per warp) up to 384 channels, one warp per pixel beyond: five spectra per pixel live
  // in shared memory.  Measured on 128^3 x 256 channels: 8 lanes 1.35 ms, 16 lanes 1.05 ms, 32 lanes 1.24 ms.
  const int lpp = nv <= 384 ? 16 : 32;
  const int ppw = 32 / lpp;
  const int nvp = (nv + lpp - 1) / lpp * lpp;
  const size_t per_warp = (size_t)5 * nvp * ppw * sizeof(float) + (size_t)kAdjRecFields * 32 * sizeof(float4);   // spectra + march records
  int wpc = 4;
  while (wpc > 1 && wpc * per_warp > 200 * 1024) wpc >>= 1;
  const size_t smem = wpc * per_warp;
  if (smem > 227 * 1024) return cudaErrorInvalidConfiguration;
  const unsigned grid = (unsigned)((npix + wpc * ppw - 1) / (wpc * ppw));
#define IRIS_LAUNCH_ADJ(D_, S_, L_)                                                                                        \
  do {                                                                                                                     \
    e = cudaFuncSetAttribute(adjoint_march_kernel<D_, S_, L_>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);    \
    if (e != cudaSuccess) return e;                                                                                        \
    adjoint_march_kernel<D_, S_, L_><<<grid, wpc * 32, smem, st>>>(mc, ac, coef, dc, ncell, npix, nz, nv, nvp, what, grad); \
  } while (0)
#define IRIS_LAUNCH_ADJ_L(D_, S_)                                         \
  do {                                                                    \
    if (lpp == 8) IRIS_LAUNCH_ADJ(D_, S_, 8);                             \
    else if (lpp == 16) IRIS_LAUNCH_ADJ(D_, S_, 16);                      \
    else IRIS_LAUNCH_ADJ(D_, S_, 32);                                     \
  } while (0)
  if (dust) { if (series) IRIS_LAUNCH_ADJ_L(true, true); else IRIS_LAUNCH_ADJ_L(true, false); }
  else { if (series) IRIS_LAUNCH_ADJ_L(false, true); else IRIS_LAUNCH_ADJ_L(false, false); }
#undef IRIS_LAUNCH_ADJ_L
#undef IRIS_LAUNCH_ADJ
  e = cudaGetLastError();
  if (e == cudaSuccess) ++*launches;
  return e;
}

}  // namespace iris
