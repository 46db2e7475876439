// K3 (line-window formulation, narrow channels): the production LOS transfer kernel.
//
// Same recurrence and the same line window as transfer_window.cuh (difference form D = I^[T] - I^[C],
// Dt = D * exp(sum tau_d), updates only inside |x| <= X_w), with the instruction count per update cut to what
// the recurrence needs:
//
// 1. Profile.  When a channel is narrower than ~half a Doppler width (s = dv / b <= kSeriesMaxS), the channel
//    integral of the Gaussian profile (Eq. 4.6.3) is evaluated from the channel CENTRE x by
//    the Taylor expansion of the integrand about the centre,
//      erf(x + s/2) - erf(x - s/2) = (2 s / sqrt(pi)) exp(-x^2) [1 + (s^2/24) H_2(x) + (s^4/1920) H_4(x)
//                                     + (s^6/322560) H_6(x) + (s^8/92897280) H_8(x)],   H_n = Hermite polynomials,
//    i.e. exp(-x^2) times a polynomial in x^2 whose coefficients depend on the cell only.  Degree 4 in x^2 up to
//    s = 0.55 (truncation <= 2e-7 relative for |x| <= 3, <= 2e-9 absolute everywhere); degree 3 up to s = 0.3
//    (the dropped term is s^8 x^8 / 362880 <= 1.5e-6 relative at |x| = 3.2, where the profile is 4e-5 of its peak).
// 2. Units.  The line opacity is folded into the polynomial, and everything is carried in base-2 units, so the
//    line optical depth of the update comes out of ONE multiply:  t = tau_L log2(e) = 2^(-x'^2) * polA(x'^2),
//    x' = x sqrt(log2 e);  1 - exp(-tau_L) = 1 - 2^(-t);  1 / tau_T = log2(e) / (t + tau_d log2(e)).
// 3. Per-cell work is done ONCE per cell, not once per lane: the march is cut into chunks of LPP cells; in
//    phase A every lane turns the six coefficients of one (cell, pixel) of the chunk into a "march record"
//    (window, scaled coordinates, polynomial, dust factors) in shared memory; in phase B the LPP lanes of a pixel
//    walk the LPP cells, reading each record with broadcast LDS.128 one cell ahead of its use.
// 4. Packed arithmetic.  A lane updates the two channels of an even-aligned PAIR with the packed fp32 instructions
//    of sm_100 (fma/mul/add.rn.f32x2 -> FFMA2 / FMUL2 / FADD2): the kernel is bound by instruction issue, not by
//    the FMA pipe, and a packed instruction does two updates per issue slot (profiles/r01_pipe_microbench.md).
//    Only the MUFU operations (2 ex2 + 1 rcp per update) and the small-tau select stay scalar.  The window is
//    widened to pair boundaries; the extra channel lies beyond |x| = X_w where the update is below the window
//    threshold anyway, so no per-channel predicate is needed.  The loop is branch-free (predicated LDS.64 /
//    STS.64) and two pair-passes are written stage by stage so that four dependency chains are in flight.
//
// Mapping: a warp owns 32/LPP adjacent pixels, LPP lanes per pixel; the spectrum Dt[nv] of each pixel lives in
// shared memory for the whole march.  Pair q = c / 2 of pixel g sits at word (q / LPP) * 64 + g * 2 LPP +
// (q % LPP) * 2: each half-warp of an LDS.64 / STS.64 hits 32 distinct banks.  Records are stored
// quantity-major ([float4 index][record]) so that both the phase-A stores and the phase-B broadcast loads are
// conflict-free.
#pragma once
#include "transfer_common.cuh"
#include "transfer_window.cuh"

namespace iris {

constexpr float kSeriesMaxS = 0.55f;    // largest dv / b the centre expansion is used for
constexpr float kSeriesDeg3MaxS = 0.3f; // largest dv / b for the degree-3 polynomial

// March record of one (cell, pixel): NQ float4
//   q0 = { x0, xs, tdp | -sc, bits(qlo | nq << 16) } x0: scaled centre of channel 2 qlo, xs: scaled channel step,
//                                                    tdp = tau_d log2(e) + 1e-30 (dust), sc = S_L - T_bg (no dust),
//                                                    window = pairs qlo .. qlo + nq - 1 (nq = 0: empty)
//   q1 = { pA0, pA1, pA2, pA3 }                      polA(u') = As' pol(u'),  As' = a_c (2 s / sqrt(pi)) log2(e)
//   q2 = { P', -Q', -R', E_d }                       num' = t P' + m (Q' t + R')   (to be scaled by G')
//   q3 = { S_d m_d, exp(tau_d), pA4, - }             (without dust: pA4 in q2.x)
template <bool DUST, int DEG>
struct SeriesLayout {
  static constexpr int NQ = DUST ? 4 : (DEG > 3 ? 3 : 2);
};

struct SeriesRecord { float4 q0, q1, q2, q3; };

// Weights of the sum along the ray in the optically thin mode with smooth integration (Eq. 4.7.7, reading S25): composite
// Simpson's rule over the largest odd number of cells, the last interval of an even count by the trapezoidal rule.
__device__ __forceinline__ float ray_simpson_weight(int n, int nz) {
  const int Rs = (nz & 1) ? nz : nz - 1;
  float wn = 0.0f;
  if (Rs >= 3 && n < Rs) wn = (n == 0 || n == Rs - 1) ? (1.0f / 3.0f) : ((n & 1) ? (4.0f / 3.0f) : (2.0f / 3.0f));
  if (!(nz & 1) && nz >= 2 && n >= nz - 2) wn += 0.5f;
  return wn;
}

// Phase A: coefficients of one cell -> march record.
// MODE 0: optically thick formal step (the hot path).  MODE 1: selectively thin, formal (Eq. 4.8.13 - 4.8.15): the
// polynomial gives the erf difference itself, q2 = { e_c w(tau_d), a_c w(tau_d), -, E_d }.  MODE 2: optically thin, formal
// (Eq. 4.7.3 - 4.7.6): the polynomial gives E = e_c dErf, no attenuation (E_d = exp(tau_d) = 1), continuum adds tau_d S_d.
// MODE 3: optically thick formal step on the fine velocity grid (Eq. 4.5.1): the spectrum holds the nv m + 1 POINTS
// k / m (channel-edge units), the profile is the point value (2 s / sqrt(pi)) exp(-x^2) of Eq. 3.3.3 in erf-difference
// units (polynomial = 1), the points are spaced s / m Doppler widths; Simpson's rule over a channel is the epilogue.
template <bool DUST, int DEG, int MODE = 0>
// wn: weight of the cell in the sum along the ray (MODE 2 only; 1 for the midpoint sum of Eq. 4.7.6).
__device__ __forceinline__ SeriesRecord make_series_record(float e_c, float a_c, float c_los, float s, float tau_d,
                                                           float S_d, float T_bg, int nv, int fine_m, float wn = 1.0f) {
  constexpr float LOG2E = 1.4426950408889634f;
  SeriesRecord r;
  int klo, khi;
  const float s_amp = s;                       // the amplitude is per channel width in every mode
  if (MODE == 3) {                             // point k sits where "channel" k of width 1 / m has its centre
    c_los = fmaf(c_los, (float)fine_m, 0.5f);
    s = s / (float)fine_m;
  }
  int W = line_window(e_c, a_c, c_los, s, nv, klo, khi);
  int qlo = 0, nq = 0;
  if (W > 0) { qlo = klo >> 1; nq = (khi >> 1) - qlo + 1; }
  // |a_c| is kept above 1e-10 e_c: the source function e_c / a_c stays finite where the opacity crosses zero
  // (changes tau_L by < 1e-10 e_c, i.e. < 1e-7 for a 1000 K line)
  const float a_min = fmaxf(1.0e-10f * e_c, 1.0e-30f);
  const float a_safe = fabsf(a_c) < a_min ? a_min : a_c;
  const float sp = 1.1283791670955126f * s_amp;             // 2 s / sqrt(pi)
  const float As = a_safe * sp, Es = (MODE == 2 ? wn : 1.0f) * e_c * sp;
  const float Asp = (MODE == 0 || MODE == 3) ? As * LOG2E : (MODE == 1 ? sp : Es);   // what the polynomial is scaled by
  const float xs = 1.2011224087864498f * s;                 // s sqrt(log2 e)
  r.q0.x = ((float)(2 * qlo) + 0.5f - c_los) * xs;
  r.q0.y = xs;
  r.q0.w = __int_as_float(qlo | (nq << 16));
  // polynomial in u = x^2, rescaled to u' = u log2(e) (p'_k = p_k ln(2)^k) and multiplied by As'
  const float s2 = MODE == 3 ? 0.0f : s * s, s4 = s2 * s2, s6 = s4 * s2, s8 = s4 * s4;
  const float p0 = 1.0f - s2 * (1.0f / 12.0f) + s4 * (1.0f / 160.0f) - s6 * (1.0f / 2688.0f) + s8 * (1.0f / 55296.0f);
  const float p1 = s2 * (1.0f / 6.0f) - s4 * (1.0f / 40.0f) + s6 * (1.0f / 448.0f) - s8 * (1.0f / 6912.0f);
  const float p2 = s4 * (1.0f / 120.0f) - s6 * (1.0f / 672.0f) + s8 * (1.0f / 6912.0f);
  const float p3 = s6 * (1.0f / 5040.0f) - s8 * (1.0f / 25920.0f);
  const float p4 = s8 * (1.0f / 362880.0f);
  constexpr float L1 = 0.6931471805599453f, L2 = L1 * L1, L3 = L2 * L1, L4 = L2 * L2;
  r.q1 = make_float4(Asp * p0, Asp * (p1 * L1), Asp * (p2 * L2), Asp * (p3 * L3));
  r.q3.z = DEG > 3 ? Asp * (p4 * L4) : 0.0f;
  r.q3.w = 0.0f;
  if (MODE == 2) {
    r.q0.z = 0.0f;
    r.q2 = make_float4(0.0f, 0.0f, 0.0f, 1.0f);
    r.q3.x = wn * tau_d * S_d;
    r.q3.y = 1.0f;
  } else if (MODE == 1) {
    const float td_e = fminf(tau_d, kMaxTauDCell);
    const float E_d = exp_neg(td_e);
    const float m_d = one_minus_exp_neg(td_e);
    const float w_d = fabsf(tau_d) < 1.0e-3f ? fmaf(tau_d, fmaf(tau_d, 1.0f / 6.0f, -0.5f), 1.0f) : m_d * rcp_approx(tau_d);
    r.q0.z = 0.0f;
    r.q2 = make_float4(e_c * w_d, a_c * w_d, 0.0f, E_d);
    r.q3.x = S_d * m_d;
    r.q3.y = ex2_approx(td_e * LOG2E);
  } else if (DUST) {
    const float td_e = fminf(tau_d, kMaxTauDCell);
    const float E_d = exp_neg(td_e);
    const float m_d = one_minus_exp_neg(td_e);
    const float iA = LOG2E * rcp_approx(Asp);
    r.q0.z = fmaf(tau_d, LOG2E, 1.0e-30f);
    r.q2.x = m_d * fmaf(-S_d, As, Es) * iA;
    r.q2.y = -E_d * Es * iA;
    r.q2.z = -E_d * S_d * tau_d * LOG2E;
    r.q2.w = E_d;
    r.q3.x = S_d * m_d;
    r.q3.y = ex2_approx(td_e * LOG2E);
  } else {
    r.q0.z = T_bg - Es * rcp_approx(As);      // -sc = C - S_L, C = T_bg throughout
    r.q2 = make_float4(r.q3.z, 0.0f, 0.0f, 1.0f);   // pA4 travels in q2.x when there is no dust (NQ = 3)
    r.q3.x = 0.0f; r.q3.y = 1.0f;
  }
  return r;
}

// (packed fp32 pairs -- f32x2, pk, pk1, upk, fma2, mul2, add2 -- are in iris_math.cuh)

// Per-cell operands of the update, duplicated into both halves of a packed register.
struct SeriesCellOps {
  f32x2 p0, p1, p2, p3, p4;     // polA
  f32x2 tdp_or_nsc;             // dust: tau_d log2(e) + 1e-30;  no dust: -(S_L - T_bg)
  f32x2 CG, Pn, nQn, nRn;       // dust only (scaled by G')
};

// P consecutive pair-passes of one lane (pairs q, q + LPP, ...), written stage by stage over the 2 P channels so
// that 2 P independent dependency chains are in flight (the SM issues in order: a lane-serial update would leave
// the issue slot idle for the latency of every MUFU / FMA of the chain).  d: the lane's words of pair q; pairs at
// or beyond qend are computed but neither loaded nor stored.  xx: scaled centres of the two channels of pair q.
// CIRC: the spectra are circular buffers of rmask + 1 rows (see the kernel); col = the lane's column of its first row, row its
// first row: pass k works on row (row + k) & rmask.
template <bool DUST, int DEG, int LPP, int P, int MODE = 0, bool CIRC = false>
__device__ __forceinline__ void series_passes(float* col, int row, int rmask, f32x2 xx, f32x2 step2, const SeriesCellOps& o) {
  float* dk[P];
#pragma unroll
  for (int k = 0; k < P; ++k) dk[k] = col + (CIRC ? ((row + k) & rmask) : (row + k)) * 64;
  constexpr float L1 = 0.6931471805599453f, L2 = L1 * L1, L3 = L2 * L1, L4 = L2 * L2;
  const f32x2 ONE = pk1(1.0f), NEG1 = pk1(-1.0f);
  const f32x2 C4 = pk1(L4 / 24.0f), C3 = pk1(-L3 / 6.0f), C2 = pk1(L2 / 2.0f), C1 = pk1(-L1);   // -(1 - 2^-t) / t
  f32x2 Dt[P], u[P], pol[P], t[P], mn[P], qq[P];
#pragma unroll
  for (int k = 0; k < P; ++k) {
    const float2 v = *reinterpret_cast<const float2*>(dk[k]);
    Dt[k] = pk(v.x, v.y);
    u[k] = mul2(xx, xx);
    xx = add2(xx, step2);
  }
#pragma unroll
  for (int k = 0; k < P; ++k) pol[k] = DEG > 3 ? fma2(fma2(o.p4, u[k], o.p3), u[k], o.p2) : fma2(o.p3, u[k], o.p2);
#pragma unroll
  for (int k = 0; k < P; ++k) pol[k] = fma2(pol[k], u[k], o.p1);
#pragma unroll
  for (int k = 0; k < P; ++k) pol[k] = fma2(pol[k], u[k], o.p0);
#pragma unroll
  for (int k = 0; k < P; ++k) {
    float u0, u1;
    upk(u[k], u0, u1);
    t[k] = mul2(pk(ex2_approx(-u0), ex2_approx(-u1)), pol[k]);      // tau_L log2(e)  (MODE 1: dErf, MODE 2: e_c dErf)
  }
  if constexpr (MODE == 1 || MODE == 2) {
    // thin: Dt += E.  selectively thin: Dt' = max(Dt + K dErf, -C' G'),  K = G' w(tau_d) (e_c - a_c C') in o.Pn, the clamp in o.CG
#pragma unroll
    for (int k = 0; k < P; ++k) {
      if (MODE == 2) Dt[k] = add2(Dt[k], t[k]);
      else {
        const f32x2 v = fma2(o.Pn, t[k], Dt[k]);
        float v0, v1, c0, c1;
        upk(v, v0, v1);
        upk(o.CG, c0, c1);
        Dt[k] = pk(fmaxf(v0, c0), fmaxf(v1, c1));
      }
      float2 w;
      upk(Dt[k], w.x, w.y);
      *reinterpret_cast<float2*>(dk[k]) = w;
    }
  } else {
  float t0[P], t1[P], f0[P], f1[P];
#pragma unroll
  for (int k = 0; k < P; ++k) {
    upk(t[k], t0[k], t1[k]);
    f0[k] = ex2_approx(-t0[k]);
    f1[k] = ex2_approx(-t1[k]);
    qq[k] = fma2(t[k], C4, C3);
  }
#pragma unroll
  for (int k = 0; k < P; ++k) qq[k] = fma2(qq[k], t[k], C2);
#pragma unroll
  for (int k = 0; k < P; ++k) qq[k] = fma2(qq[k], t[k], C1);
#pragma unroll
  for (int k = 0; k < P; ++k) {
    // mn = -(1 - exp(-tau_L)) = 2^-t - 1; Taylor below tau_L = 0.08
    const f32x2 sm = mul2(qq[k], t[k]);
    const f32x2 bg = add2(pk(f0[k], f1[k]), NEG1);
    float s0, s1, b0, b1;
    upk(sm, s0, s1);
    upk(bg, b0, b1);
    mn[k] = pk(fabsf(t0[k]) < 0.115f ? s0 : b0, fabsf(t1[k]) < 0.115f ? s1 : b1);
  }
  if (DUST) {
    f32x2 rr[P], num[P];
#pragma unroll
    for (int k = 0; k < P; ++k) {
      const f32x2 tt = add2(t[k], o.tdp_or_nsc);
      float a0, a1;
      upk(tt, a0, a1);
      rr[k] = pk(rcp_approx(a0), rcp_approx(a1));
      num[k] = fma2(o.nQn, t[k], o.nRn);                       // -(Q t + R)
    }
#pragma unroll
    for (int k = 0; k < P; ++k) {
      num[k] = fma2(mn[k], num[k], mul2(t[k], o.Pn));           // t P + m (Q t + R)
      Dt[k] = fma2(add2(Dt[k], o.CG), mn[k], Dt[k]);            // Dt - (Dt + C G) m
    }
#pragma unroll
    for (int k = 0; k < P; ++k) Dt[k] = fma2(rr[k], num[k], Dt[k]);
  } else {
#pragma unroll
    for (int k = 0; k < P; ++k) Dt[k] = fma2(add2(Dt[k], o.tdp_or_nsc), mn[k], Dt[k]);   // Dt + (sc - Dt) m
  }
  (void)ONE;
#pragma unroll
  for (int k = 0; k < P; ++k) {
    float2 v;
    upk(Dt[k], v.x, v.y);
    *reinterpret_cast<float2*>(dk[k]) = v;
  }
  }
}

// __launch_bounds__ names a minimum of 3 CTAs per SM (what the 1024-channel spectra allow): without it ptxas holds the
// kernel to 68 registers and schedules the two pair-passes of the loop back to back; with it it takes 86 registers and
// overlaps them (large: 6.61 -> 6.27 ms).
// CIRC (reachable-range spectra): a pixel's lines only ever touch the channels its line-of-sight velocities reach, a
// fraction of the band, but whole spectra of 4 pixels per warp are what limits the resident warps (12 per SM at 1024
// channels).  With CIRC a spectrum is a CIRCULAR buffer of rb = rmask + 1 rows of LPP pairs (a power of two, half the band or
// less): row r of the spectrum lives in buffer row r & rmask, which is one-to-one as long as the rows a pixel has
// touched so far span at most rb rows.  The kernel tracks that span per pixel; a pixel that exceeds it is appended to
// the hand-over list `hand` ([0] count of this launch, [1] count since the public call began, [2..] pixel indices) and a
// second launch of the full-size variant over that list (`plist`, `pcount`) recomputes it.  Rows never touched are zero.
template <int LPP, bool DUST, int DEG, int MODE, bool CIRC = false>
__global__ void __launch_bounds__(128, 3)
transfer_series_kernel(MarchConsts mc, const float* __restrict__ coef, int64_t ncell, int npix, int nz, int nv,
                       int nvp, float* __restrict__ out, float* __restrict__ out_cont, int rmask, int* __restrict__ hand,
                       const int* __restrict__ plist, const int* __restrict__ pcount) {
  extern __shared__ float4 smem4[];
  constexpr int PPW = 32 / LPP;
  constexpr int NQ = SeriesLayout<DUST, DEG>::NQ;
  constexpr int ROW = 2 * 32;                   // words per row of LPP pairs x PPW pixels
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, wpc = blockDim.x >> 5;
  const int g = lane / LPP, i = lane % LPP;
  const int pix0 = (blockIdx.x * wpc + warp) * PPW;
  // list-driven launch: the warp's pixels are entries pix0 .. pix0 + PPW - 1 of the list
  const int nlist = plist != nullptr ? *pcount : 0;
  if (plist != nullptr && pix0 >= nlist) return;
  auto pixel_of = [&](int slot) { return plist != nullptr ? (slot < nlist ? plist[slot] : npix) : slot; };
  const int pix = pixel_of(pix0 + g);
  const bool valid = pix < npix;
  const int nvb = CIRC ? (rmask + 1) * 2 * LPP : nvp;      // points of the buffer that holds a spectrum
  const int npair = nvb / 2;                    // nvp is a multiple of 2 LPP
  const int npts = MODE == 3 ? nv * mc.fine_m + 1 : nv;      // spectral points held per pixel
  // shared memory: records [wpc][NQ][32], then spectra [wpc][npair / LPP rows][ROW]
  float4* rec = smem4 + (size_t)warp * (NQ * 32);
  float* spec = reinterpret_cast<float*>(smem4 + (size_t)wpc * (NQ * 32));
  float* sp = spec + (size_t)warp * nvb * PPW + g * (2 * LPP);      // pair q of this pixel: sp[(q / LPP) * ROW + (q % LPP) * 2]
  for (int q = i; q < npair; q += LPP) *reinterpret_cast<float2*>(sp + (q / LPP) * ROW + i * 2) = make_float2(0.0f, 0.0f);

  float C = mc.T_bg;      // continuum before the current cell
  float G = 1.0f;         // exp(dust optical depth accumulated so far), since the last rescale
  int row_min = 0x3fffffff, row_max = -1;       // CIRC: rows of the spectrum pixel ga (= lane % PPW) has touched
  bool overflow = false;                        // CIRC: they no longer fit the buffer

  // phase A: lane L makes record L of the chunk = (cell L / PPW, pixel L % PPW)
  const int ja = lane / PPW, ga = lane % PPW;
  const float* p = coef + min(pixel_of(pix0 + ga), npix - 1) + (int64_t)ja * npix;
  float l_e = 0.0f, l_a = 0.0f, l_c = 0.0f, l_s = 1.0f, l_td = 0.0f, l_sd = 0.0f;
  if (ja < nz) {
    l_e = p[0]; l_a = p[ncell]; l_c = p[2 * ncell]; l_s = p[3 * ncell];
    if (DUST) { l_td = p[4 * ncell]; l_sd = p[5 * ncell]; }
  }

  // rare: fold the accumulated dust attenuation into the stored spectrum (keeps G inside the fp32 range)
  auto rescale_spectrum = [&]() {
    const float inv = 1.0f / G;
    __syncwarp(__activemask());
    for (int qq = i; qq < npair; qq += LPP) {
      float2* w = reinterpret_cast<float2*>(sp + (qq / LPP) * ROW + i * 2);
      float2 v = *w;
      v.x *= inv; v.y *= inv;
      *w = v;
    }
    G = 1.0f;
  };

  // one cell of phase B for this lane's pixel, given the cell's record in registers
  auto cell_step = [&](const float4& q0, const float4& q1, const float4& q2, const float4& q3) {
    const int kk = __float_as_int(q0.w);
    const int qlo = kk & 0xffff, nq = (int)((unsigned)kk >> 16);
    const int npass = (nq + LPP - 1) / LPP;      // pair-passes of THIS pixel (the warp runs the longest of its pixels)
    float CG = 0.0f, Pn = 0.0f, Qn = 0.0f, Rn = 0.0f;
    if (DUST) {
      const float Gn = G * q3.y;
      CG = C * G;
      C = fmaf(C, q2.w, q3.x);
      if (MODE == 1) {                       // selectively thin: K = G' w_d (e_c - a_c C'), clamp at I_T = 0: D >= -C'
        Pn = Gn * fmaf(-q2.y, C, q2.x);
        CG = -C * Gn;
      } else {
        Pn = q2.x * Gn; Qn = q2.y * Gn; Rn = q2.z * Gn;
      }
      G = Gn;
    }
    if (npass > 0) {
      SeriesCellOps o;
      o.p0 = pk1(q1.x); o.p1 = pk1(q1.y); o.p2 = pk1(q1.z); o.p3 = pk1(q1.w);
      o.p4 = pk1(DUST ? q3.z : q2.x);
      o.tdp_or_nsc = pk1(q0.z);
      o.CG = pk1(CG); o.Pn = pk1(Pn); o.nQn = pk1(Qn); o.nRn = pk1(Rn);
      const int q = qlo + i;
      const float x = fmaf((float)(2 * i), q0.y, q0.x);
      f32x2 xx = pk(x, x + q0.y);
      const f32x2 step2 = pk1((float)(2 * LPP) * q0.y);
      float* col = sp + (q % LPP) * 2;             // the lane's column; pass k works on row q / LPP + k
      int row = q / LPP;
      // (checked build) the pairs of every pass of this lane lie inside the spectra of this warp
      IRIS_CHECK_SMEM(col + (CIRC ? (row & rmask) : row) * ROW, 8, spec + (size_t)warp * nvb * PPW, spec + (size_t)(warp + 1) * nvb * PPW);
      IRIS_CHECK_SMEM(col + (CIRC ? ((row + npass - 1) & rmask) : row + npass - 1) * ROW, 8, spec + (size_t)warp * nvb * PPW,
                      spec + (size_t)(warp + 1) * nvb * PPW);
      int rem = npass;
      while (rem >= 2) {
        series_passes<DUST, DEG, LPP, 2, MODE, CIRC>(col, row, rmask, xx, step2, o);
        xx = add2(xx, add2(step2, step2)); row += 2; rem -= 2;
      }
      if (rem == 1) series_passes<DUST, DEG, LPP, 1, MODE, CIRC>(col, row, rmask, xx, step2, o);
    }
    if (DUST && G > kFoldG) rescale_spectrum();
  };

  bool chunk_busy = true;
  for (int z0 = 0; z0 < nz; z0 += LPP) {
    // ---- phase A: one record per lane
    {
      float wn = 1.0f;
      if (MODE == 2 && mc.ray_simpson) wn = ray_simpson_weight(z0 + ja, nz);
      const SeriesRecord r = make_series_record<DUST, DEG, MODE>(l_e, l_a, l_c, l_s, l_td, l_sd, mc.T_bg, npts, mc.fine_m, wn);
      chunk_busy = __any_sync(0xffffffffu, ((unsigned)__float_as_int(r.q0.w) >> 16) != 0u);   // also: phase B is done
      if (CIRC) {
        // rows of the spectrum the chunk touches, per pixel ga (lanes ga, ga + PPW, ...): qlo / LPP .. (qlo + LPP npass - 1) / LPP
        const int kk = __float_as_int(r.q0.w), qlo_r = kk & 0xffff, nq_r = (int)((unsigned)kk >> 16);
        int lo = nq_r > 0 ? qlo_r / LPP : 0x3fffffff;
        int hi = nq_r > 0 ? (qlo_r + (nq_r + LPP - 1) / LPP * LPP - 1) / LPP : -1;
#pragma unroll
        for (int o = PPW; o < 32; o <<= 1) {
          lo = min(lo, __shfl_xor_sync(0xffffffffu, lo, o));
          hi = max(hi, __shfl_xor_sync(0xffffffffu, hi, o));
        }
        row_min = min(row_min, lo);
        row_max = max(row_max, hi);
        if (row_max - row_min > rmask) overflow = true;      // (noticed after the fact: the pixel is recomputed anyway)
      }
      rec[lane] = r.q0;
      rec[32 + lane] = r.q1;
      if (NQ > 2) rec[64 + lane] = r.q2;
      if (NQ > 3) rec[96 + lane] = r.q3;
      // prefetch the next chunk's coefficients
      const int zn = z0 + LPP + ja;
      l_e = 0.0f; l_a = 0.0f; l_td = 0.0f;
      if (zn < nz) {
        p += (int64_t)LPP * npix;
        l_e = p[0]; l_a = p[ncell]; l_c = p[2 * ncell]; l_s = p[3 * ncell];
        if (DUST) { l_td = p[4 * ncell]; l_sd = p[5 * ncell]; }
      }
      __syncwarp();
    }
    // ---- phase B: the LPP lanes of a pixel walk the cells of the chunk, records read one cell ahead
    const int ncz = min(LPP, nz - z0);
    const float4* rq = rec + g;
    if (!chunk_busy) {
      // no pixel of the warp has a line in any cell of the chunk (columns whose velocity is outside the band): only
      // the continuum and the accumulated dust attenuation advance
      if (DUST) {
        for (int j = 0; j < ncz; ++j) {
          const float E_d = rq[64 + j * PPW].w;
          const float4 c3 = rq[96 + j * PPW];
          C = fmaf(C, E_d, c3.x);
          G *= c3.y;
          if (G > kFoldG) rescale_spectrum();
        }
      }
      continue;
    }
    float4 a0 = rq[0], a1 = rq[32], a2 = NQ > 2 ? rq[64] : float4{}, a3 = NQ > 3 ? rq[96] : float4{};
    for (int j = 0; j < ncz; j += 2) {
      const int jb = min(j + 1, ncz - 1) * PPW;
      const float4 b0 = rq[jb], b1 = rq[32 + jb], b2 = NQ > 2 ? rq[64 + jb] : float4{}, b3 = NQ > 3 ? rq[96 + jb] : float4{};
      cell_step(a0, a1, a2, a3);
      __syncwarp();      // the lane -> pair mapping follows each cell's window: cell j + 1 reads pairs other lanes wrote in cell j
      const int jn = min(j + 2, ncz - 1) * PPW;
      a0 = rq[jn]; a1 = rq[32 + jn];
      if (NQ > 2) a2 = rq[64 + jn];
      if (NQ > 3) a3 = rq[96 + jn];
      if (j + 1 < ncz) cell_step(b0, b1, b2, b3);
      __syncwarp();
    }
  }
  __syncwarp();

  if (CIRC) {
    // the range of THIS lane's pixel g is held by the lanes with ga = g (lane g is one of them)
    row_min = __shfl_sync(0xffffffffu, row_min, g);
    row_max = __shfl_sync(0xffffffffu, row_max, g);
    overflow = __shfl_sync(0xffffffffu, (int)overflow, g) != 0;
    // hand the pixel over when its rows did not fit the buffer (the full-size variant recomputes it)
    if (overflow && valid && i == 0) { hand[2 + atomicAdd(hand, 1)] = pix; atomicAdd(hand + 1, 1); }
  }
  // buffer word of pair q (q = i + LPP row for this lane); CIRC: rows outside the touched range are zero
  auto pair_at = [&](int q) {
    const int row = q / LPP;
    if (!CIRC) return *reinterpret_cast<const float2*>(sp + row * ROW + (q % LPP) * 2);
    if (row < row_min || row > row_max) return make_float2(0.0f, 0.0f);
    return *reinterpret_cast<const float2*>(sp + (row & rmask) * ROW + (q % LPP) * 2);
  };
  const float invG = 1.0f / G;
  if (MODE == 3) {
    // Simpson's rule over the m + 1 points of every channel (Eq. 4.5.1), then subtraction / conversion
    if (valid && out != nullptr) {
      const int m = mc.fine_m;
      const float wgt = invG / (3.0f * (float)m);
      auto point = [&](int k) { const float2 v = pair_at(k >> 1); return (k & 1) ? v.y : v.x; };
      for (int c = i; c < nv; c += LPP) {
        float acc = 0.0f;
        for (int j = 0; j < m; j += 2) acc += point(c * m + j) + 4.0f * point(c * m + j + 1) + point(c * m + j + 2);
        out[(int64_t)pix * nv + c] = convert_out(acc * wgt, C, mc);
      }
    }
    if (valid && out_cont != nullptr && i == 0) out_cont[pix] = C * mc.inv_KRJ;
    return;
  }
  if (valid) {
    if (out != nullptr) {
      float* o = out + (int64_t)pix * nv;
      const bool al = ((((int64_t)pix * nv) & 1) == 0);      // float2 stores need an even element offset
      if (MODE != 1 && mc.out_mode <= OUT_I_TOT && al && (nv & 1) == 0) {
        // the units that are linear in D (Rayleigh-Jeans Kelvin or intensity, with or without the continuum): one
        // multiply-add per value, four pairs per lane in flight (the loop is latency-bound: LDS -> FMA -> STG)
        const float sc = mc.out_mode >= OUT_I_SUB ? mc.inv_KRJ : 1.0f;
        const float a = invG * sc, b = (mc.out_mode & 1) ? C * sc : 0.0f;
        float2* o2 = reinterpret_cast<float2*>(o);
        const int nq = nv / 2;
        int q = i;
        for (; q + 3 * LPP < nq; q += 4 * LPP) {
          float2 v[4];
#pragma unroll
          for (int k = 0; k < 4; ++k) v[k] = pair_at(q + k * LPP);
#pragma unroll
          for (int k = 0; k < 4; ++k) o2[q + k * LPP] = make_float2(fmaf(v[k].x, a, b), fmaf(v[k].y, a, b));
        }
        for (; q < nq; q += LPP) {
          const float2 v = pair_at(q);
          o2[q] = make_float2(fmaf(v.x, a, b), fmaf(v.y, a, b));
        }
      } else
      for (int q = i; 2 * q < nv; q += LPP) {
        const float2 v = pair_at(q);
        // (selectively thin: the ReLU keeps I_T = D + C >= 0; the clamp was applied to the dust-scaled spectrum, and
        // unscaling it can leave D one rounding below -C)
        const float d0 = MODE == 1 ? fmaxf(v.x * invG, -C) : v.x * invG, d1 = MODE == 1 ? fmaxf(v.y * invG, -C) : v.y * invG;
        const float r0 = convert_out(d0, C, mc);
        if (2 * q + 1 < nv) {
          const float r1 = convert_out(d1, C, mc);
          if (al) *reinterpret_cast<float2*>(o + 2 * q) = make_float2(r0, r1);
          else { o[2 * q] = r0; o[2 * q + 1] = r1; }
        } else {
          o[2 * q] = r0;
        }
      }
    }
    if (out_cont != nullptr && i == 0) out_cont[pix] = C * mc.inv_KRJ;
  }
}

// Warps per CTA that leave most warps resident for `per_warp` bytes of shared memory per warp, and that number of warps
// (shared memory and, through the occupancy query, registers).
template <typename Kernel>
inline void series_residency(Kernel kernel, size_t per_warp, int& wpc, int& resident) {
  wpc = 1; resident = 0;
  for (int w = 4; w >= 1; w >>= 1) {
    const size_t smem = w * per_warp;
    if (smem + 1024 > 227 * 1024) continue;
    if (cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) { cudaGetLastError(); continue; }
    int nb = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, kernel, w * 32, smem) != cudaSuccess) { cudaGetLastError(); continue; }
    if (nb * w > resident) { resident = nb * w; wpc = w; }
  }
}

// hand: nullptr, or the hand-over buffer of the context ([0] zeroed by the caller): the reachable-range variant (CIRC) is
// then used when it keeps at least a quarter more warps resident than whole spectra, followed by the full-size variant
// over the pixels it handed over.  *used_circ reports the choice.
template <int LPP, bool DUST, int DEG, int MODE = 0>
inline cudaError_t launch_transfer_series_t(const MarchConsts& mc, const float* coef, int64_t ncell, int npix, int nz,
                                            int nv, float* out, float* out_cont, cudaStream_t st, int* hand = nullptr,
                                            int* used_circ = nullptr) {
  constexpr int PPW = 32 / LPP;
  constexpr int NQ = SeriesLayout<DUST, DEG>::NQ;
  const int npts = MODE == 3 ? nv * mc.fine_m + 1 : nv;
  // whole rows of LPP channel pairs, plus one row: the last pass of a window runs all LPP lanes of the pixel, up to
  // LPP - 1 pairs past the window (their update is below the window threshold, or lands in this padding)
  const int nvp = (npts + 2 * LPP - 1) / (2 * LPP) * (2 * LPP) + 2 * LPP;
  const size_t rec_per_warp = (size_t)NQ * 32 * sizeof(float4);
  const size_t spec_per_warp = (size_t)PPW * nvp * sizeof(float);
  int wpc = 1, best = 0;
  series_residency(transfer_series_kernel<LPP, DUST, DEG, MODE, false>, rec_per_warp + spec_per_warp, wpc, best);
  if (best == 0) return cudaErrorInvalidConfiguration;
  const size_t smem = wpc * (rec_per_warp + spec_per_warp);
  const int ppc = wpc * PPW;
  const unsigned grid = (unsigned)((npix + ppc - 1) / ppc);
  cudaError_t e;
  if (used_circ) *used_circ = 0;
  if constexpr (MODE == 0) {
    if (hand != nullptr) {
      // circular buffers of rb rows: the largest power of two that is at most half the rows of a whole spectrum
      const int rows_full = nvp / (2 * LPP);
      int rb = 8;
      while (2 * rb * 2 <= rows_full) rb <<= 1;
      const size_t circ_per_warp = rec_per_warp + (size_t)PPW * rb * 2 * LPP * sizeof(float);
      int wpc_c = 1, best_c = 0;
      if (2 * rb <= rows_full) series_residency(transfer_series_kernel<LPP, DUST, DEG, 0, true>, circ_per_warp, wpc_c, best_c);
      if (4 * best_c >= 5 * best) {
        const size_t smem_c = wpc_c * circ_per_warp;
        const int ppc_c = wpc_c * PPW;
        if ((e = cudaFuncSetAttribute(transfer_series_kernel<LPP, DUST, DEG, 0, true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                      (int)smem_c)) != cudaSuccess) return e;
        transfer_series_kernel<LPP, DUST, DEG, 0, true><<<(unsigned)((npix + ppc_c - 1) / ppc_c), wpc_c * 32, smem_c, st>>>(
            mc, coef, ncell, npix, nz, nv, nvp, out, out_cont, rb - 1, hand, nullptr, nullptr);
        if ((e = cudaGetLastError()) != cudaSuccess) return e;
        if (used_circ) *used_circ = 1;
        // the pixels it handed over, with whole spectra (the warps beyond the list return at once)
        if ((e = cudaFuncSetAttribute(transfer_series_kernel<LPP, DUST, DEG, 0, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                      (int)smem)) != cudaSuccess) return e;
        transfer_series_kernel<LPP, DUST, DEG, 0, false><<<grid, wpc * 32, smem, st>>>(mc, coef, ncell, npix, nz, nv, nvp, out, out_cont, 0,
                                                                                     nullptr, hand + 2, hand);
        return cudaGetLastError();
      }
    }
  }
  e = cudaFuncSetAttribute(transfer_series_kernel<LPP, DUST, DEG, MODE, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  transfer_series_kernel<LPP, DUST, DEG, MODE, false><<<grid, wpc * 32, smem, st>>>(mc, coef, ncell, npix, nz, nv, nvp, out, out_cont, 0,
                                                                                 nullptr, nullptr, nullptr);
  return cudaGetLastError();
}

// s_max: upper bound of dv / b over all cells (dv / microturbulence); selects the polynomial degree.
// mode: 0 optically thick, 1 selectively thin, 2 optically thin (formal integration, channel-integrated profile), 3 optically
// thick on the fine velocity grid of mc.fine_m intervals per channel; modes 1 - 3 always run the dust instantiation
// (tau_d = S_d = 0 planes when the dust is off).  hand / used_circ: see launch_transfer_series_t (mode 0 only).
inline cudaError_t launch_transfer_series(const MarchConsts& mc, const float* coef, int64_t ncell, int npix, int nz, int nv,
                                          bool dust, float s_max, float* out, float* out_cont, cudaStream_t st, int mode = 0,
                                          int* hand = nullptr, int* used_circ = nullptr) {
  const bool deg3 = s_max <= kSeriesDeg3MaxS;
  if (mode == 1) return deg3 ? launch_transfer_series_t<8, true, 3, 1>(mc, coef, ncell, npix, nz, nv, out, out_cont, st)
                             : launch_transfer_series_t<8, true, 4, 1>(mc, coef, ncell, npix, nz, nv, out, out_cont, st);
  if (mode == 2) return deg3 ? launch_transfer_series_t<8, true, 3, 2>(mc, coef, ncell, npix, nz, nv, out, out_cont, st)
                             : launch_transfer_series_t<8, true, 4, 2>(mc, coef, ncell, npix, nz, nv, out, out_cont, st);
  if (mode == 3) return launch_transfer_series_t<8, true, 3, 3>(mc, coef, ncell, npix, nz, nv, out, out_cont, st);
  if (dust) return deg3 ? launch_transfer_series_t<8, true, 3>(mc, coef, ncell, npix, nz, nv, out, out_cont, st, hand, used_circ)
                        : launch_transfer_series_t<8, true, 4>(mc, coef, ncell, npix, nz, nv, out, out_cont, st, hand, used_circ);
  return deg3 ? launch_transfer_series_t<8, false, 3>(mc, coef, ncell, npix, nz, nv, out, out_cont, st, hand, used_circ)
              : launch_transfer_series_t<8, false, 4>(mc, coef, ncell, npix, nz, nv, out, out_cont, st, hand, used_circ);
}

}  // namespace iris
