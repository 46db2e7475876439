// K3 with the SMOOTH integrator (trapezoidal first step Eq. 4.8.12, BDF2 Eq. 4.8.10, ReLU of PAPER.md:709) in the
// optically thick and the selectively thin mode, as a LINE-WINDOW march: the windowed counterpart of
// transfer_modes_kernel<0 / 1, true, *>.
//
// Same difference form as transfer_modes.cuh (D = I^[T] - I^[C] next to the scalar continuum C):
//   n = 0     D_0 = 0
//   n = 1     D_1 = [(E_0 - A_0 C_0) + (E_1 - A_1 C_1) + (2 - a_0) D_0] / (2 + a_1)
//   n >= 2    D_n = [2 (E_n - A_n C_n) + 4 D_n-1 - D_n-2] / (3 + 2 a_n),     a_n = A_n + tau_d,n  (thick)
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
// PRODUCT of rho over those K cells.  With rho(tau_d) <= exp(1.6 tau_d) / 3 on [0, 0.25] the product stays below 1e-5
// (3^-12 = 1.9e-6 without dust) while the SUM of tau_d over the last 12 cells is <= ln(1e-5 3^12) / 1.6 = 1.04: the
// pixel is handed over when that sum is exceeded or a single cell has tau_d >= 0.25.
//
// Organisation (as in transfer_series.cuh): the march is cut into chunks of 16 cells.  In phase A the lane (pixel g,
// cell j) turns the six coefficients of ITS cell into a march record in shared memory, once: line window, hull of the
// windows of the last 12 cells (running halfword maxima over 2, 4, 8 cells with the previous chunk's registers), the
// tau_d criterion (a prefix sum), profile constants, and the continuum C_n and the dominant solution d_n, which are
// linear two-term recurrences along the ray and come out of ONE inclusive scan of 2 x 2 matrices + vectors over the 16
// lanes (a clamped continuum is a hand-over anyway).  In phase B the 16 lanes of a pixel walk the 16 cells, reading each
// record with broadcast LDS.128 and updating the points of its hull, two passes of 32 points staged together.  Cells 0
// and 1 (initial value, trapezoidal step) are done before the chunks.
//
// Selectively thin mode (MarchConsts::sel_thin, Eq. 4.8.13 - 4.8.15): a_n = tau_d, i.e. the same steps with the line
// opacity taken out of the two denominators; nothing else changes.  Its absorption saturates at I^[T] = 0 (the ReLU
// clamps D at -C_n) inside the hull, where every step is explicit.  A point that was clamped and then released carries
// a = (I_m - C_m) / d_m, and a d_n + C_n = I_m d_n / d_m + (C_n - C_m d_n / d_m) is the attenuated intensity plus what the
// dust has emitted since: not negative unless the recessive solution or rounding makes it so, which the far-point test
// catches per pixel (8 of the medium cube's 65536 pixels; with the per-CUBE gate of the first version every thick workload
// went to the dense kernel, which is why this mode used to stay there).
//
// Mapping as in transfer_window.cuh: LPP = 16 lanes per pixel, 2 pixels per warp, both spectra of a pixel in shared
// memory, point k at word (k / LPP) * 32 + g * LPP + k % LPP of its array.  Profile: the point value of Eq. 3.3.3 on
// the fine grid (fine_m intervals per channel, Simpson's rule over a channel in the epilogue, Eq. 4.5.1), or the
// channel integral from the channel centre (fine_m = 0; needs dv <= 0.55 b, see transfer_series.cuh).
#pragma once
#include <type_traits>
#include "transfer_common.cuh"
#include "transfer_window.cuh"
#include "transfer_series.cuh"       // packed f32x2 helpers

namespace iris {

constexpr int kSmoothLPP = 16;          // lanes per pixel
constexpr int kSmoothKeep = 12;         // cells a window stays active (K <= kSmoothLPP: lane i remembers cell n = i mod K)
constexpr float kSmoothMaxTau12 = 1.04f;       // largest sum of tau_d over the kept cells for which a released point's
                                               // recessive / dominant ratio stays below 1e-5 (see the header)

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

// Records of phase A (one per lane = (pixel g, cell j of the chunk)), field-major in shared memory: rec[f * 32 + lane]
//   f0 = { g2 = 2 (e_c - a_c C_n), a2 = 2 a_c, den0 = 3 + 2 tau_d, 1 / d_n }   (point profile: g2, a2 times its amplitude p0)
//   f1 = { 4 d_n-1, -d_n-2, relu_add, relu_min }
//   f2 = { xb = s sqrt(log2 e) per point, (1/2 - c_los) xb, bits(elo | ehi << 16) of the hull, d_n }
//   f3 = { p0, p1, p2, p3 }   profile polynomial (point profile: p0 only)
//   f4 = { p4, C_n before the ReLU, -, - }
constexpr int kSmoothRecFields = 5;

template <bool POINT>
__global__ void __launch_bounds__(128)
transfer_smooth_window_kernel(MarchConsts mc, const float* __restrict__ coef, int64_t ncell, int npix, int nz, int nv,
                              int nvp /* padded points per spectrum */, float* __restrict__ out,
                              float* __restrict__ out_cont, int* __restrict__ gate, int* __restrict__ gate_list) {
  extern __shared__ float sm[];
  constexpr unsigned FULL = 0xffffffffu;
  constexpr int LPP = kSmoothLPP, PPW = 32 / LPP, K = kSmoothKeep;
  constexpr float SQL2E = 1.2011224087864498f;              // sqrt(log2 e)
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, wpc = blockDim.x >> 5;
  const int g = lane / LPP, i = lane % LPP, gbase = g * LPP;
  const unsigned gmask = 0xffffu << gbase;
  const int pix_raw = (blockIdx.x * wpc + warp) * PPW + g;
  const bool valid = pix_raw < npix;
  const int pix = valid ? pix_raw : npix - 1;                   // idle groups shadow the last pixel and write nothing
  const int m = mc.fine_m;
  const float self_abs = mc.sel_thin ? 0.0f : 1.0f;   // selectively thin mode: a_n = tau_d, the line term drops out of
                                                      // the denominators of Eq. 4.8.10 / 4.8.12 and nothing else changes
  constexpr bool point = POINT;           // fine grid with the point profile (m > 0) or channel integrals (m = 0)
  const int npts = point ? nv * m + 1 : nv;
  const size_t arr = (size_t)nvp * PPW;
  const size_t warp_floats = 2 * arr + (size_t)kSmoothRecFields * 32 * 4;
  float* wbase = sm + (size_t)warp * warp_floats;
  float4* rec = reinterpret_cast<float4*>(wbase);                      // [kSmoothRecFields][32]
  float* specA = wbase + kSmoothRecFields * 32 * 4 + gbase;            // the two spectra of this pixel alternate roles
  float* specB = specA + arr;
#define IDX(k) (((k) / LPP) * 32 + ((k) % LPP))
  for (int k = i; k < nvp; k += LPP) { specA[IDX(k)] = 0.0f; specB[IDX(k)] = 0.0f; }
  __syncwarp();
  const float* lo_ok = wbase + kSmoothRecFields * 32 * 4;             // (checked build) region of this warp's spectra
  const float* hi_ok = lo_ok + 2 * arr;
  (void)lo_ok; (void)hi_ok;

  // position of a point in the units line_window works in (point k is the "channel" [k, k + 1) of width 1 / m whose
  // centre it is), and its spacing in Doppler widths
  const float fm = point ? (float)m : 1.0f, inv_fm = 1.0f / fm;
  float u_min = 0.0f;                       // most negative U this lane has stored
  bool risk = false;

  // ---- cells 0 and 1 (every lane of the pixel works them out): D_0 = 0, C_0 = T_bg; trapezoidal step to cell 1
  // (Eq. 4.8.12) over the windows of both cells.  U_1 = D_1 / d_1 with d_1 = d_0 = 1 goes to specB.
  const float* p = coef + pix;
  const float e_0 = p[0], a_0 = p[ncell], s_0 = p[3 * ncell] * inv_fm, td_0 = p[4 * ncell], Jd_0 = td_0 * p[5 * ncell];
  const float c_0 = point ? fmaf(p[2 * ncell], fm, 0.5f) : p[2 * ncell];
  int klo0, khi0;
  const unsigned word0 = line_window(e_0, a_0, c_0, s_0, npts, klo0, khi0) > 0 ? (((unsigned)khi0 << 16) | (0xffffu - (unsigned)klo0)) : 0u;
  float C_1 = mc.T_bg, td_1 = 0.0f;         // continuum at cell 1 (after the ReLU) and its dust depth
  unsigned word1 = 0u;
  if (nz > 1) {
    const float* p1 = p + npix;
    const float e_c = p1[0], a_c = p1[ncell], s_ch = p1[3 * ncell], td = p1[4 * ncell], Jd = td * p1[5 * ncell];
    const float c_los = point ? fmaf(p1[2 * ncell], fm, 0.5f) : p1[2 * ncell];
    const float s = s_ch * inv_fm;
    td_1 = td;
    int klo, khi;
    word1 = line_window(e_c, a_c, c_los, s, npts, klo, khi) > 0 ? (((unsigned)khi << 16) | (0xffffu - (unsigned)klo)) : 0u;
    const unsigned un = __vmaxu2(word0, word1);
    const int elo = 0xffff - (int)(un & 0xffffu), ehi = (int)(un >> 16);
    const float C_unc = (Jd_0 + Jd + (2.0f - td_0) * mc.T_bg) * rcp_approx(2.0f + td);
    C_1 = fmaxf(C_unc, 0.0f);
    const float relu_add = C_unc >= 0.0f ? 0.0f : C_unc, relu_min = C_unc >= 0.0f ? -C_unc : 0.0f;
    if (C_unc < 0.0f) risk = true;
    if (ehi >= elo) {
      SmoothProfile<POINT> prof, prof0;
      prof.set(s_ch);
      prof0.set(s_0 * fm);
      const float xstep = (float)LPP * s * SQL2E;
      float xs = ((float)(elo + i) + 0.5f - c_los) * (s * SQL2E);
      for (int k = elo + i; k <= ehi; k += LPP, xs += xstep) {
        const float pw = prof.at(xs);
        const float pw0 = prof0.at(((float)k + 0.5f - c_0) * (s_0 * SQL2E));
        const float E = e_c * pw, A = a_c * pw, E0 = e_0 * pw0, A0 = a_0 * pw0;
        const float Du = ((E0 - A0 * mc.T_bg) + (E - A * C_unc)) * rcp_approx(fmaf(self_abs, A, 2.0f + td));
        const float U = fmaxf(Du + relu_add, relu_min);                  // ReLU on D + C and on C; d_1 = 1
        IRIS_CHECK_SMEM(specB + IDX(k), 4, lo_ok, hi_ok);
        specB[IDX(k)] = U;
        u_min = fminf(u_min, U);
      }
    }
    __syncwarp();
  }

  // ---- cells 2 .. nz - 1 in chunks of LPP cells: phase A makes one record per (pixel, cell), phase B walks them
  // running state of the scans: continuum and dominant solution at the last two cells before the chunk
  float C_a = C_1, C_b = mc.T_bg;           // C at n0 - 1 and n0 - 2
  float d_a = 1.0f, d_b = 1.0f;             // d at n0 - 1 and n0 - 2
  // history of the previous chunk, lane i <-> cell n0 - LPP + i: window words (and their running maxima over 2 and 4
  // cells) for the hull of the last K cells, inclusive prefix sums of tau_d for the release criterion
  unsigned pv = i == LPP - 2 ? word0 : (i == LPP - 1 ? word1 : 0u);
  unsigned pm2, pm4;
  {
    const unsigned t1 = __shfl_up_sync(FULL, pv, 1);
    pm2 = __vmaxu2(pv, i >= 1 ? t1 : 0u);
    const unsigned t2 = __shfl_up_sync(FULL, pm2, 2);
    pm4 = __vmaxu2(pm2, i >= 2 ? t2 : 0u);
  }
  float pT = i == LPP - 2 ? td_0 : (i == LPP - 1 ? td_0 + td_1 : 0.0f);      // prefix of tau_d up to cell n0 - LPP + i
  float T_run = td_0 + td_1;
  float* cur = specB;                       // U_n-1 when cell n is entered
  float* prv = specA;                       // V = U_n-2; receives U_n
  float C_fin = C_1, d_fin = 1.0f;          // continuum and dominant solution at the last cell of the column

  const float* pc = coef + pix + (int64_t)(2 + i) * npix;
  float l_e = 0.0f, l_a = 0.0f, l_c = 0.0f, l_s = 1.0f, l_td = 0.0f, l_sd = 0.0f;
  if (2 + i < nz) { l_e = pc[0]; l_a = pc[ncell]; l_c = pc[2 * ncell]; l_s = pc[3 * ncell]; l_td = pc[4 * ncell]; l_sd = pc[5 * ncell]; }
  for (int n0 = 2; n0 < nz; n0 += LPP) {
    const int n = n0 + i;
    const bool mine = n < nz;
    // ---- phase A: this lane's cell
    const float e_c = l_e, a_c = l_a, s_ch = l_s, td = mine ? l_td : 0.0f, Jd = td * l_sd;
    const float c_los = point ? fmaf(l_c, fm, 0.5f) : l_c;      // in point units
    const float s = s_ch * inv_fm;                              // Doppler widths per point
    {
      const int zn = n + LPP;
      l_e = 0.0f; l_a = 0.0f; l_td = 0.0f;
      if (zn < nz) {
        pc += (int64_t)LPP * npix;
        l_e = pc[0]; l_a = pc[ncell]; l_c = pc[2 * ncell]; l_s = pc[3 * ncell]; l_td = pc[4 * ncell]; l_sd = pc[5 * ncell];
      }
    }
    int klo, khi;
    const unsigned v = (mine && line_window(e_c, a_c, c_los, s, npts, klo, khi) > 0)
                           ? (((unsigned)khi << 16) | (0xffffu - (unsigned)klo)) : 0u;
    // hull of the windows of cells n - K + 1 .. n (K = 12 = 8 + 4): running halfword maxima over 2, 4, 8 cells, the
    // cells before the chunk taken from the previous chunk's registers (lane i - k + LPP of pv / pm2 / pm4)
    auto back = [&](unsigned cur_v, unsigned prev_v, int k) {
      const unsigned a = __shfl_sync(FULL, cur_v, gbase + ((i - k) & (LPP - 1)));
      const unsigned b = __shfl_sync(FULL, prev_v, gbase + ((i - k) & (LPP - 1)));
      return i >= k ? a : b;
    };
    const unsigned m2 = __vmaxu2(v, back(v, pv, 1));
    const unsigned m4 = __vmaxu2(m2, back(m2, pm2, 2));
    const unsigned m8 = __vmaxu2(m4, back(m4, pm4, 4));
    const unsigned hull = __vmaxu2(m8, back(m4, pm4, 8));
    static_assert(K == 12, "the hull is built from running maxima over 8 + 4 cells");
    pv = v; pm2 = m2; pm4 = m4;
    // release criterion (header): a point the windows have left is a d_n only while the recessive solution has died,
    // rho(tau_d) <= exp(1.6 tau_d) / 3 for tau_d <= 0.25, so 3^-12 exp(1.6 sum of tau_d over the last 12 cells) <= 1e-5
    float Tp = td;
#pragma unroll
    for (int o = 1; o < LPP; o <<= 1) {
      const float t = __shfl_up_sync(FULL, Tp, o);
      if (i >= o) Tp += t;
    }
    Tp += T_run;
    {
      const float a = __shfl_sync(FULL, Tp, gbase + ((i - K) & (LPP - 1))), b = __shfl_sync(FULL, pT, gbase + ((i - K) & (LPP - 1)));
      const float before = i >= K ? a : b;
      if (mine && (td >= 0.25f || Tp - before > kSmoothMaxTau12)) risk = true;
    }
    pT = Tp;
    T_run = __shfl_sync(FULL, Tp, gbase + LPP - 1);
    // continuum and dominant solution: y_n = alpha y_n-1 + beta y_n-2 + gamma with alpha = 4 r, beta = -r, gamma = 2 J_d r,
    // r = 1 / (3 + 2 tau_d) (Eq. 4.8.10 without a line; the dominant solution has gamma = 0).  Inclusive scan over the
    // cells of the chunk of the maps (y_n-1, y_n-2) -> (y_n, y_n-1): matrix M (2 x 2) and vector w.
    const float r = rcp_approx(fmaf(2.0f, td, 3.0f));
    float m11 = mine ? 4.0f * r : 1.0f, m12 = mine ? -r : 0.0f, m21 = mine ? 1.0f : 0.0f, m22 = mine ? 0.0f : 1.0f;
    float w1 = mine ? 2.0f * Jd * r : 0.0f, w2 = 0.0f;
#pragma unroll
    for (int o = 1; o < LPP; o <<= 1) {
      // the map of the o cells before: applied first
      float q11 = __shfl_up_sync(FULL, m11, o), q12 = __shfl_up_sync(FULL, m12, o), q21 = __shfl_up_sync(FULL, m21, o),
            q22 = __shfl_up_sync(FULL, m22, o), z1 = __shfl_up_sync(FULL, w1, o), z2 = __shfl_up_sync(FULL, w2, o);
      if (i >= o) {
        const float n11 = fmaf(m11, q11, m12 * q21), n12 = fmaf(m11, q12, m12 * q22);
        const float n21 = fmaf(m21, q11, m22 * q21), n22 = fmaf(m21, q12, m22 * q22);
        const float nw1 = fmaf(m11, z1, fmaf(m12, z2, w1)), nw2 = fmaf(m21, z1, fmaf(m22, z2, w2));
        m11 = n11; m12 = n12; m21 = n21; m22 = n22; w1 = nw1; w2 = nw2;
      }
    }
    const float C_unc = fmaf(m11, C_a, fmaf(m12, C_b, w1));               // continuum at this cell before the ReLU
    const float d_n = fmaf(m11, d_a, m12 * d_b), d_n1 = fmaf(m21, d_a, m22 * d_b);     // d at n and n - 1
    float d_n2 = __shfl_up_sync(FULL, d_n1, 1);                             // d at n - 2
    if (i == 0) d_n2 = d_b;
    // what a window cannot see (header): the continuum clamped, the dominant solution losing its sign
    if (mine && (C_unc < 0.0f || !(d_n > 1.0e-6f * d_n1))) risk = true;
    {
      // the state after the chunk, from its last cell (cells beyond the column carry identity maps)
      const int last = gbase + LPP - 1;
      const float Cl = __shfl_sync(FULL, C_unc, last), Cl1 = __shfl_sync(FULL, fmaf(m21, C_a, fmaf(m22, C_b, w2)), last);
      const float dl = __shfl_sync(FULL, d_n, last), dl1 = __shfl_sync(FULL, d_n1, last);
      // (the column's last cell, for the epilogue)
      const int fin = gbase + min(LPP - 1, nz - 1 - n0);
      C_fin = fmaxf(__shfl_sync(FULL, C_unc, fin), 0.0f);
      d_fin = __shfl_sync(FULL, d_n, fin);
      C_a = fmaxf(Cl, 0.0f); C_b = fmaxf(Cl1, 0.0f); d_a = dl; d_b = dl1;
    }
    // record
    {
      SmoothProfile<POINT> prof;
      prof.set(s_ch);
      const float xb = s * SQL2E;
      const int elo = 0xffff - (int)(hull & 0xffffu), ehi = (int)(hull >> 16);
      const bool any = mine && ehi >= elo;
      // (point profile: its constant amplitude p0 is folded into the two line coefficients here, once per cell)
      const float amp2 = POINT ? 2.0f * prof.p0 : 2.0f;
      rec[lane] = make_float4(amp2 * fmaf(-a_c, C_unc, e_c), amp2 * self_abs * a_c, fmaf(2.0f, td, 3.0f), rcp_approx(d_n));
      rec[32 + lane] = make_float4(4.0f * d_n1, -d_n2, C_unc >= 0.0f ? 0.0f : C_unc, C_unc >= 0.0f ? -C_unc : 0.0f);
      rec[64 + lane] = make_float4(xb, (0.5f - c_los) * xb, __int_as_float(any ? (elo | (ehi << 16)) : 0x0000ffff), d_n);
      rec[96 + lane] = make_float4(prof.p0, prof.p1, prof.p2, prof.p3);
      rec[128 + lane] = make_float4(prof.p4, C_unc, 0.0f, 0.0f);
    }
    __syncwarp();
    // ---- phase B: the LPP lanes of a pixel walk the cells of the chunk
    const int ncz = min(LPP, nz - n0);
    for (int j = 0; j < ncz; ++j) {
      const int rl = gbase + j;
      const float4 r0 = rec[rl], r1 = rec[32 + rl], r2 = rec[64 + rl], r3 = rec[96 + rl], r4 = rec[128 + rl];
      const int hw = __float_as_int(r2.z);
      const int elo = hw & 0xffff, ehi = (int)((unsigned)hw >> 16);
      // a ReLU that would fire on a far point a d_n + C_n < 0 (header)
      if (fmaf(u_min, r2.w, r4.y) < 0.0f) risk = true;
      if (ehi >= elo) {
        // BDF2: D_n = [2 p (e_c - a_c C_n) + 4 U d_n-1 - V d_n-2] / (3 + 2 tau_d + 2 a_c p), on even-aligned PAIRS of
        // points with packed arithmetic (fma / mul / add.rn.f32x2): a lane takes points k, k + 1, the LPP lanes of a
        // pixel 2 LPP consecutive points (two rows of its spectra) per pass.  A pair may reach one point beyond the
        // hull on either side; the step is as valid there.
        const f32x2 g2 = pk1(r0.x), a2 = pk1(r0.y), den0 = pk1(r0.z), idn = pk1(r0.w);
        const f32x2 c4 = pk1(r1.x), cm = pk1(r1.y), radd = pk1(r1.z);
        const float relu_min = r1.w;
        const f32x2 pp0 = pk1(r3.x), pp1 = pk1(r3.y), pp2 = pk1(r3.z), pp3 = pk1(r3.w), pp4 = pk1(r4.x);
        const int k0 = (elo & ~1) + 2 * i;
        const float xb = r2.x, xa = fmaf((float)k0, xb, r2.y);
        f32x2 xx = pk(xa, xa + xb);
        const f32x2 xstep2 = pk1(2.0f * (float)LPP * xb);
        // NP passes of a lane written stage by stage (loads, profile, step, stores): the passes are independent, but
        // the compiler cannot move a load of the next pass above a store of this one, and a pass alone is one
        // dependent chain LDS -> MUFU -> FMA -> MUFU -> STS that the few resident warps do not cover
        int wk = IDX(k0);                            // word of the lane's pair in the pass at hand
        auto passes = [&](auto np_tag, int) {
          constexpr int NP = decltype(np_tag)::value;
          f32x2 Uv[NP], Vv[NP], pw[NP];
#pragma unroll
          for (int q = 0; q < NP; ++q) {
            const int w = wk + 64 * q;               // = IDX(k + 2 LPP q): a pass is two rows of the pixel further
            IRIS_CHECK_SMEM(cur + w, 8, lo_ok, hi_ok);
            IRIS_CHECK_SMEM(prv + w, 8, lo_ok, hi_ok);
            const float2 Uo = *reinterpret_cast<const float2*>(cur + w), Vo = *reinterpret_cast<const float2*>(prv + w);
            Uv[q] = pk(Uo.x, Uo.y); Vv[q] = pk(Vo.x, Vo.y);
            const f32x2 u = mul2(xx, xx);
            xx = add2(xx, xstep2);
            float u0, u1;
            upk(u, u0, u1);
            pw[q] = pk(ex2_approx(-u0), ex2_approx(-u1));
            if (!POINT) pw[q] = mul2(pw[q], fma2(fma2(fma2(fma2(pp4, u, pp3), u, pp2), u, pp1), u, pp0));
          }
#pragma unroll
          for (int q = 0; q < NP; ++q) {
            const f32x2 lin = fma2(Uv[q], c4, mul2(Vv[q], cm));
            const f32x2 den = fma2(pw[q], a2, den0);
            float e0, e1;
            upk(den, e0, e1);
            const f32x2 Du = add2(mul2(fma2(pw[q], g2, lin), pk(rcp_approx(e0), rcp_approx(e1))), radd);
            float D0, D1;
            upk(Du, D0, D1);
            Uv[q] = mul2(pk(fmaxf(D0, relu_min), fmaxf(D1, relu_min)), idn);          // ReLU on D + C and on C
          }
#pragma unroll
          for (int q = 0; q < NP; ++q) {
            float2 Un;
            upk(Uv[q], Un.x, Un.y);
            // (a pair may end on the padding point npts of the last row: it gets the value the step gives there, nobody
            // reads it as a point, and through u_min it can only make the hand-over test more careful)
            *reinterpret_cast<float2*>(prv + wk + 64 * q) = Un;
            u_min = fminf(u_min, fminf(Un.x, Un.y));
          }
          wk += 64 * NP;
        };
        int k = k0;
        for (; k + 2 * LPP <= ehi; k += 4 * LPP) passes(std::integral_constant<int, 2>{}, k);
        if (k <= ehi) passes(std::integral_constant<int, 1>{}, k);
      }
      __syncwarp();
      { float* t = cur; cur = prv; prv = t; }      // what was written is now "n - 1"
    }
    // keep the dominant solution inside the fp32 range (dust attenuates it like exp(-tau_d)); rare
    if (d_a < 1.0e-12f) {
      const float f = d_a;
      for (int k = i; k < nvp; k += LPP) { cur[IDX(k)] *= f; prv[IDX(k)] *= f; }
      u_min *= f;
      d_b /= f; d_a = 1.0f; d_fin /= f;
    }
    __syncwarp();
  }
  __syncwarp();
  // hand the pixel over: gate[0] = pixels listed by this launch, gate[1] = pixels handed over since the public call began
  const bool group_risk = (__ballot_sync(FULL, risk && valid) & gmask) != 0u;
  if (group_risk && i == 0) { gate_list[atomicAdd(gate, 1)] = pix; atomicAdd(gate + 1, 1); }

  if (valid) {
    // the points are D = U d; nz = 1 leaves D = 0
    const float dfin = nz > 1 ? d_fin : 0.0f;
    const float C = C_fin;
    if (out != nullptr && mc.out_mode <= OUT_I_TOT) {
      // the units that are linear in D: one multiply-add per channel, four channels per lane in flight (the loop is a
      // chain LDS -> FMA -> STG; see the epilogue of transfer_series_kernel)
      const float sc = mc.out_mode >= OUT_I_SUB ? mc.inv_KRJ : 1.0f;
      const float cadd = (mc.out_mode & 1) ? C : 0.0f;      // total = (D + C) sc is exactly 0 where the ReLU holds D at -C
      float* o = out + (int64_t)pix * nv;
      // (the ReLU keeps I_T = D + C >= 0 at every step; D = U d_fin can come out one rounding below -C: clamp)
      if (point) {
        const float a = dfin / (3.0f * (float)m);
        auto channel = [&](int c) {
          float acc = 0.0f;
          for (int j = 0; j < m; j += 2) acc += cur[IDX(c * m + j)] + 4.0f * cur[IDX(c * m + j + 1)] + cur[IDX(c * m + j + 2)];
          return acc;
        };
        int c = i;
        for (; c + 3 * LPP < nv; c += 4 * LPP) {
          float v[4];
#pragma unroll
          for (int k = 0; k < 4; ++k) v[k] = channel(c + k * LPP);
#pragma unroll
          for (int k = 0; k < 4; ++k) o[c + k * LPP] = (fmaxf(v[k] * a, -C) + cadd) * sc;
        }
        for (; c < nv; c += LPP) o[c] = (fmaxf(channel(c) * a, -C) + cadd) * sc;
      } else {
        const float a = dfin;
        int c = i;
        for (; c + 3 * LPP < nv; c += 4 * LPP) {
          float v[4];
#pragma unroll
          for (int k = 0; k < 4; ++k) v[k] = cur[IDX(c + k * LPP)];
#pragma unroll
          for (int k = 0; k < 4; ++k) o[c + k * LPP] = (fmaxf(v[k] * a, -C) + cadd) * sc;
        }
        for (; c < nv; c += LPP) o[c] = (fmaxf(cur[IDX(c)] * a, -C) + cadd) * sc;
      }
    } else if (out != nullptr) {
      if (point) {
        const float wgt = dfin / (3.0f * (float)m);
        for (int c = i; c < nv; c += LPP) {
          float acc = 0.0f;
          for (int j = 0; j < m; j += 2) acc += cur[IDX(c * m + j)] + 4.0f * cur[IDX(c * m + j + 1)] + cur[IDX(c * m + j + 2)];
          out[(int64_t)pix * nv + c] = convert_out(fmaxf(acc * wgt, -C), C, mc);
        }
      } else {
        for (int c = i; c < nv; c += LPP) out[(int64_t)pix * nv + c] = convert_out(fmaxf(cur[IDX(c)] * dfin, -C), C, mc);
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
  return (size_t)2 * (32 / kSmoothLPP) * nvp * sizeof(float) + (size_t)5 * 32 * sizeof(float4);      // spectra + march records
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
