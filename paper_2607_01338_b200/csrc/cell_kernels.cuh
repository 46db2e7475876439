// K1 (level populations) and K2 (per-cell transfer coefficients), one thread per cell.
//
// K1 solves the statistical equilibrium of Eq. 3.6.1 with the rates of
// Eq. 3.6.2-3.6.3 and 3.7.1-3.7.2 for the level FRACTIONS x_i.  The system is the stationary
// distribution of a continuous-time Markov chain on the levels; it is solved in registers by the
// subtraction-free Grassmann-Taksar-Heyman state elimination, which carries component-wise relative
// accuracy over the ~30 decades the populations span (partial-pivot GE in fp32 does not guarantee it).
//
// K2 turns (x_u, x_l, n_H2, T_gas, T_dust, v_los) into the six scaled per-cell coefficients the march
// consumes (Eq. 3.3.1-3.3.4, 3.2.1-3.2.2, 4.6.3-4.6.4 folded with the step h and the unit conversion):
//   e_c   = K_RJ (h nu0 / 4 pi) X n x_u A_ul h / (2 dnu_W)            [K per unit erf-difference]
//   a_c   =      (h nu0 / 4 pi) X n (x_l B_lu - x_u B_ul) h / (2 dnu_W)  [optical depth per unit erf-difference]
//   c_los = (v_los - v0) / dv + 1/2     line centre in channel-edge index units (edge k <-> index k)
//   s     = dv / b,  b = sqrt(2 k T / m_a + xi^2)                     [Doppler widths per channel]
//   tau_d = kappa rho_gas h                                            [dust optical depth of the cell]
//   S_d   = K_RJ B_nu0(T_dust) = (h nu0 / k) / (exp(h nu0 / k T_dust) - 1)   [K]
// so that for channel k:  tau_L = a_c * dErf_k,  J_L = e_c * dErf_k,  dErf_k = erf((k+1-c_los) s) - erf((k-c_los) s).
// Intensities are carried as Rayleigh-Jeans-equivalent Kelvin (I * c^2 / (2 k nu0^2)): CGS intensities
// (~1e-15) times path lengths (~1e18) would otherwise leave the fp32 range (PAPER.md:268 warns of this).
#pragma once
#include "iris_math.cuh"

namespace iris {

constexpr int kMaxLevels = 10;
constexpr int kMaxPairs = kMaxLevels * (kMaxLevels - 1) / 2;

// Bandwidth (largest |i - j| with a non-zero rate) up to which the banded elimination is instantiated.
constexpr int kBandNarrow = 2;

// pair index of (u > l)
__host__ __device__ constexpr int pair_index(int u, int l) { return u * (u - 1) / 2 + l; }

// Tabulated collision rates (several partners folded on the host: K_ul(T) = sum_p f_p K^p_ul(T)),
// interpolated linearly in temperature and held constant outside the grid.  Device arrays owned by the context:
// T[nT] ascending, K[nT][kMaxPairs] = { K_ul, K_ul g_u / g_l } (both times LevelConsts::rate_scale).
struct CollTable {
  const float* T;
  const float2* K;
  int nT;
};

struct LevelConsts {
  float ndE2[kMaxLevels];       // -(E_i - E_{i-1}) / k * log2(e)  [K], i >= 1: Boltzmann factor = 2^(ndE2 / T)
  // per pair (u > l), packed so that one 16-byte constant load feeds both rate FMAs:
  //   x = K_ul(T_ref), y = A_ul + B_ul J_ul = A_ul (1 + n_gamma), z = K_ul(T_ref) g_u / g_l, w = B_lu J_ul
  float4 pr[kMaxPairs];
  float inv_Tref, Texp;
  float rate_scale;             // every rate above has been multiplied by this (1 / largest Einstein A)
  CollTable tb;                 // tb.K == nullptr: the power law K_ul(T_ref) (T / T_ref)^Texp of pr[].x / pr[].z
};

// interval t0 and weight w of temperature T: K = K[t0] + w (K[t0 + 1] - K[t0])
__device__ __forceinline__ void locate_temperature(const CollTable& tb, float T, int& t0, float& w) {
  if (tb.nT < 2) { t0 = 0; w = 0.0f; return; }
  int lo = 0, hi = tb.nT - 1;              // invariant: T[lo] <= T < T[hi] once T is inside the grid
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (T >= tb.T[mid]) lo = mid; else hi = mid;
  }
  t0 = lo;
  const float a = tb.T[lo], b = tb.T[lo + 1];
  w = fminf(fmaxf((T - a) / (b - a), 0.0f), 1.0f);
}

// Boltzmann factors of adjacent levels, q[i] = exp(-(E_i - E_{i-1}) / T), i >= 1: one MUFU.EX2 each.  The product
// ndE2 / T is formed with its rounding error (FMA residual) and the error is applied to first order, so the factor
// keeps ~2 ulp even where |ndE2 / T| ~ 15 (T = 5 K), where the rounding of the argument alone would cost 1e-6.
template <int N>
__device__ __forceinline__ void boltzmann_adjacent(const LevelConsts& lc, float T, float (&q)[N]) {
  const float invT = 1.0f / T;
#pragma unroll
  for (int i = 1; i < N; ++i) {
    const float t = lc.ndE2[i] * invT;
    const float r = fmaf(lc.ndE2[i], invT, -t);
    const float e = ex2_approx(t);
    q[i] = fmaf(e * 0.6931471805599453f, r, e);
  }
}

struct CoefConsts {
  int upper, lower;
  float gr;          // g_u / g_l of the line
  float c_e, c_a;    // e_c = c_e n x_u ; a_c = c_a n (x_l gr - x_u)
  float c_d;         // tau_d = c_d n  (0 if dust off)
  float hnu_k;       // h nu0 / k  [K]
  float c_b, xi2;    // b^2 = c_b T + xi2  [(cm/s)^2]
  float dv, inv_dv, v0;
  float T_inf;
  int dust_on;
  float pick_upper[kMaxLevels], pick_lower[kMaxLevels];   // one-hot vectors of the line's levels
};

// Level fractions of one cell.  N is a template parameter so that the rate matrix lives in registers.
// BW is the bandwidth of the rate matrix: rates i -> j with |i - j| > BW are zero (the host checks this against
// the molecule, iris_so_create).  State elimination of the highest state m only couples the states m-BW..m-1
// among themselves, so the band is preserved and the elimination costs O(N BW^2) instead of O(N^3); BW = N-1 is
// the dense case.  The rigid-rotor workloads (radiative dJ = 1, collisional dJ <= 2) have BW = 2.
// The fractions do not change when every rate is multiplied by one constant; the host divides all rates by the
// largest Einstein A (LevelConsts::rate_scale), which keeps the pivots far from the fp32 denormal range so that
// the reciprocals can be MUFU.RCP (1 ulp, flush-to-zero).
template <int N, int BW, bool TABLE = false>
__device__ __forceinline__ void level_fractions(const LevelConsts& lc, float n, float T, float (&x)[N],
                                                float* inv_tot = nullptr) {
  const CollTable* tb = &lc.tb;
  float R[N][N];   // R[i][j]: rate i -> j (i != j); only |i - j| <= BW is touched
  // power law: n * (T / T_ref)^p times K_ul(T_ref); table: n times the interpolated K_ul(T)
  float kf = n, wt = 0.0f;
  int t0 = 0;
  if (TABLE) locate_temperature(*tb, T, t0, wt);
  else kf = n * pow_approx(T * lc.inv_Tref, lc.Texp);
  float q[N];      // Boltzmann factors of adjacent levels, exp(-(E_i - E_{i-1}) / T)
  boltzmann_adjacent<N>(lc, T, q);
#pragma unroll
  for (int u = 1; u < N; ++u) {
    float bz = 1.0f;
#pragma unroll
    for (int l = u - 1; l >= 0; --l) {
      if (u - l > BW) continue;
      bz *= q[l + 1];                                   // exp(-(E_u - E_l) / T), Eq. 3.7.2
      const float4 pr = lc.pr[pair_index(u, l)];
      float Kd = pr.x, Kg = pr.z;
      if (TABLE) {
        const float2 k0 = tb->K[t0 * kMaxPairs + pair_index(u, l)];
        const float2 k1 = tb->K[min(t0 + 1, tb->nT - 1) * kMaxPairs + pair_index(u, l)];
        Kd = fmaf(wt, k1.x - k0.x, k0.x);
        Kg = fmaf(wt, k1.y - k0.y, k0.y);
      }
      R[u][l] = fmaf(kf, Kd, pr.y);
      R[l][u] = fmaf(kf * bz, Kg, pr.w);
    }
  }
  // GTH elimination of states N-1 .. 1
#pragma unroll
  for (int m = N - 1; m >= 1; --m) {
    const int lo = m - BW > 0 ? m - BW : 0;
    float s = 0.0f;
#pragma unroll
    for (int j = 0; j < m; ++j)
      if (j >= lo) s += R[m][j];
    const float inv = rcp_approx(s);
#pragma unroll
    for (int i = 0; i < m; ++i)
      if (i >= lo) R[i][m] *= inv;
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
  const float inv = rcp_approx(tot);
  if (inv_tot != nullptr) { *inv_tot = inv; return; }      // caller scales the levels it needs
#pragma unroll
  for (int j = 0; j < N; ++j) x[j] *= inv;
}

// Six coefficient planes of one cell from its line-level fractions.
__device__ __forceinline__ void cell_coefficients(const CoefConsts& cc, float n, float T, float Td, float vlos,
                                                  float xu, float xl, float (&o)[6]) {
  float e = cc.c_e * n * xu;
  float a = cc.c_a * n * fmaf(xl, cc.gr, -xu);
  if (T > cc.T_inf) { e = 0.0f; a = 0.0f; }
  o[0] = e;
  o[1] = a;
  o[2] = fmaf(vlos - cc.v0, cc.inv_dv, 0.5f);
  o[3] = cc.dv * rsqrtf(fmaf(cc.c_b, T, cc.xi2));
  o[4] = cc.c_d * n;
  o[5] = cc.dust_on ? cc.hnu_k * rcp_approx(expm1_pos(cc.hnu_k * rcp_approx(Td))) : 0.0f;
}

// K1: pop[N][ncell]
template <int N, int BW, bool TABLE>
__global__ void __launch_bounds__(128) levelpop_kernel(LevelConsts lc, int64_t ncell, const float* __restrict__ nH2,
                                                       const float* __restrict__ Tgas, float* __restrict__ pop) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= ncell) return;
  float x[N];
  level_fractions<N, BW, TABLE>(lc, nH2[i], Tgas[i], x);
#pragma unroll
  for (int l = 0; l < N; ++l) pop[(int64_t)l * ncell + i] = x[l];
}

// K1 + K2 fused: coef[6][ncell]; populations never leave registers.
template <int N, int BW, bool TABLE>
__global__ void __launch_bounds__(128) cellcoef_kernel(LevelConsts lc, CoefConsts cc, int64_t ncell,
                                                       const float* __restrict__ nH2, const float* __restrict__ Tgas,
                                                       const float* __restrict__ Tdust, const float* __restrict__ vlos,
                                                       float* __restrict__ coef) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= ncell) return;
  const float n = nH2[i], T = Tgas[i];
  float x[N], inv;
  level_fractions<N, BW, TABLE>(lc, n, T, x, &inv);      // unnormalised fractions and 1 / their sum
  // the two levels of the line, picked with one-hot constant vectors (static indexing keeps x[] in registers; a
  // dot product with constant operands is half the instructions of N compare-select pairs)
  float xu = 0.0f, xl = 0.0f;
#pragma unroll
  for (int l = 0; l < N; ++l) {
    xu = fmaf(x[l], cc.pick_upper[l], xu);
    xl = fmaf(x[l], cc.pick_lower[l], xl);
  }
  xu *= inv; xl *= inv;
  float o[6];
  cell_coefficients(cc, n, T, Tdust[i], vlos[i], xu, xl, o);
#pragma unroll
  for (int q = 0; q < 6; ++q) coef[(int64_t)q * ncell + i] = o[q];
}

// ---- K1 + K2 for TWO cells per thread (cells 2 t and 2 t + 1) with packed fp32 arithmetic ------------------------------
// cellcoef_kernel is bound by instruction issue (86 % of the issue slots, FMA pipe half idle), and 60 % of its
// instructions are scalar FFMA / FMUL / FADD of the rate matrix, the elimination and the back substitution.  Here both
// cells of a thread go through those steps in the two halves of f32x2 registers (fma / mul / add.rn.f32x2: one issue slot
// for two cells); the operations and their order are those of level_fractions / cell_coefficients, element by element, so
// the results are bit-identical.  MUFU operations (reciprocals, the power law, exp(x) - 1, rsqrt) stay scalar.  The fields
// are read and the planes written as 8-byte accesses.  Power-law collision rates only (TABLE variants keep the scalar kernel).
template <int N, int BW>
__device__ __forceinline__ void level_fractions2(const LevelConsts& lc, float n0, float n1, float T0, float T1, f32x2 (&x)[N],
                                                 f32x2& inv_tot) {
  f32x2 R[N][N];
  const f32x2 kf = pk(n0 * pow_approx(T0 * lc.inv_Tref, lc.Texp), n1 * pow_approx(T1 * lc.inv_Tref, lc.Texp));
  f32x2 q[N];
  {
    const float i0 = 1.0f / T0, i1 = 1.0f / T1;
    const f32x2 invT = pk(i0, i1), ninvT = pk(-i0, -i1);
#pragma unroll
    for (int i = 1; i < N; ++i) {
      const f32x2 c = pk1(lc.ndE2[i]);
      const f32x2 nt = mul2(c, ninvT);                    // -t exactly (there is no packed negation)
      const f32x2 r = fma2(c, invT, nt);
      float ta, tb;
      upk(nt, ta, tb);
      const f32x2 e = pk(ex2_approx(-ta), ex2_approx(-tb));
      q[i] = fma2(mul2(e, pk1(0.6931471805599453f)), r, e);
    }
  }
#pragma unroll
  for (int u = 1; u < N; ++u) {
    f32x2 bz = pk1(1.0f);
#pragma unroll
    for (int l = u - 1; l >= 0; --l) {
      if (u - l > BW) continue;
      bz = mul2(bz, q[l + 1]);
      const float4 pr = lc.pr[pair_index(u, l)];
      R[u][l] = fma2(kf, pk1(pr.x), pk1(pr.y));
      R[l][u] = fma2(mul2(kf, bz), pk1(pr.z), pk1(pr.w));
    }
  }
#pragma unroll
  for (int m = N - 1; m >= 1; --m) {
    const int lo = m - BW > 0 ? m - BW : 0;
    f32x2 sum = pk1(0.0f);
#pragma unroll
    for (int j = 0; j < m; ++j)
      if (j >= lo) sum = add2(sum, R[m][j]);
    float sa, sb;
    upk(sum, sa, sb);
    const f32x2 inv = pk(rcp_approx(sa), rcp_approx(sb));
#pragma unroll
    for (int i = 0; i < m; ++i)
      if (i >= lo) R[i][m] = mul2(R[i][m], inv);
#pragma unroll
    for (int i = 0; i < m; ++i)
#pragma unroll
      for (int j = 0; j < m; ++j)
        if (i != j && i >= lo && j >= lo) R[i][j] = fma2(R[i][m], R[m][j], R[i][j]);
  }
  x[0] = pk1(1.0f);
  f32x2 tot = pk1(1.0f);
#pragma unroll
  for (int j = 1; j < N; ++j) {
    f32x2 sum = pk1(0.0f);
#pragma unroll
    for (int i = 0; i < j; ++i)
      if (j - i <= BW) sum = fma2(x[i], R[i][j], sum);
    x[j] = sum;
    tot = add2(tot, sum);
  }
  float ta, tb;
  upk(tot, ta, tb);
  inv_tot = pk(rcp_approx(ta), rcp_approx(tb));
}

template <int N, int BW>
__global__ void __launch_bounds__(128) cellcoef2_kernel(LevelConsts lc, CoefConsts cc, int64_t ncell,
                                                        const float* __restrict__ nH2, const float* __restrict__ Tgas,
                                                        const float* __restrict__ Tdust, const float* __restrict__ vlos,
                                                        float* __restrict__ coef) {
  // ncell is even and every pointer 8-byte aligned (the host checks)
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (2 * t >= ncell) return;
  const float2 n = reinterpret_cast<const float2*>(nH2)[t], T = reinterpret_cast<const float2*>(Tgas)[t];
  const float2 Td = reinterpret_cast<const float2*>(Tdust)[t], v = reinterpret_cast<const float2*>(vlos)[t];
  f32x2 x[N], inv;
  level_fractions2<N, BW>(lc, n.x, n.y, T.x, T.y, x, inv);
  f32x2 xu2 = pk1(0.0f), xl2 = pk1(0.0f);
#pragma unroll
  for (int l = 0; l < N; ++l) {
    xu2 = fma2(x[l], pk1(cc.pick_upper[l]), xu2);
    xl2 = fma2(x[l], pk1(cc.pick_lower[l]), xl2);
  }
  xu2 = mul2(xu2, inv); xl2 = mul2(xl2, inv);
  float xu0, xu1, xl0, xl1;
  upk(xu2, xu0, xu1);
  upk(xl2, xl0, xl1);
  float o0[6], o1[6];
  cell_coefficients(cc, n.x, T.x, Td.x, v.x, xu0, xl0, o0);
  cell_coefficients(cc, n.y, T.y, Td.y, v.y, xu1, xl1, o1);
#pragma unroll
  for (int q = 0; q < 6; ++q) reinterpret_cast<float2*>(coef + (int64_t)q * ncell)[t] = make_float2(o0[q], o1[q]);
}

// ---- Grid precomputation and lookup (section 4.2, and section 4.3) -------------
// Instead of the level balance per cell, the two line coefficients per tracer abundance (Eq. 4.2.1) are tabulated
// once per context on a (n_H2, T_gas) grid with geometrically spaced nodes and interpolated at run time: multilinear
// in the variables n_H2 and T_gas inside the grid cell that holds the point, the same form continued outside the
// grid ("linear behavior ... outside observability grid bounds and between grid points").  The device
// holds, per grid cell, the value at its lower corner and its three finite differences ("the grid gradients are also
// computed") for both coefficients, so a lookup is two 16-byte loads and six multiply-adds:
//   f(n, T) = f00 + fx u + fy v + fxy u v,   u = (n - n_i) / (n_i+1 - n_i),  v = (T - T_j) / (T_j+1 - T_j)
// with f = E = n x_u (emission) and f = A = n (x_l g_u / g_l - x_u) (absorption); e_c = c_e E, a_c = c_a A.
struct GridConsts {
  const float2* nodes_n;   // [nn]  { n_i, 1 / (n_i+1 - n_i) }   (the last entry repeats the last interval)
  const float2* nodes_T;   // [nT]  { T_j, 1 / (T_j+1 - T_j) }
  const float4* cells;     // [2][nT - 1][nn - 1]  { f00, fx, fy, fxy } of E, then of A
  int nn, nT;
  float log2_n_lo, inv_dlog2_n, log2_T_lo, inv_dlog2_T;   // cell index = floor((log2 v - log2 lo) * inv_dlog2)
};

// node values E, A at (n_i, T_j): nodeval[2][nT][nn]
template <int N, int BW, bool TABLE>
__global__ void __launch_bounds__(128) grid_nodes_kernel(LevelConsts lc, CoefConsts cc, GridConsts gc,
                                                         float* __restrict__ nodeval) {
  const int q = blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= gc.nn * gc.nT) return;
  const int i = q % gc.nn, j = q / gc.nn;
  const float n = gc.nodes_n[i].x, T = gc.nodes_T[j].x;
  float x[N], inv;
  level_fractions<N, BW, TABLE>(lc, n, T, x, &inv);
  float xu = 0.0f, xl = 0.0f;
#pragma unroll
  for (int l = 0; l < N; ++l) {
    xu = fmaf(x[l], cc.pick_upper[l], xu);
    xl = fmaf(x[l], cc.pick_lower[l], xl);
  }
  xu *= inv; xl *= inv;
  nodeval[q] = n * xu;
  nodeval[gc.nn * gc.nT + q] = n * fmaf(xl, cc.gr, -xu);
}

// per grid cell: lower-corner value and finite differences
__global__ void __launch_bounds__(128) grid_cells_kernel(int nn, int nT, const float* __restrict__ nodeval,
                                                         float4* __restrict__ cells) {
  const int q = blockIdx.x * blockDim.x + threadIdx.x;
  const int nc = (nn - 1) * (nT - 1);
  if (q >= 2 * nc) return;
  const int plane = q / nc, r = q % nc, i = r % (nn - 1), j = r / (nn - 1);
  const float* g = nodeval + (size_t)plane * nn * nT;
  const float f00 = g[j * nn + i], f10 = g[j * nn + i + 1], f01 = g[(j + 1) * nn + i], f11 = g[(j + 1) * nn + i + 1];
  cells[q] = make_float4(f00, f10 - f00, f01 - f00, (f11 - f10) - (f01 - f00));
}

// K2 with the lookup in place of K1: coef[6][ncell].  One cell of the lookup:
__device__ __forceinline__ void grid_cell(const CoefConsts& cc, const GridConsts& gc, float n, float T, float Td, float vlos,
                                          float (&o)[6]) {
  // grid cell (clamped to the first / last one: the multilinear form is continued outside the grid; a point that
  // lands in a neighbouring cell by the rounding of the logarithm sees the same value, the interpolant is continuous)
  const float fi = floorf((__log2f(fmaxf(n, 1.0e-37f)) - gc.log2_n_lo) * gc.inv_dlog2_n);
  const float fj = floorf((__log2f(fmaxf(T, 1.0e-37f)) - gc.log2_T_lo) * gc.inv_dlog2_T);
  const int i = (int)fminf(fmaxf(fi, 0.0f), (float)(gc.nn - 2)), j = (int)fminf(fmaxf(fj, 0.0f), (float)(gc.nT - 2));
  const float2 gn = __ldg(gc.nodes_n + i), gT = __ldg(gc.nodes_T + j);
  const float u = (n - gn.x) * gn.y, v = (T - gT.x) * gT.y;
  const int nc = (gc.nn - 1) * (gc.nT - 1), q = j * (gc.nn - 1) + i;
  const float4 fe = __ldg(gc.cells + q), fa = __ldg(gc.cells + nc + q);
  const float E = fmaf(fmaf(fe.w, v, fe.y), u, fmaf(fe.z, v, fe.x));
  const float A = fmaf(fmaf(fa.w, v, fa.y), u, fmaf(fa.z, v, fa.x));
  cell_coefficients(cc, 1.0f, T, Td, vlos, E, 0.0f, o);      // Doppler width, line centre, Planck source; e = c_e E
  o[1] = T > cc.T_inf ? 0.0f : cc.c_a * A;
  o[4] = cc.c_d * n;
}

// Four consecutive cells per thread (16-byte loads and stores: the kernel moves 40 bytes per cell and nothing else
// bounds it); `aligned` = every plane starts on a 16-byte boundary, else the scalar tail loop takes all cells.
__global__ void __launch_bounds__(256) cellcoef_grid_kernel(CoefConsts cc, GridConsts gc, int64_t ncell, int aligned,
                                                            const float* __restrict__ nH2, const float* __restrict__ Tgas,
                                                            const float* __restrict__ Tdust, const float* __restrict__ vlos,
                                                            float* __restrict__ coef) {
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t c0 = 4 * t;
  if (c0 >= ncell) return;
  if (aligned && c0 + 4 <= ncell) {
    const float4 n4 = *reinterpret_cast<const float4*>(nH2 + c0), T4 = *reinterpret_cast<const float4*>(Tgas + c0),
                 d4 = *reinterpret_cast<const float4*>(Tdust + c0), v4 = *reinterpret_cast<const float4*>(vlos + c0);
    float o[4][6];
    grid_cell(cc, gc, n4.x, T4.x, d4.x, v4.x, o[0]);
    grid_cell(cc, gc, n4.y, T4.y, d4.y, v4.y, o[1]);
    grid_cell(cc, gc, n4.z, T4.z, d4.z, v4.z, o[2]);
    grid_cell(cc, gc, n4.w, T4.w, d4.w, v4.w, o[3]);
#pragma unroll
    for (int k = 0; k < 6; ++k)
      *reinterpret_cast<float4*>(coef + (int64_t)k * ncell + c0) = make_float4(o[0][k], o[1][k], o[2][k], o[3][k]);
    return;
  }
  for (int64_t c = c0; c < min(c0 + 4, ncell); ++c) {
    float o[6];
    grid_cell(cc, gc, nH2[c], Tgas[c], Tdust[c], vlos[c], o);
#pragma unroll
    for (int k = 0; k < 6; ++k) coef[(int64_t)k * ncell + c] = o[k];
  }
}

// K2 alone, from caller-supplied populations pop[N][ncell].
__global__ void __launch_bounds__(256) coef_from_pop_kernel(CoefConsts cc, int64_t ncell, const float* __restrict__ nH2,
                                                            const float* __restrict__ Tgas,
                                                            const float* __restrict__ Tdust,
                                                            const float* __restrict__ vlos,
                                                            const float* __restrict__ pop, float* __restrict__ coef) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= ncell) return;
  float o[6];
  cell_coefficients(cc, nH2[i], Tgas[i], Tdust[i], vlos[i], pop[(int64_t)cc.upper * ncell + i],
                    pop[(int64_t)cc.lower * ncell + i], o);
#pragma unroll
  for (int q = 0; q < 6; ++q) coef[(int64_t)q * ncell + i] = o[q];
}

}  // namespace iris
