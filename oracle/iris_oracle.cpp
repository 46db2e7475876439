// ORACLE -- TEST INFRASTRUCTURE ONLY.  Not part of the product path.
//
// Plain, slow, float64, scalar C++ restatement of the IRIS-SO hot path of arxiv/paper_2607_01338
// (PAPER.md sections 3-4), written from the paper's equations in the paper's order and notation.
// It shares no code, header, table or constant generator with the CUDA path
// (paper_2607_01338_b200/csrc) and neither includes the other.  Only tests/, __graft_entry__.smoke()
// and bench.py's cpu_baseline / --impl reference legs may call it.
//
// Every function cites the passage it follows.  Readings of garbled / silent passages are the ones
// listed in DESIGN.md ("Readings") and SURVEY.md section 8(c).
//
// Pins (tests/test_oracle_pins.py): every function below is pinned by closed forms, limits,
// invariants or brute force -- none is "parity unpinned".
//
// Units: CGS throughout.  Field arrays are float32 [nz][ny][nx] (x fastest, k = 0 far side) and are
// widened to double on load; every intermediate and every output is double.

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>

namespace {

// O1 constants: CODATA-2018 exact SI values converted to CGS.
constexpr double kH = 6.62607015e-27;    // erg s
constexpr double kK = 1.380649e-16;      // erg / K
constexpr double kC = 2.99792458e10;     // cm / s
constexpr double kPi = 3.14159265358979323846;

}  // namespace

extern "C" {

// Parameter record of the oracle (declared here on its own; the CUDA path has its own struct).
struct orc_config {
  int32_t nx, ny, nz;
  double cell_cm;
  int32_t n_levels;
  const double *energy_K, *weight, *einstein_A, *coll_down_ref;
  double coll_T_ref, coll_T_exp;
  int32_t line_upper, line_lower;
  double nu0_Hz, mol_mass_g, abundance, microturb_cms, T_bar, T_cmb, T_inf;
  int32_t dust_on;
  double kappa_gas_cm2_g, mass_per_H2_g;
  int32_t nv;
  double v0_cms, dv_cms;
  int32_t subtract_continuum, subtract_space, out_unit;
  double beam_fwhm_px, noise_mu, noise_sigma;
  int32_t noise_gamma_mode;
  uint64_t seed;
  // transfer / integration modes of sections 4.4 - 4.8; all 0 = the hot path (reading R1)
  int32_t transfer_mode;   // 0 optically thick (4.5), 1 selectively thin (4.6), 2 optically thin (4.7)
  int32_t integration;     // 0 formal, 1 smooth (4.8: TR first step + BDF2; 4.7.7: Simpson in thin mode)
  int32_t subsample;       // thick mode only: 0 = channel-integrated profile (R1); odd f >= 1 = fine velocity
                           // grid with f added midpoints per channel + Simpson over frequency (4.5, Eq. 4.5.1)
  // tabulated collision rates of several partners (LAMDA tables "interpolated in temperature";
  // H, para-H2, ortho-H2 at 3:1, He at 0.1 per H).  coll_n_partners = 0: the power law above.
  int32_t coll_n_partners, coll_nT;
  const double *coll_T_grid;        // [nT] ascending temperatures
  const double *coll_table;         // [P][nT][n_levels * n_levels]  K_ul of partner p at T_grid[t], 0 where u <= l
  const double *coll_partner_frac;  // [P] number density of partner p per n_H2
  // grid precomputation of section 4.2 and the lookup of section 4.3; reading S31
  int32_t coef_grid;                // 0: level balance solved per cell; 1: coefficients interpolated from the grid
  int32_t grid_n_density, grid_n_temp;      // nodes along n_H2 and T_gas (paper: 128 and 64)
  double grid_nH2_lo, grid_nH2_hi, grid_T_lo, grid_T_hi;   // first and last node of each axis
  // 0: dust source, background and unit conversion at nu0 (reading S6); 1: at every channel's own frequency (PAPER.md:513,
  // "the Doppler-shifted Planck source function"; reading S32).  Hot-path mode only.
  int32_t dust_per_channel;
};

// Planck function B_nu(T), Eq. 3.2.1 = Eq. 3.6.2 = Eq. 4.9.1.
// T <= 0 gives 0 (no radiation field; "pure" OT case).
double orc_planck(double nu, double T) {
  if (!(T > 0.0)) return 0.0;
  return 2.0 * kH * nu * nu * nu / (kC * kC) / std::expm1(kH * nu / (kK * T));
}

// Inverse of Eq. 4.9.1: Planck brightness temperature of an intensity.
// Reading R7: odd extension for I < 0, T_B(0) = 0.
double orc_planck_TB(double nu, double I) {
  if (I == 0.0) return 0.0;
  double a = std::fabs(I);
  double T = (kH * nu / kK) / std::log1p(2.0 * kH * nu * nu * nu / (kC * kC * a));
  return I < 0.0 ? -T : T;
}

// Eq. 4.9.2: T_RJ = c^2 I / (2 k nu^2).
double orc_rayleigh_jeans_T(double nu, double I) { return kC * kC * I / (2.0 * kK * nu * nu); }

// ---------------------------------------------------------------------------------------------
// O3  Level balance, Eq. 3.6.1 - 3.6.3 with Eq. 3.7.1 - 3.7.2.
// Builds the transition rates R[i*N + j] = C_ij + A_ij + B_ij J_ij   (i -> j, per unit n_i, i != j).
//   C_ij = K_ij n_H2                                   (Eq. 3.6.3, single partner H2)
//   K_ul(T) = K_ul(T_ref) (T / T_ref)^p for u > l      (input table)
//   K_lu = K_ul (g_u / g_l) exp(-(E_u - E_l) / T_gas)  (Eq. 3.7.2, detailed balance)
//   B_ul = c^2 / (2 h nu^3) A_ul,  B_lu = (g_u / g_l) B_ul   (Eq. 3.7.1)
//   J_ul = B_nu_ul(T_bar)                              (Eq. 3.6.2, reading G2: the temperature is T_bar)
// Tabulated de-excitation rate per unit n_H2 (reading S30): every partner's table is interpolated linearly
// in temperature between its grid points and held constant outside the grid (the LAMDA convention), and the partners
// add with their number densities per n_H2:  K_ul(T) = sum_p f_p K^p_ul(T)   (Eq. 3.6.3 summed over partners).
static double table_rate(const orc_config *c, int u, int l, double T) {
  const int N = c->n_levels, nT = c->coll_nT;
  const double *Tg = c->coll_T_grid;
  int t0 = 0;
  double w = 0.0;
  if (nT > 1) {
    if (T <= Tg[0]) { t0 = 0; w = 0.0; }
    else if (T >= Tg[nT - 1]) { t0 = nT - 2; w = 1.0; }
    else {
      while (t0 + 2 < nT && T >= Tg[t0 + 1]) ++t0;
      w = (T - Tg[t0]) / (Tg[t0 + 1] - Tg[t0]);
    }
  }
  double K = 0.0;
  for (int p = 0; p < c->coll_n_partners; ++p) {
    const double *tab = c->coll_table + ((int64_t)p * nT) * N * N;
    const double k0 = tab[(int64_t)t0 * N * N + u * N + l];
    const double k1 = nT > 1 ? tab[(int64_t)(t0 + 1) * N * N + u * N + l] : k0;
    K += c->coll_partner_frac[p] * (k0 + w * (k1 - k0));
  }
  return K;
}

void orc_rates(const orc_config *c, double nH2, double Tgas, double *R) {
  const int N = c->n_levels;
  for (int i = 0; i < N * N; ++i) R[i] = 0.0;
  for (int u = 1; u < N; ++u) {
    for (int l = 0; l < u; ++l) {
      const double dE = c->energy_K[u] - c->energy_K[l];   // (E_u - E_l) / k, Kelvin
      const double gr = c->weight[u] / c->weight[l];
      double down = 0.0, up = 0.0;
      if (c->coll_n_partners > 0) {
        const double K = table_rate(c, u, l, Tgas);
        down += K * nH2;
        up += K * gr * std::exp(-dE / Tgas) * nH2;
      } else {
        const double Kul = c->coll_down_ref[u * N + l];
        if (Kul != 0.0) {
          const double K = Kul * std::pow(Tgas / c->coll_T_ref, c->coll_T_exp);
          down += K * nH2;
          up += K * gr * std::exp(-dE / Tgas) * nH2;
        }
      }
      const double A = c->einstein_A[u * N + l];
      if (A != 0.0) {
        const double nu = kK * dE / kH;
        const double Bul = kC * kC / (2.0 * kH * nu * nu * nu) * A;
        const double Blu = gr * Bul;
        const double J = orc_planck(nu, c->T_bar);
        down += A + Bul * J;
        up += Blu * J;
      }
      R[u * N + l] = down;
      R[l * N + u] = up;
    }
  }
}

// Statistical-equilibrium matrix of Eq. 3.6.1: (M x)_i = sum_{j != i} [x_j R_ji - x_i R_ij].
// Row 0 is NOT yet replaced here (used by the stationarity pin).
void orc_balance_matrix(const orc_config *c, double nH2, double Tgas, double *M) {
  const int N = c->n_levels;
  std::vector<double> R(N * N);
  orc_rates(c, nH2, Tgas, R.data());
  for (int i = 0; i < N; ++i) {
    double out = 0.0;
    for (int j = 0; j < N; ++j) {
      if (j == i) continue;
      M[i * N + j] = R[j * N + i];
      out += R[i * N + j];
    }
    M[i * N + i] = -out;
  }
}

// Dense partial-pivot Gaussian elimination, A x = b, A is n x n row-major (destroyed).
static void solve_ge(int n, double *A, double *b, double *x) {
  for (int k = 0; k < n; ++k) {
    int p = k;
    double best = std::fabs(A[k * n + k]);
    for (int r = k + 1; r < n; ++r)
      if (std::fabs(A[r * n + k]) > best) { best = std::fabs(A[r * n + k]); p = r; }
    if (p != k) {
      for (int j = 0; j < n; ++j) { double t = A[k * n + j]; A[k * n + j] = A[p * n + j]; A[p * n + j] = t; }
      double t = b[k]; b[k] = b[p]; b[p] = t;
    }
    for (int r = k + 1; r < n; ++r) {
      const double f = A[r * n + k] / A[k * n + k];
      if (f == 0.0) continue;
      for (int j = k; j < n; ++j) A[r * n + j] -= f * A[k * n + j];
      b[r] -= f * b[k];
    }
  }
  for (int k = n - 1; k >= 0; --k) {
    double s = b[k];
    for (int j = k + 1; j < n; ++j) s -= A[k * n + j] * x[j];
    x[k] = s / A[k * n + k];
  }
}

// Level fractions x_i (sum = 1) of one cell: Eq. 3.6.1 with the ground-state row replaced by the
// conservation equation, N = 1 (fractions; linearity in abundance).
void orc_levelpop_cell(const orc_config *c, double nH2, double Tgas, double *x) {
  const int N = c->n_levels;
  std::vector<double> M(N * N), b(N, 0.0);
  orc_balance_matrix(c, nH2, Tgas, M.data());
  for (int j = 0; j < N; ++j) M[j] = 1.0;
  b[0] = 1.0;
  solve_ge(N, M.data(), b.data(), x);
}

// pop[N][ncell] for arrays of cells.
void orc_levelpop(const orc_config *c, int64_t ncell, const float *nH2, const float *Tgas, double *pop) {
  const int N = c->n_levels;
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < ncell; ++i) {
    double x[32];
    orc_levelpop_cell(c, (double)nH2[i], (double)Tgas[i], x);
    for (int l = 0; l < N; ++l) pop[(int64_t)l * ncell + i] = x[l];
  }
}

// ---------------------------------------------------------------------------------------------
// O4  Per-cell coefficients.
//   j^[L]     = (h nu0 / 4 pi) n_u A_ul                       Eq. 3.3.1
//   alpha^[L] = (h nu0 / 4 pi) (n_l B_lu - n_u B_ul)          Eq. 3.3.2
//   n_i = X n_H2 x_i                                          Eq. 4.2.1, reading S16
//   b = sqrt(2 k T / m_a + xi^2)   (Delta nu_D = nu0 b / c)   Eq. 3.3.4, reading S1
//   alpha^[D] = kappa rho_gas, rho_gas = mass_per_H2 n_H2     Eq. 3.2.2, reading S3
//   S^[D] = B_nu0(T_dust)                                     Eq. 3.2.1, reading S6
//   no line above T_inf
// out5 = {j0, kappa0, b, alpha_d, S_d}
void orc_cell_coefficients(const orc_config *c, double nH2, double Tgas, double Tdust, const double *x,
                           double *out5) {
  const int N = c->n_levels;
  const int u = c->line_upper, l = c->line_lower;
  const double nu0 = c->nu0_Hz;
  const double A = c->einstein_A[u * N + l];
  const double Bul = kC * kC / (2.0 * kH * nu0 * nu0 * nu0) * A;
  const double Blu = c->weight[u] / c->weight[l] * Bul;
  const double ntr = c->abundance * nH2;
  double j0 = kH * nu0 / (4.0 * kPi) * ntr * x[u] * A;
  double k0 = kH * nu0 / (4.0 * kPi) * ntr * (x[l] * Blu - x[u] * Bul);
  if (Tgas > c->T_inf) { j0 = 0.0; k0 = 0.0; }
  out5[0] = j0;
  out5[1] = k0;
  out5[2] = std::sqrt(2.0 * kK * Tgas / c->mol_mass_g + c->microturb_cms * c->microturb_cms);
  out5[3] = c->dust_on ? c->kappa_gas_cm2_g * c->mass_per_H2_g * nH2 : 0.0;
  out5[4] = c->dust_on ? orc_planck(nu0, Tdust) : 0.0;
}

// ---------------------------------------------------------------------------------------------
// O4b  Grid precomputation (section 4.2) and runtime lookup (section 4.3).
// "the frequency-independent line emission and absorption coefficients j^[L], alpha^[L] ... are solved over a 3D grid of
// dimensions gas density, H2 abundance, and gas kinetic temperature"; "the grid gradients are also computed to allow
// the runtime computation ... via a fast linear interpolation ... emission and absorption that exhibit linear
// behavior, rather than merely constant behavior, outside observability grid bounds and between grid points"; grids
// are "per tracer abundance" (Eq. 4.2.1: j = chi j~, alpha = chi alpha~).
// Reading S31: the per-cell inputs of this path are n_H2 and T_gas (all hydrogen molecular, collision
// partners in fixed proportion to n_H2), so the H2-abundance axis has a single node and the grid is two-dimensional;
// nodes are spaced geometrically between the configured end points (the paper states neither spacing nor bounds);
// the interpolation is multilinear IN THE VARIABLES n_H2 and T_gas inside the grid cell that contains the point, its
// gradients being the finite differences of the node values; outside the grid the nearest cell's multilinear form is
// continued (linear extrapolation along each axis).
// grid[2][nT][nn]: j~ = j0 / X and alpha~ = kappa0 / X at the nodes.
double orc_grid_node(double lo, double hi, int n, int i) {
  return n > 1 ? lo * std::pow(hi / lo, (double)i / (double)(n - 1)) : lo;
}

void orc_grid_build(const orc_config *c, double *grid) {
  const int nn = c->grid_n_density, nT = c->grid_n_temp;
  orc_config c1 = *c;
  c1.abundance = 1.0;                 // per tracer abundance, Eq. 4.2.1
  c1.T_inf = std::numeric_limits<double>::infinity();     // the T_inf mask is applied after the lookup
#pragma omp parallel for schedule(static)
  for (int q = 0; q < nn * nT; ++q) {
    const int i = q % nn, j = q / nn;
    const double n = orc_grid_node(c->grid_nH2_lo, c->grid_nH2_hi, nn, i);
    const double T = orc_grid_node(c->grid_T_lo, c->grid_T_hi, nT, j);
    double x[32], o[5];
    orc_levelpop_cell(&c1, n, T, x);
    orc_cell_coefficients(&c1, n, T, T, x, o);
    grid[q] = o[0];
    grid[(int64_t)nn * nT + q] = o[1];
  }
}

// Multilinear interpolation / extrapolation of one grid plane g[nT][nn] at (n, T).
double orc_grid_lookup_plane(const double *g, int nn, int nT, double n_lo, double n_hi, double T_lo, double T_hi,
                             double n, double T) {
  // index of the grid cell: the last node not above the point, clamped to the first / last cell
  auto cell_of = [](double lo, double hi, int cnt, double v) {
    if (cnt < 2) return 0;
    int i = (int)std::floor(std::log(v / lo) / std::log(hi / lo) * (cnt - 1));
    if (!(v > 0.0)) i = 0;
    i = std::max(0, std::min(cnt - 2, i));
    // the logarithm may land one cell off at a node: settle it with the node values themselves
    while (i > 0 && v < orc_grid_node(lo, hi, cnt, i)) --i;
    while (i < cnt - 2 && v >= orc_grid_node(lo, hi, cnt, i + 1)) ++i;
    return i;
  };
  const int i = cell_of(n_lo, n_hi, nn, n), j = cell_of(T_lo, T_hi, nT, T);
  const int i1 = std::min(i + 1, nn - 1), j1 = std::min(j + 1, nT - 1);
  const double n0 = orc_grid_node(n_lo, n_hi, nn, i), n1 = orc_grid_node(n_lo, n_hi, nn, i1);
  const double T0 = orc_grid_node(T_lo, T_hi, nT, j), T1 = orc_grid_node(T_lo, T_hi, nT, j1);
  const double u = n1 > n0 ? (n - n0) / (n1 - n0) : 0.0, v = T1 > T0 ? (T - T0) / (T1 - T0) : 0.0;
  const double f00 = g[(int64_t)j * nn + i], f10 = g[(int64_t)j * nn + i1], f01 = g[(int64_t)j1 * nn + i],
               f11 = g[(int64_t)j1 * nn + i1];
  return f00 + (f10 - f00) * u + (f01 - f00) * v + (f11 - f10 - f01 + f00) * u * v;
}

// j0, kappa0 of one cell from the grid: lookup, abundance applied last, then the T_inf mask.
void orc_grid_cell(const orc_config *c, const double *grid, double nH2, double Tgas, double *j0, double *k0) {
  const int nn = c->grid_n_density, nT = c->grid_n_temp;
  *j0 = c->abundance * orc_grid_lookup_plane(grid, nn, nT, c->grid_nH2_lo, c->grid_nH2_hi, c->grid_T_lo, c->grid_T_hi, nH2, Tgas);
  *k0 = c->abundance * orc_grid_lookup_plane(grid + (int64_t)nn * nT, nn, nT, c->grid_nH2_lo, c->grid_nH2_hi, c->grid_T_lo,
                                             c->grid_T_hi, nH2, Tgas);
  if (Tgas > c->T_inf) { *j0 = 0.0; *k0 = 0.0; }
}

// coef[5][ncell]; pop may be NULL (then solved here, or looked up in the grid when coef_grid = 1) or [N][ncell].
void orc_coefficients(const orc_config *c, int64_t ncell, const float *nH2, const float *Tgas,
                      const float *Tdust, const double *pop, double *coef) {
  const int N = c->n_levels;
  std::vector<double> grid;
  const bool use_grid = !pop && c->coef_grid != 0;
  if (use_grid) {
    grid.resize((size_t)2 * c->grid_n_density * c->grid_n_temp);
    orc_grid_build(c, grid.data());
  }
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < ncell; ++i) {
    double x[32], o[5];
    if (use_grid) {
      for (int l = 0; l < N; ++l) x[l] = 0.0;       // the populations are not needed: the grid holds the line coefficients
      orc_cell_coefficients(c, (double)nH2[i], (double)Tgas[i], (double)Tdust[i], x, o);
      orc_grid_cell(c, grid.data(), (double)nH2[i], (double)Tgas[i], &o[0], &o[1]);
    } else {
      if (pop) for (int l = 0; l < N; ++l) x[l] = pop[(int64_t)l * ncell + i];
      else orc_levelpop_cell(c, (double)nH2[i], (double)Tgas[i], x);
      orc_cell_coefficients(c, (double)nH2[i], (double)Tgas[i], (double)Tdust[i], x, o);
    }
    for (int q = 0; q < 5; ++q) coef[(int64_t)q * ncell + i] = o[q];
  }
}

// ---------------------------------------------------------------------------------------------
// O5  Channel-averaged (integrated) Gaussian profile, Eq. 4.4.1 applied to Eq. 3.3.3
// (PAPER.md:378), i.e. Eq. 4.6.3 (reading G1: erf difference between channel edges).
// Worked in velocity space (reading G9): channel k has centre v_k = v0 + k dv and edges v_k -+ dv/2;
// a cell emits at channel velocity v = v_los.  Delta nu_W = nu0 dv / c.
//   phibar_k = [erf((v_k + dv/2 - v_los)/b) - erf((v_k - dv/2 - v_los)/b)] / (2 Delta nu_W)   [1/Hz]
double orc_phibar(const orc_config *c, int k, double vlos, double b) {
  const double vk = c->v0_cms + k * c->dv_cms;
  const double dnuW = c->nu0_Hz * c->dv_cms / kC;
  const double hi = (vk + 0.5 * c->dv_cms - vlos) / b;
  const double lo = (vk - 0.5 * c->dv_cms - vlos) / b;
  return (std::erf(hi) - std::erf(lo)) / (2.0 * dnuW);
}

// Point profile phi(nu) of Eq. 3.3.3 evaluated at the frequency that corresponds to velocity v
// (used only by the brute-force pin).  Delta nu_D = nu0 b / c (Eq. 3.3.4).
double orc_phi_point(const orc_config *c, double v, double vlos, double b) {
  const double dnuD = c->nu0_Hz * b / kC;
  const double x = (v - vlos) / b;
  return std::exp(-x * x) / (dnuD * std::sqrt(kPi));
}

// w(tau) = (1 - e^-tau) / tau, w(0) = 1: the formal step S (1 - e^-tau) written as j h w(tau)
// (reading S13: identical for alpha != 0, defined for alpha = 0 and alpha < 0).
static double w_of_tau(double tau) { return tau == 0.0 ? 1.0 : -std::expm1(-tau) / tau; }

// O6  Formal integration step, Eq. 4.8.5 - 4.8.7:
//   I_{n+1} = I_n e^-tau + S (1 - e^-tau),  S = j / alpha,  tau = h alpha.
static double formal_step(double I, double j, double alpha, double h) {
  const double tau = alpha * h;
  return I * std::exp(-tau) + j * h * w_of_tau(tau);
}

// ---------------------------------------------------------------------------------------------
// O6b  The other transfer / integration modes of the paper (sections 4.5 - 4.8), one spectral point of one
// column at a time.  A "point" carries a profile weight per cell:
//   p_n = phibar_k(cell n)            channel-integrated profile, Eq. 4.6.3 (coarse grid)
//   p_n = phi(nu_point; cell n)       point profile, Eq. 3.3.3 (fine grid of the thick mode, section 4.5)
// and the per-cell coefficients  jL_n = j0_n p_n,  aL_n = kappa0_n p_n,  jD_n = alpha_d,n S_d,n,  aD_n = alpha_d,n.
//
// Readings: S23 selectively thin uses the continuum intensity of the SAME grid index as the
// coefficients (formal: the continuum after its own step of that cell, "we simply solve for the continuum step
// first"); S24 smooth integration treats cell n as the point x_n = n h with y_0 = I_bg at the
// farthest cell and takes R - 1 steps (TR for the first, BDF2 after); S25 thin-smooth Simpson panels
// span two cell spacings [x_2m, x_2m+2] (Eq. 4.7.7 with its h = 2 cell spacings, "sum of order floor((R-1)/2)"),
// a left-over last interval (R even) is integrated by the trapezoidal rule; S26 the ReLU of PAPER.md:709, 717, 738
// is applied after every smooth step and after every selectively-thin step, to total and continuum alike.
static double relu(double x) { return x > 0.0 ? x : 0.0; }

// p[n], n = 0..R-1: profile weights of this spectral point; cont[n]: continuum intensity at grid index n as
// produced by orc_continuum_column for the same integration (needed by the selectively thin mode).
// Returns the total intensity of this spectral point at the observer.
static double total_point(const orc_config *c, int R, const double *p, const double *j0, const double *k0,
                          const double *ad, const double *Sd, const double *cont, double Ibg) {
  const double h = c->cell_cm;
  const int mode = c->transfer_mode;
  if (mode == 2) {                                   // optically thin, Eq. 4.7.3 - 4.7.4
    if (c->integration == 0) {                       // Eq. 4.7.6: midpoint sum
      double I = Ibg;
      for (int n = 0; n < R; ++n) I += h * (j0[n] * p[n] + ad[n] * Sd[n]);
      return I;
    }
    double I = Ibg;                                  // Eq. 4.7.7: Simpson panels of two cell spacings
    int n = 0;
    for (; n + 2 < R; n += 2) {
      const double f0 = j0[n] * p[n] + ad[n] * Sd[n], f1 = j0[n + 1] * p[n + 1] + ad[n + 1] * Sd[n + 1],
                   f2 = j0[n + 2] * p[n + 2] + ad[n + 2] * Sd[n + 2];
      I += (2.0 * h / 6.0) * (f0 + 4.0 * f1 + f2);
    }
    if (n + 1 < R) I += 0.5 * h * ((j0[n] * p[n] + ad[n] * Sd[n]) + (j0[n + 1] * p[n + 1] + ad[n + 1] * Sd[n + 1]));
    return I;
  }
  // thick (Eq. 4.8.6 - 4.8.8) or selectively thin (Eq. 4.8.14 - 4.8.15) coefficients at grid index n;
  // Ic = continuum intensity paired with index n
  auto jT = [&](int n, double Ic) {
    return mode == 0 ? j0[n] * p[n] + ad[n] * Sd[n] : j0[n] * p[n] + ad[n] * Sd[n] - k0[n] * p[n] * Ic;
  };
  auto aT = [&](int n) { return mode == 0 ? k0[n] * p[n] + ad[n] : ad[n]; };
  if (c->integration == 0) {                         // formal, Eq. 4.8.5; cont[n] = continuum after cell n
    double I = Ibg;
    for (int n = 0; n < R; ++n) {
      I = formal_step(I, jT(n, cont[n]), aT(n), h);
      if (mode == 1) I = relu(I);
    }
    return I;
  }
  // smooth: y_0 = I_bg at x_0; TR (Eq. 4.8.12) for the first step, BDF2 (Eq. 4.8.10) after; cont[n] = continuum at x_n
  if (R < 2) return Ibg;
  double Im = Ibg;
  double I = relu((h * (jT(0, cont[0]) + jT(1, cont[1])) + (2.0 - h * aT(0)) * Im) / (2.0 + h * aT(1)));
  for (int n = 2; n < R; ++n) {
    const double In = relu((2.0 * h * jT(n, cont[n]) + 4.0 * I - Im) / (3.0 + 2.0 * h * aT(n)));
    Im = I;
    I = In;
  }
  return I;
}

// Continuum baseline of one column, Eq. 3.1.3 with Eq. 4.4.3 - 4.4.5, in the chosen mode
// and integration.  cont[n] as total_point expects it; returns the continuum at the observer.
static double continuum_column(const orc_config *c, int R, const double *ad, const double *Sd, double Ibg, double *cont) {
  const double h = c->cell_cm;
  if (c->transfer_mode == 2) {                       // thin: Eq. 4.7.5 (cont[] unused by total_point)
    std::vector<double> zero(R, 0.0);
    for (int n = 0; n < R; ++n) cont[n] = 0.0;
    return total_point(c, R, zero.data(), zero.data(), zero.data(), ad, Sd, cont, Ibg);
  }
  if (c->integration == 0) {
    double I = Ibg;
    for (int n = 0; n < R; ++n) {
      I = formal_step(I, ad[n] * Sd[n], ad[n], h);
      if (c->transfer_mode == 1) I = relu(I);
      cont[n] = I;
    }
    return I;
  }
  cont[0] = Ibg;
  if (R < 2) return Ibg;
  cont[1] = relu((h * (ad[0] * Sd[0] + ad[1] * Sd[1]) + (2.0 - h * ad[0]) * cont[0]) / (2.0 + h * ad[1]));
  for (int n = 2; n < R; ++n)
    cont[n] = relu((2.0 * h * ad[n] * Sd[n] + 4.0 * cont[n - 1] - cont[n - 2]) / (3.0 + 2.0 * h * ad[n]));
  return cont[R - 1];
}

// One column in any mode other than the hot path.  Coarse grid: one point per channel with phibar.  Fine grid
// (thick mode, subsample = f odd): points at spacing dv / (f + 1) from the lower edge of channel 0; the channel
// average is the composite Simpson rule over the (f + 1) / 2 panels of the channel (Eq. 4.5.1, 4.4.1 - 4.4.2).
static void march_column_modes(const orc_config *c, const double *coef, const float *vlos, int64_t pix,
                               double *I_tot, double *I_cont) {
  const int64_t plane = (int64_t)c->nx * c->ny, ncell = plane * c->nz;
  const int R = c->nz;
  const double Ibg = orc_planck(c->nu0_Hz, c->T_cmb);
  std::vector<double> j0(R), k0(R), b(R), ad(R), Sd(R), vl(R), cont(R), p(R);
  for (int n = 0; n < R; ++n) {
    const int64_t cell = (int64_t)n * plane + pix;
    j0[n] = coef[cell]; k0[n] = coef[ncell + cell]; b[n] = coef[2 * ncell + cell];
    ad[n] = coef[3 * ncell + cell]; Sd[n] = coef[4 * ncell + cell]; vl[n] = (double)vlos[cell];
  }
  *I_cont = continuum_column(c, R, ad.data(), Sd.data(), Ibg, cont.data());
  const int f = (c->transfer_mode == 0) ? c->subsample : 0;
  if (f == 0) {
    for (int v = 0; v < c->nv; ++v) {
      for (int n = 0; n < R; ++n) p[n] = orc_phibar(c, v, vl[n], b[n]);
      I_tot[v] = total_point(c, R, p.data(), j0.data(), k0.data(), ad.data(), Sd.data(), cont.data(), Ibg);
    }
    return;
  }
  const int m = f + 1;                                // fine intervals per channel
  const double dvf = c->dv_cms / m;
  std::vector<double> If((size_t)c->nv * m + 1);
  for (size_t q = 0; q < If.size(); ++q) {
    const double vel = c->v0_cms - 0.5 * c->dv_cms + q * dvf;
    for (int n = 0; n < R; ++n) p[n] = orc_phi_point(c, vel, vl[n], b[n]);
    If[q] = total_point(c, R, p.data(), j0.data(), k0.data(), ad.data(), Sd.data(), cont.data(), Ibg);
  }
  for (int v = 0; v < c->nv; ++v) {
    double acc = 0.0;
    for (int q = 0; q < m; q += 2) acc += If[(size_t)v * m + q] + 4.0 * If[(size_t)v * m + q + 1] + If[(size_t)v * m + q + 2];
    I_tot[v] = acc * (2.0 * dvf / 6.0) / c->dv_cms;   // (1 / Delta nu_W) * integral, in velocity units
  }
}

// March one pixel column (k = 0 far ... nz-1 near; reading S11) for all channels.
// coef = {j0, kappa0, b, alpha_d, S_d} planes [5][ncell], vlos plane float32.
// Total: alpha = kappa0 phibar + alpha_d, j = j0 phibar + alpha_d S_d   (Eq. 4.8.6-4.8.7, 4.6.4)
// Continuum: alpha = alpha_d, j = alpha_d S_d                           (Eq. 3.1.3, 4.4.3-4.4.5)
// Both start from I_bg = B_nu0(T_cmb).  No ReLU clamp (smooth integrator only).
void orc_march_column(const orc_config *c, const double *coef, const float *vlos, int64_t pix,
                      double *I_tot /*[nv]*/, double *I_cont /*[1]*/) {
  if (c->transfer_mode != 0 || c->integration != 0 || c->subsample != 0) {
    march_column_modes(c, coef, vlos, pix, I_tot, I_cont);
    return;
  }
  const int64_t plane = (int64_t)c->nx * c->ny, ncell = plane * c->nz;
  const double h = c->cell_cm;
  const double Ibg = orc_planck(c->nu0_Hz, c->T_cmb);
  for (int v = 0; v < c->nv; ++v) I_tot[v] = Ibg;
  double Ic = Ibg;
  for (int k = 0; k < c->nz; ++k) {
    const int64_t cell = (int64_t)k * plane + pix;
    const double j0 = coef[cell], k0 = coef[ncell + cell], b = coef[2 * ncell + cell];
    const double ad = coef[3 * ncell + cell], Sd = coef[4 * ncell + cell];
    const double vl = (double)vlos[cell];
    for (int v = 0; v < c->nv; ++v) {
      const double pb = orc_phibar(c, v, vl, b);
      I_tot[v] = formal_step(I_tot[v], j0 * pb + ad * Sd, k0 * pb + ad, h);
    }
    Ic = formal_step(Ic, ad * Sd, ad, h);
  }
  *I_cont = Ic;
}

// O6c  The hot-path march with the dust source, the background and (in orc_observe) the unit conversion evaluated at
// every channel's own frequency instead of nu0 (the dust emission coefficients "are then computed over all
// points on the velocity/frequency-expanded physical-tensor grid according to the Doppler-shifted Planck source
// function given in Equation 3.2.1"; the dust opacity stays "constant over the small frequency window" of the line).
// Reading S32, with the classical Doppler shift of Eq. 4.3.1 and the radio convention of reading G9:
//   channel k is observed at        nu_k  = nu0 (1 - v_k / c)
//   a cell moving with v_los emits  nu'   = nu_k (1 + v_los / c)   in its own frame:  S_d = B_nu'(T_dust)
//   the background enters as        I_bg  = B_nu_k(T_cmb)
// The continuum is then a spectrum, not a scalar: I_cont[nv].  The line terms are unchanged (j0, kappa0 and the
// profile are defined at the line).
double orc_channel_frequency(const orc_config *c, int k) {
  return c->nu0_Hz * (1.0 - (c->v0_cms + k * c->dv_cms) / kC);
}

void orc_march_column_perchannel(const orc_config *c, const double *coef, const float *vlos, const float *Tdust,
                                 int64_t pix, double *I_tot /*[nv]*/, double *I_cont /*[nv]*/) {
  const int64_t plane = (int64_t)c->nx * c->ny, ncell = plane * c->nz;
  const double h = c->cell_cm;
  for (int v = 0; v < c->nv; ++v) I_tot[v] = I_cont[v] = orc_planck(orc_channel_frequency(c, v), c->T_cmb);
  for (int k = 0; k < c->nz; ++k) {
    const int64_t cell = (int64_t)k * plane + pix;
    const double j0 = coef[cell], k0 = coef[ncell + cell], b = coef[2 * ncell + cell], ad = coef[3 * ncell + cell];
    const double vl = (double)vlos[cell], Td = (double)Tdust[cell];
    for (int v = 0; v < c->nv; ++v) {
      const double Sd = c->dust_on ? orc_planck(orc_channel_frequency(c, v) * (1.0 + vl / kC), Td) : 0.0;
      const double pb = orc_phibar(c, v, vl, b);
      I_tot[v] = formal_step(I_tot[v], j0 * pb + ad * Sd, k0 * pb + ad, h);
      I_cont[v] = formal_step(I_cont[v], ad * Sd, ad, h);
    }
  }
}

// Columns pix[0..npix): I_tot[npix][nv], I_cont[npix][nv].
void orc_march_perchannel(const orc_config *c, const double *coef, const float *vlos, const float *Tdust, int64_t npix,
                          const int64_t *pix, double *I_tot, double *I_cont) {
#pragma omp parallel for schedule(dynamic, 4)
  for (int64_t p = 0; p < npix; ++p)
    orc_march_column_perchannel(c, coef, vlos, Tdust, pix[p], I_tot + p * c->nv, I_cont + p * c->nv);
}

// Columns pix[0..npix): I_tot[npix][nv], I_cont[npix].
void orc_march(const orc_config *c, const double *coef, const float *vlos, int64_t npix,
               const int64_t *pix, double *I_tot, double *I_cont) {
#pragma omp parallel for schedule(dynamic, 4)
  for (int64_t p = 0; p < npix; ++p)
    orc_march_column(c, coef, vlos, pix[p], I_tot + p * c->nv, I_cont + p);
}

// O7  Continuum subtraction and unit conversion (Eq. 4.9.1-4.9.2).
//   subtract_space 0: D = I_tot - I_cont (intensity space == RJ space), then converted to out_unit
//   subtract_space 1: T_B(I_tot) - T_B(I_cont)  (Planck space; result is in Kelvin)
//   subtract_continuum 0: I_tot converted to out_unit.
// nu: the frequency the conversion is made at (nu0, or the channel's own frequency with dust_per_channel = 1)
double orc_convert_voxel_nu(const orc_config *c, double nu, double It, double Ic) {
  if (c->subtract_continuum && c->subtract_space == 1) return orc_planck_TB(nu, It) - orc_planck_TB(nu, Ic);
  const double D = c->subtract_continuum ? It - Ic : It;
  if (c->out_unit == 0) return D;
  if (c->out_unit == 1) return orc_rayleigh_jeans_T(nu, D);
  return orc_planck_TB(nu, D);
}

double orc_convert_voxel(const orc_config *c, double It, double Ic) {
  const double nu = c->nu0_Hz;
  if (c->subtract_continuum && c->subtract_space == 1) return orc_planck_TB(nu, It) - orc_planck_TB(nu, Ic);
  const double D = c->subtract_continuum ? It - Ic : It;
  if (c->out_unit == 0) return D;
  if (c->out_unit == 1) return orc_rayleigh_jeans_T(nu, D);
  return orc_planck_TB(nu, D);
}

void orc_convert(const orc_config *c, int64_t npix, const double *I_tot, const double *I_cont, double *cube) {
  for (int64_t p = 0; p < npix; ++p)
    for (int v = 0; v < c->nv; ++v)
      cube[p * c->nv + v] = orc_convert_voxel(c, I_tot[p * c->nv + v], I_cont[p]);
}

// ---------------------------------------------------------------------------------------------
// O8  Gaussian beam, reading S8: sigma = FWHM / (2 sqrt(2 ln 2)), integer-offset
// samples g(d) ~ exp(-d^2 / 2 sigma^2), |d| <= R = ceil(4 sigma), normalised to sum 1 in 1-D, zero
// outside the image ("same" convolution).  Direct 2-D sum (not separated) per channel.
int orc_beam_radius(double fwhm_px) {
  const double sigma = fwhm_px / (2.0 * std::sqrt(2.0 * std::log(2.0)));
  return (int)std::ceil(4.0 * sigma);
}

void orc_beam_weights(double fwhm_px, double *g /*[2R+1]*/) {
  const double sigma = fwhm_px / (2.0 * std::sqrt(2.0 * std::log(2.0)));
  const int R = orc_beam_radius(fwhm_px);
  double s = 0.0;
  for (int d = -R; d <= R; ++d) { g[d + R] = std::exp(-0.5 * d * d / (sigma * sigma)); s += g[d + R]; }
  for (int d = 0; d <= 2 * R; ++d) g[d] /= s;
}

void orc_beam(int ny, int nx, int nv, double fwhm_px, const double *in, double *out) {
  const int R = orc_beam_radius(fwhm_px);
  std::vector<double> g(2 * R + 1);
  orc_beam_weights(fwhm_px, g.data());
#pragma omp parallel for schedule(static)
  for (int y = 0; y < ny; ++y)
    for (int x = 0; x < nx; ++x)
      for (int v = 0; v < nv; ++v) {
        double s = 0.0;
        for (int dy = -R; dy <= R; ++dy) {
          const int yy = y + dy;
          if (yy < 0 || yy >= ny) continue;
          for (int dx = -R; dx <= R; ++dx) {
            const int xx = x + dx;
            if (xx < 0 || xx >= nx) continue;
            s += g[dy + R] * g[dx + R] * in[((int64_t)yy * nx + xx) * nv + v];
          }
        }
        out[((int64_t)y * nx + x) * nv + v] = s;
      }
}

// ---------------------------------------------------------------------------------------------
// O9  Noise, Eq. 4.12.1: T += gamma (mu + sigma z), z ~ N(0,1) independently per voxel.
// Reading S10: z comes from the counter-based generator Philox4x32-10 (Salmon et al. 2011)
// with key = (seed lo, seed hi); one call, counter = (voxel / 4 lo, voxel / 4 hi, 0, 0), serves four consecutive
// voxels: words (r0, r1) the voxels 4c, 4c+1 and words (r2, r3) the voxels 4c+2, 4c+3; a word pair gives
// u1 = ((ra >> 8) + 0.5) 2^-24, u2 = ((rb >> 8) + 0.5) 2^-24 and the two independent Box-Muller deviates
// z = sqrt(-2 ln u1) cos(2 pi u2) for the even voxel, sqrt(-2 ln u1) sin(2 pi u2) for the odd one.
// gamma (reading S9): mode 0 -> 1; mode 1 -> one draw per cube,
// gamma = (r0 >> 8) 2^-24 of counter (0, 0, 1, 0).
void orc_philox4x32_10(uint64_t seed, uint64_t ctr_lo, uint64_t ctr_hi, uint32_t out[4]) {
  uint32_t c0 = (uint32_t)ctr_lo, c1 = (uint32_t)(ctr_lo >> 32), c2 = (uint32_t)ctr_hi, c3 = (uint32_t)(ctr_hi >> 32);
  uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
  for (int r = 0; r < 10; ++r) {
    const uint64_t p0 = (uint64_t)0xD2511F53u * c0;
    const uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
    const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
    const uint32_t n1 = (uint32_t)p1;
    const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
    const uint32_t n3 = (uint32_t)p0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

double orc_normal(uint64_t seed, uint64_t voxel) {
  uint32_t r[4];
  orc_philox4x32_10(seed, voxel >> 2, 0, r);
  const int p = (int)((voxel >> 1) & 1);
  const double u1 = ((double)(r[2 * p] >> 8) + 0.5) / 16777216.0;
  const double u2 = ((double)(r[2 * p + 1] >> 8) + 0.5) / 16777216.0;
  const double R = std::sqrt(-2.0 * std::log(u1));
  return (voxel & 1) ? R * std::sin(2.0 * kPi * u2) : R * std::cos(2.0 * kPi * u2);
}

double orc_noise_gamma(const orc_config *c) {
  if (c->noise_gamma_mode == 0) return 1.0;
  uint32_t r[4];
  orc_philox4x32_10(c->seed, 0, 1, r);
  return (double)(r[0] >> 8) / 16777216.0;
}

void orc_noise(const orc_config *c, int64_t nvox, double *cube) {
  const double gamma = orc_noise_gamma(c);
  for (int64_t i = 0; i < nvox; ++i)
    cube[i] += gamma * (c->noise_mu + c->noise_sigma * orc_normal(c->seed, (uint64_t)i));
}

// ---------------------------------------------------------------------------------------------
// Whole path (stage list PAPER.md:467): level balance -> coefficients -> transfer (total + continuum)
// -> continuum subtraction + units -> beam -> noise.  cube[ny][nx][nv].
// stage_mask bit 0: apply beam (if fwhm > 0); bit 1: apply noise (if configured).
void orc_observe(const orc_config *c, const float *nH2, const float *Tgas, const float *Tdust,
                 const float *vlos, int stage_mask, double *cube) {
  const int64_t plane = (int64_t)c->nx * c->ny, ncell = plane * c->nz;
  std::vector<double> coef(5 * ncell);
  orc_coefficients(c, ncell, nH2, Tgas, Tdust, nullptr, coef.data());
#pragma omp parallel for schedule(dynamic, 4)
  for (int64_t p = 0; p < plane; ++p) {
    std::vector<double> It(c->nv);
    if (c->dust_per_channel) {
      std::vector<double> Icv(c->nv);
      orc_march_column_perchannel(c, coef.data(), vlos, Tdust, p, It.data(), Icv.data());
      for (int v = 0; v < c->nv; ++v)
        cube[p * c->nv + v] = orc_convert_voxel_nu(c, orc_channel_frequency(c, v), It[v], Icv[v]);
      continue;
    }
    double Ic;
    orc_march_column(c, coef.data(), vlos, p, It.data(), &Ic);
    for (int v = 0; v < c->nv; ++v) cube[p * c->nv + v] = orc_convert_voxel(c, It[v], Ic);
  }
  if ((stage_mask & 1) && c->beam_fwhm_px > 0.0) {
    std::vector<double> tmp(cube, cube + plane * c->nv);
    orc_beam(c->ny, c->nx, c->nv, c->beam_fwhm_px, tmp.data(), cube);
  }
  if ((stage_mask & 2) && (c->noise_sigma != 0.0 || c->noise_mu != 0.0)) orc_noise(c, plane * c->nv, cube);
}

// ---------------------------------------------------------------------------------------------
// Brute-force pin (SURVEY 8(c) pin 8): monochromatic RTE, Eq. 3.1.2 with the POINT
// profile Eq. 3.3.3, solved exactly per cell (coefficients constant in a cell) at nsub frequencies
// per channel (midpoints), then channel-averaged, Eq. 4.4.2.  Not the method: the
// method applies the channel-AVERAGED profile inside the step (reading R1); the two agree as tau -> 0.
void orc_brute_column(const orc_config *c, const double *coef, const float *vlos, int64_t pix, int nsub,
                      double *I_avg /*[nv]*/) {
  const int64_t plane = (int64_t)c->nx * c->ny, ncell = plane * c->nz;
  const double h = c->cell_cm;
  const double Ibg = orc_planck(c->nu0_Hz, c->T_cmb);
  for (int v = 0; v < c->nv; ++v) {
    double acc = 0.0;
    for (int s = 0; s < nsub; ++s) {
      const double vel = c->v0_cms + (v - 0.5) * c->dv_cms + (s + 0.5) * c->dv_cms / nsub;
      double I = Ibg;
      for (int k = 0; k < c->nz; ++k) {
        const int64_t cell = (int64_t)k * plane + pix;
        const double phi = orc_phi_point(c, vel, (double)vlos[cell], coef[2 * ncell + cell]);
        const double ad = coef[3 * ncell + cell];
        I = formal_step(I, coef[cell] * phi + ad * coef[4 * ncell + cell], coef[ncell + cell] * phi + ad, h);
      }
      acc += I;
    }
    I_avg[v] = acc / nsub;
  }
}

// ---------------------------------------------------------------------------------------------
// O10  Gradient of L = sum_voxels w * cube(noise-free, beam-convolved) with respect to n_H2.
//
// (a) Finite differences (the definition): central differences with relative step eps on the listed
// cells, in whatever transfer mode / integration / velocity grid the configuration names (the column goes through
// the march of that mode).  Only the column holding the cell changes and the beam is linear, so L changes by
// sum_v what[pixel][v] * d(cube_raw[pixel][v]) with what = G^T w (beam adjoint = same symmetric
// zero-padded convolution, reading S20); `what` is computed by the caller with orc_beam.
static void raw_column(const orc_config *c, const float *nH2, const float *Tgas, const float *Tdust,
                       const float *vlos, int64_t pix, int64_t cell_mod, double n_mod, double *out,
                       double x_mod = 1.0 /* factor on the tracer abundance of cell_mod */) {
  const int64_t plane = (int64_t)c->nx * c->ny;
  const double h = c->cell_cm;
  const double Ibg = orc_planck(c->nu0_Hz, c->T_cmb);
  std::vector<double> It(c->nv, Ibg);
  double Ic = Ibg;
  if (c->transfer_mode != 0 || c->integration != 0 || c->subsample != 0) {
    // the other transfer / integration modes: the column's coefficients as a one-pixel cube through the march of O6b
    orc_config c1 = *c;
    c1.nx = 1; c1.ny = 1;
    std::vector<double> coef((size_t)5 * c->nz);
    std::vector<float> vl(c->nz);
    for (int k = 0; k < c->nz; ++k) {
      const int64_t cell = (int64_t)k * plane + pix;
      const double n = cell == cell_mod ? n_mod : (double)nH2[cell];
      double x[32], o[5];
      orc_levelpop_cell(c, n, (double)Tgas[cell], x);
      orc_cell_coefficients(c, n, (double)Tgas[cell], (double)Tdust[cell], x, o);
      if (cell == cell_mod) { o[0] *= x_mod; o[1] *= x_mod; }
      for (int q = 0; q < 5; ++q) coef[(size_t)q * c->nz + k] = o[q];
      vl[k] = vlos[cell];
    }
    march_column_modes(&c1, coef.data(), vl.data(), 0, It.data(), &Ic);
    for (int v = 0; v < c->nv; ++v) out[v] = orc_convert_voxel(c, It[v], Ic);
    return;
  }
  for (int k = 0; k < c->nz; ++k) {
    const int64_t cell = (int64_t)k * plane + pix;
    const double n = cell == cell_mod ? n_mod : (double)nH2[cell];
    double x[32], o[5];
    orc_levelpop_cell(c, n, (double)Tgas[cell], x);
    orc_cell_coefficients(c, n, (double)Tgas[cell], (double)Tdust[cell], x, o);
    if (cell == cell_mod) { o[0] *= x_mod; o[1] *= x_mod; }      // j0, kappa0 are linear in the abundance (Eq. 4.2.1)
    for (int v = 0; v < c->nv; ++v) {
      const double pb = orc_phibar(c, v, (double)vlos[cell], o[2]);
      It[v] = formal_step(It[v], o[0] * pb + o[3] * o[4], o[1] * pb + o[3], h);
    }
    Ic = formal_step(Ic, o[3] * o[4], o[3], h);
  }
  for (int v = 0; v < c->nv; ++v) out[v] = orc_convert_voxel(c, It[v], Ic);
}

void orc_grad_fd(const orc_config *c, const float *nH2, const float *Tgas, const float *Tdust,
                 const float *vlos, const double *what /*[ny][nx][nv]*/, int64_t nprobe,
                 const int64_t *cells, double eps, double *grad /*[nprobe]*/) {
  const int64_t plane = (int64_t)c->nx * c->ny;
#pragma omp parallel for schedule(dynamic, 1)
  for (int64_t q = 0; q < nprobe; ++q) {
    const int64_t cell = cells[q], pix = cell % plane;
    const double n0 = (double)nH2[cell], dn = eps * n0;
    std::vector<double> a(c->nv), b(c->nv);
    raw_column(c, nH2, Tgas, Tdust, vlos, pix, cell, n0 + dn, a.data());
    raw_column(c, nH2, Tgas, Tdust, vlos, pix, cell, n0 - dn, b.data());
    double s = 0.0;
    for (int v = 0; v < c->nv; ++v) s += what[pix * c->nv + v] * (a[v] - b[v]);
    grad[q] = s / (2.0 * dn);
  }
}

// (a') Abundance-only gradient ("abundance-only differentiability"): dL / d ln X_c for a per-cell factor on
// the tracer abundance, by central differences (the level fractions do not depend on the abundance: Eq. 4.2.1).
void orc_grad_fd_abundance(const orc_config *c, const float *nH2, const float *Tgas, const float *Tdust,
                           const float *vlos, const double *what, int64_t nprobe, const int64_t *cells, double eps,
                           double *grad) {
  const int64_t plane = (int64_t)c->nx * c->ny;
#pragma omp parallel for schedule(dynamic, 1)
  for (int64_t q = 0; q < nprobe; ++q) {
    const int64_t cell = cells[q], pix = cell % plane;
    std::vector<double> a(c->nv), b(c->nv);
    raw_column(c, nH2, Tgas, Tdust, vlos, pix, cell, (double)nH2[cell], a.data(), 1.0 + eps);
    raw_column(c, nH2, Tgas, Tdust, vlos, pix, cell, (double)nH2[cell], b.data(), 1.0 - eps);
    double s = 0.0;
    for (int v = 0; v < c->nv; ++v) s += what[pix * c->nv + v] * (a[v] - b[v]);
    grad[q] = s / (2.0 * eps);
  }
}

// (b) Analytic reverse-scan adjoint in float64, for out_unit = T_RJ or I with
// intensity-space subtraction.  Used to pin (a) against itself on every cell of a small cube and as
// the dense reference for the GPU adjoint.  grad[ncell].
//   forward:  I_{k+1} = I_k e^-tau + j h w(tau)
//   dI_{k+1}/dalpha = h [ -I_k e^-tau + j h w'(tau) ],  w'(tau) = (e^-tau (1 + tau) - 1) / tau^2
//   dI_{k+1}/dj     = h w(tau)
//   lambda_k = lambda_{k+1} e^-tau,  lambda_nz = scale * what
//   chain: dj0/dn = j0/n + (h nu0 / 4 pi) X n A dx_u/dn (same for kappa0), M dx/dn = -M_col x with the
//   conservation row zeroed on the right-hand side; d alpha_d / dn = kappa mass_per_H2.
static double wprime_of_tau(double tau) {
  if (std::fabs(tau) < 1e-4) return -0.5 + tau / 3.0 - tau * tau / 8.0;
  return (std::exp(-tau) * (1.0 + tau) - 1.0) / (tau * tau);
}

// (b') Reverse-mode derivative of total_point in the optically thick mode (transfer_mode 0), formal or smooth: one spectral
// point with profile weights p[n], adjoint seed lam_out = dL / dI_observer.  Adds dL/dj0_n, dL/dkappa0_n, dL/dalpha_d,n
// to gj, gk, gad.  Written as the chain rule applied to the formulas of total_point, statement by statement:
//   formal  I_n+1 = I_n e^-tau + jT h w(tau):  as in (b)
//   BDF2    y_n = relu(N_n / D_n),  N_n = 2 h jT_n + 4 y_n-1 - y_n-2,  D_n = 3 + 2 h aT_n           (Eq. 4.8.10)
//           u = lam_n / D_n where N_n / D_n > 0, else 0 (ReLU):  dL/djT_n = 2 h u,  dL/daT_n = -2 h u y_n,
//           lam_n-1 += 4 u,  lam_n-2 -= u
//   TR      y_1 = relu(N_1 / D_1),  N_1 = h (jT_0 + jT_1) + (2 - h aT_0) y_0,  D_1 = 2 + h aT_1        (Eq. 4.8.12)
//           u = lam_1 / D_1:  dL/djT_0 = dL/djT_1 = h u,  dL/daT_0 = -h u y_0,  dL/daT_1 = -h u y_1   (y_0 = I_bg is fixed)
//   jT = j0 p + alpha_d S_d,  aT = kappa0 p + alpha_d  (Eq. 4.8.6 - 4.8.7)
static void total_point_adjoint(const orc_config *c, int R, const double *p, const double *j0, const double *k0,
                                const double *ad, const double *Sd, double Ibg, double lam_out, double *gj, double *gk,
                                double *gad) {
  const double h = c->cell_cm;
  auto jT = [&](int n) { return j0[n] * p[n] + ad[n] * Sd[n]; };
  auto aT = [&](int n) { return k0[n] * p[n] + ad[n]; };
  auto spread = [&](int n, double dLdj, double dLda) {
    gj[n] += dLdj * p[n];
    gk[n] += dLda * p[n];
    gad[n] += dLda + Sd[n] * dLdj;
  };
  if (c->integration == 0) {
    std::vector<double> I(R + 1);
    I[0] = Ibg;
    for (int n = 0; n < R; ++n) I[n + 1] = formal_step(I[n], jT(n), aT(n), h);
    double lam = lam_out;
    for (int n = R - 1; n >= 0; --n) {
      const double tau = aT(n) * h, e = std::exp(-tau);
      spread(n, lam * h * w_of_tau(tau), lam * h * (-I[n] * e + jT(n) * h * wprime_of_tau(tau)));
      lam *= e;
    }
    return;
  }
  if (R < 2) return;                                   // total_point returns I_bg: no dependence on the cells
  std::vector<double> y(R), yu(R), lam(R, 0.0);
  y[0] = yu[0] = Ibg;
  yu[1] = (h * (jT(0) + jT(1)) + (2.0 - h * aT(0)) * y[0]) / (2.0 + h * aT(1));
  y[1] = relu(yu[1]);
  for (int n = 2; n < R; ++n) {
    yu[n] = (2.0 * h * jT(n) + 4.0 * y[n - 1] - y[n - 2]) / (3.0 + 2.0 * h * aT(n));
    y[n] = relu(yu[n]);
  }
  lam[R - 1] = lam_out;
  for (int n = R - 1; n >= 2; --n) {
    if (!(yu[n] > 0.0)) continue;                      // the ReLU passes nothing
    const double u = lam[n] / (3.0 + 2.0 * h * aT(n));
    spread(n, 2.0 * h * u, -2.0 * h * u * y[n]);
    lam[n - 1] += 4.0 * u;
    lam[n - 2] -= u;
  }
  if (yu[1] > 0.0) {
    const double u = lam[1] / (2.0 + h * aT(1));
    spread(0, h * u, -h * u * y[0]);
    spread(1, h * u, -h * u * y[1]);
  }
}

// dL/dj0, dL/dkappa0, dL/dalpha_d of every cell of one column in the thick mode with the smooth integrator and / or the
// fine velocity grid (the configurations march_column_modes serves with transfer_mode = 0).  what[nv]: dL / d(cube_raw).
// The cube is scale (I_tot[v] - I_cont) with I_tot[v] the Simpson average of the fine points (Eq. 4.5.1), so the seed of a
// fine point is the sum over the channels it belongs to of scale what[v] (Simpson coefficient) / (3 m).
static void column_adjoint_modes(const orc_config *c, int R, const double *j0, const double *k0, const double *b,
                                 const double *ad, const double *Sd, const double *vl, const double *what, double scale,
                                 double *gj, double *gk, double *gad) {
  const double Ibg = orc_planck(c->nu0_Hz, c->T_cmb);
  std::vector<double> p(R), zero(R, 0.0);
  for (int n = 0; n < R; ++n) gj[n] = gk[n] = gad[n] = 0.0;
  double lamC = 0.0;
  for (int v = 0; v < c->nv; ++v) if (c->subtract_continuum) lamC -= scale * what[v];
  const int f = c->subsample;
  if (f == 0) {
    for (int v = 0; v < c->nv; ++v) {
      for (int n = 0; n < R; ++n) p[n] = orc_phibar(c, v, vl[n], b[n]);
      total_point_adjoint(c, R, p.data(), j0, k0, ad, Sd, Ibg, scale * what[v], gj, gk, gad);
    }
  } else {
    const int m = f + 1;
    const double dvf = c->dv_cms / m;
    for (int64_t q = 0; q <= (int64_t)c->nv * m; ++q) {
      double seed = 0.0;
      for (int64_t v = q / m - 1; v <= q / m; ++v) {     // a point on a channel edge belongs to both channels
        if (v < 0 || v >= c->nv) continue;
        const int64_t jq = q - v * m;                    // index of the point inside channel v: 0 .. m
        if (jq < 0 || jq > m) continue;
        const double simpson = (jq == 0 || jq == m) ? 1.0 : ((jq & 1) ? 4.0 : 2.0);
        seed += scale * what[v] * simpson / (3.0 * m);
      }
      const double vel = c->v0_cms - 0.5 * c->dv_cms + q * dvf;
      for (int n = 0; n < R; ++n) p[n] = orc_phi_point(c, vel, vl[n], b[n]);
      total_point_adjoint(c, R, p.data(), j0, k0, ad, Sd, Ibg, seed, gj, gk, gad);
    }
  }
  // the continuum is the same march with no line (continuum_column): p = 0
  total_point_adjoint(c, R, zero.data(), j0, k0, ad, Sd, Ibg, lamC, gj, gk, gad);
}

static void grad_adjoint_impl(const orc_config *c, const float *nH2, const float *Tgas, const float *Tdust,
                              const float *vlos, const double *what, double *grad, bool wrt_abundance) {
  const int64_t plane = (int64_t)c->nx * c->ny;
  const int N = c->n_levels, nz = c->nz, nv = c->nv;
  const double h = c->cell_cm;
  const double Ibg = orc_planck(c->nu0_Hz, c->T_cmb);
  const double scale = c->out_unit == 1 ? kC * kC / (2.0 * kK * c->nu0_Hz * c->nu0_Hz) : 1.0;
  const int u = c->line_upper, l = c->line_lower;
  const double A = c->einstein_A[u * N + l];
  const double Bul = kC * kC / (2.0 * kH * c->nu0_Hz * c->nu0_Hz * c->nu0_Hz) * A;
  const double Blu = c->weight[u] / c->weight[l] * Bul;
  const double pref = kH * c->nu0_Hz / (4.0 * kPi);
#pragma omp parallel for schedule(dynamic, 4)
  for (int64_t pix = 0; pix < plane; ++pix) {
    std::vector<double> co(5 * nz), It((int64_t)(nz + 1) * nv), Ic(nz + 1), lam(nv), xs(nz * N);
    for (int k = 0; k < nz; ++k) {
      const int64_t cell = (int64_t)k * plane + pix;
      orc_levelpop_cell(c, (double)nH2[cell], (double)Tgas[cell], &xs[k * N]);
      orc_cell_coefficients(c, (double)nH2[cell], (double)Tgas[cell], (double)Tdust[cell], &xs[k * N], &co[5 * k]);
    }
    std::vector<double> gj(nz, 0.0), gk(nz, 0.0), gad(nz, 0.0);
    const bool hot = c->transfer_mode == 0 && c->integration == 0 && c->subsample == 0;
    if (!hot) {
      // thick mode with the smooth integrator and / or the fine grid: (b').  The other transfer modes have no analytic
      // adjoint here (finite differences (a) serve them): NaN.
      std::vector<double> a0(nz), a1(nz), a2(nz), a3(nz), a4(nz), vl(nz);
      for (int k = 0; k < nz; ++k) {
        a0[k] = co[5 * k]; a1[k] = co[5 * k + 1]; a2[k] = co[5 * k + 2]; a3[k] = co[5 * k + 3]; a4[k] = co[5 * k + 4];
        vl[k] = (double)vlos[(int64_t)k * plane + pix];
      }
      if (c->transfer_mode == 0)
        column_adjoint_modes(c, nz, a0.data(), a1.data(), a2.data(), a3.data(), a4.data(), vl.data(), what + pix * nv, scale,
                             gj.data(), gk.data(), gad.data());
      else
        for (int k = 0; k < nz; ++k) gj[k] = gk[k] = gad[k] = std::nan("");
    }
    for (int v = 0; v < nv; ++v) It[v] = Ibg;
    Ic[0] = Ibg;
    for (int k = 0; hot && k < nz; ++k) {
      const int64_t cell = (int64_t)k * plane + pix;
      const double *o = &co[5 * k];
      for (int v = 0; v < nv; ++v) {
        const double pb = orc_phibar(c, v, (double)vlos[cell], o[2]);
        It[(int64_t)(k + 1) * nv + v] = formal_step(It[(int64_t)k * nv + v], o[0] * pb + o[3] * o[4], o[1] * pb + o[3], h);
      }
      Ic[k + 1] = formal_step(Ic[k], o[3] * o[4], o[3], h);
    }
    double lamC = 0.0;   // adjoint of the continuum: -sum_v lambda (subtraction), if enabled
    for (int v = 0; v < nv; ++v) { lam[v] = scale * what[pix * nv + v]; if (c->subtract_continuum) lamC -= lam[v]; }
    for (int k = nz - 1; k >= 0; --k) {
      const int64_t cell = (int64_t)k * plane + pix;
      const double *o = &co[5 * k];
      double g_j0 = gj[k], g_k0 = gk[k], g_ad = gad[k];
      for (int v = 0; hot && v < nv; ++v) {
        const double pb = orc_phibar(c, v, (double)vlos[cell], o[2]);
        const double al = o[1] * pb + o[3], j = o[0] * pb + o[3] * o[4], tau = al * h, e = std::exp(-tau);
        const double dIda = h * (-It[(int64_t)k * nv + v] * e + j * h * wprime_of_tau(tau));
        const double dIdj = h * w_of_tau(tau);
        g_k0 += lam[v] * dIda * pb;
        g_j0 += lam[v] * dIdj * pb;
        g_ad += lam[v] * (dIda + o[4] * dIdj);
        lam[v] *= e;
      }
      if (hot) {  // continuum branch
        const double tau = o[3] * h, e = std::exp(-tau), j = o[3] * o[4];
        const double dIda = h * (-Ic[k] * e + j * h * wprime_of_tau(tau));
        g_ad += lamC * (dIda + o[4] * h * w_of_tau(tau));
        lamC *= e;
      }
      // chain through the level balance: M dx = -(dM/dn) x, conservation row: sum dx = 0
      const double n = (double)nH2[cell], T = (double)Tgas[cell];
      std::vector<double> M(N * N), M1(N * N), rhs(N, 0.0), dx(N);
      orc_balance_matrix(c, n, T, M.data());
      // dM/dn: the balance matrix is affine in n; difference of two evaluations is exact up to rounding
      orc_balance_matrix(c, 2.0 * n, T, M1.data());
      const double *x = &xs[k * N];
      for (int i = 1; i < N; ++i) {
        double s = 0.0;
        for (int jx = 0; jx < N; ++jx) s += (M1[i * N + jx] - M[i * N + jx]) / n * x[jx];
        rhs[i] = -s;
      }
      for (int jx = 0; jx < N; ++jx) M[jx] = 1.0;
      rhs[0] = 0.0;
      solve_ge(N, M.data(), rhs.data(), dx.data());
      const double X = c->abundance;
      double dj0 = pref * X * A * (x[u] + n * dx[u]);
      double dk0 = pref * X * ((x[l] + n * dx[l]) * Blu - (x[u] + n * dx[u]) * Bul);
      if (T > c->T_inf) { dj0 = 0.0; dk0 = 0.0; }
      const double dad = c->dust_on ? c->kappa_gas_cm2_g * c->mass_per_H2_g : 0.0;
      grad[cell] = wrt_abundance ? g_j0 * co[5 * k] + g_k0 * co[5 * k + 1]      // d / d ln X_c: j0, kappa0 linear in X
                                 : g_j0 * dj0 + g_k0 * dk0 + g_ad * dad;
    }
  }
}

void orc_grad_adjoint(const orc_config *c, const float *nH2, const float *Tgas, const float *Tdust,
                      const float *vlos, const double *what, double *grad) {
  grad_adjoint_impl(c, nH2, Tgas, Tdust, vlos, what, grad, false);
}

void orc_grad_adjoint_abundance(const orc_config *c, const float *nH2, const float *Tgas, const float *Tdust,
                                const float *vlos, const double *what, double *grad) {
  grad_adjoint_impl(c, nH2, Tgas, Tdust, vlos, what, grad, true);
}

// ---------------------------------------------------------------------------------------------
// O11  Density tracing ("simple observation", section 5.10): "a projection of column density per
// unit velocity over dimensions of longitude, latitude, and velocity".  Reading S28: every cell adds its
// column density n_H2 h to the channel that contains its line-of-sight velocity (channel k covers
// [v0 + (k - 1/2) dv, v0 + (k + 1/2) dv)), cells outside the band add nothing, and the cube is that sum divided by
// the channel width: cube[ny][nx][nv] in cm^-2 per (cm/s).
void orc_density_trace(const orc_config *c, const float *nH2, const float *vlos, double *cube) {
  const int64_t plane = (int64_t)c->nx * c->ny;
  for (int64_t i = 0; i < plane * c->nv; ++i) cube[i] = 0.0;
  for (int k = 0; k < c->nz; ++k)
    for (int64_t p = 0; p < plane; ++p) {
      const int64_t cell = (int64_t)k * plane + p;
      const double pos = ((double)vlos[cell] - c->v0_cms) / c->dv_cms + 0.5;
      const double fl = std::floor(pos);
      if (fl < 0.0 || fl >= (double)c->nv) continue;
      cube[p * c->nv + (int64_t)fl] += (double)nH2[cell] * c->cell_cm / c->dv_cms;
    }
}

// O12  Error metrics of section 5.1.  T1, T2: cubes [ny][nx][nv] (l = x, b = y).
//   TSRE(T1, T2) = 2 |T1 - T2| / (|T1| + |T2|) if min(|T1|, |T2|) > T_min, else 0             Eq. 5.1.1
//   mean-TSRE_lbv = mean over all voxels; mean-TSRE_lb / _lv = mean over the pixels of the images obtained by
//   averaging each cube over v / over b first (Eq. 5.1.2 - 5.1.3; reading G8: both arguments of TSRE_lv are l-v
//   images; reading S29: the means run over ALL elements, inactive ones counting 0, as the equations are written)
//   TAM(T) = mean of T over the voxels with |T| > T_min                                        Eq. 5.1.4 - 5.1.5
// out = { TSRE_lbv, TSRE_lb, TSRE_lv, TAM(T1), TAM(T2), max T1, max T2, active(T1), active(T2) }; TAM of a cube with
// no active voxel is 0.
static double tsre(double a, double b, double Tmin) {
  const double fa = std::fabs(a), fb = std::fabs(b);
  return (fa > Tmin && fb > Tmin) ? 2.0 * std::fabs(a - b) / (fa + fb) : 0.0;
}

void orc_metrics(int ny, int nx, int nv, const double *T1, const double *T2, double Tmin, double *out) {
  const int64_t plane = (int64_t)ny * nx, nvox = plane * nv;
  double s_lbv = 0.0, tam1 = 0.0, tam2 = 0.0, mx1 = -INFINITY, mx2 = -INFINITY;
  int64_t n1 = 0, n2 = 0;
  for (int64_t i = 0; i < nvox; ++i) {
    s_lbv += tsre(T1[i], T2[i], Tmin);
    if (std::fabs(T1[i]) > Tmin) { tam1 += T1[i]; ++n1; }
    if (std::fabs(T2[i]) > Tmin) { tam2 += T2[i]; ++n2; }
    mx1 = std::max(mx1, T1[i]); mx2 = std::max(mx2, T2[i]);
  }
  double s_lb = 0.0;
  for (int64_t p = 0; p < plane; ++p) {
    double a = 0.0, b = 0.0;
    for (int v = 0; v < nv; ++v) { a += T1[p * nv + v]; b += T2[p * nv + v]; }
    s_lb += tsre(a / nv, b / nv, Tmin);
  }
  double s_lv = 0.0;
  for (int x = 0; x < nx; ++x)
    for (int v = 0; v < nv; ++v) {
      double a = 0.0, b = 0.0;
      for (int y = 0; y < ny; ++y) { a += T1[((int64_t)y * nx + x) * nv + v]; b += T2[((int64_t)y * nx + x) * nv + v]; }
      s_lv += tsre(a / ny, b / ny, Tmin);
    }
  out[0] = s_lbv / (double)nvox; out[1] = s_lb / (double)plane; out[2] = s_lv / ((double)nx * nv);
  out[3] = n1 ? tam1 / (double)n1 : 0.0; out[4] = n2 ? tam2 / (double)n2 : 0.0;
  out[5] = mx1; out[6] = mx2; out[7] = (double)n1; out[8] = (double)n2;
}

}  // extern "C"
