// Host side of the C ABI declared in include/iris_so.h: configuration, constant folding (in double),
// scratch management and kernel launches.  Every step of the path runs in the kernels of this directory;
// there is no CPU fallback.
#include "../../include/iris_so.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "cell_kernels.cuh"
#include "post_kernels.cuh"
#include "transfer_dense.cuh"
#include "transfer_window.cuh"
#include "transfer_series.cuh"
#include "transfer_modes.cuh"
#include "transfer_smooth.cuh"
#include "adjoint_kernels.cuh"
#include "adjoint_modes.cuh"
#include "diagnostics.cuh"

// Scratch of iris_so_observe_raw_static (the entry point that allocates nothing): the six coefficient planes of at most
// IRIS_SO_STATIC_MAX_CELLS cells, 12 MiB on every GPU that loads the library.  In HOST code this name is a host-side
// stand-in, not a device address: static_scratch_of_device() resolves it with cudaGetSymbolAddress once per device and
// the kernels are given that pointer.
static __device__ __align__(256) float g_static_coef[6 * (size_t)IRIS_SO_STATIC_MAX_CELLS];

namespace {

// CODATA-2018 exact SI values in CGS (this translation unit's own copy).
constexpr double H_PLANCK = 6.62607015e-27;
constexpr double K_BOLTZ = 1.380649e-16;
constexpr double C_LIGHT = 2.99792458e10;
constexpr double PI = 3.14159265358979323846;

thread_local std::string g_create_error;

}  // namespace

struct iris_so_ctx {
  iris_so_config cfg;
  std::vector<double> energy, weight, A, Kd;
  std::vector<double> Keff;     // tabulated rates folded over the partners: [nT][N*N] per unit n_H2 (empty: power law)
  std::vector<double> Tgrid;
  float* d_colltab = nullptr;   // device copy: nT temperatures, then nT * kMaxPairs float2 {K, K g_u/g_l} * rate_scale
  float* d_grid = nullptr;      // coefficient grid (coef_grid = 1): node tables, node values, cell coefficients
  iris::GridConsts gc;
  iris::LevelConsts lc;
  iris::CoefConsts cc;
  iris::MarchConsts mc;
  iris::BeamConsts bc;
  iris::NoiseConsts nc;
  iris::AdjointConsts ac;
  int band = 1;                 // largest u - l with a non-zero radiative or collisional rate
  int device = 0, sm_count = 0;
  int64_t ncell = 0, npix = 0, nvox = 0;
  float* d_coef = nullptr;      // [6][ncell]
  float* d_tmp = nullptr;       // cube-sized temporary (beam)
  float* d_stage = nullptr;     // host-path staging: 4 fields + cube
  float* d_adj = nullptr;       // adjoint scratch
  size_t adj_bytes = 0;
  uint64_t scratch_bytes = 0;
  uint64_t launches = 0;
  std::string err;
  // optional per-stage timing (iris_so_profile)
  struct ProfRec { int stage; uint64_t launches; cudaEvent_t a, b; };
  bool profiling = false;
  std::vector<ProfRec> recs;
  std::vector<cudaEvent_t> event_pool;
  unsigned long long* d_counter = nullptr;
  int* d_gate = nullptr;          // [0] pixels transfer_smooth_window_kernel handed over to the dense kernel (zeroed per launch),
                                  // [1] their number accumulated over the launches of one public call (slabs of the host path),
                                  // [2 ..] the list of those pixels (npix entries)
  double* d_metrics = nullptr;
  // reachable-range spectra of the series kernel (transfer_series.cuh, CIRC): used while few pixels have to be handed over
  bool circ_ok = true;
  int* h_hand = nullptr;          // pinned: pixels handed over by the last launch that used them
  cudaEvent_t ev_hand = nullptr;  // recorded after the copy into h_hand
  bool hand_pending = false;
  int64_t hand_npix = 0;          // pixels of that launch
  float* d_static_coef = nullptr;   // device address of g_static_coef on ctx->device (nullptr: static_err says why)
  std::string static_err;
  cudaStream_t s_in = nullptr, s_out = nullptr;      // copy streams of the host-buffer path
  std::vector<cudaEvent_t> slab_events;
};

namespace {

iris_so_status fail(iris_so_ctx* ctx, iris_so_status s, const std::string& msg) {
  if (ctx) ctx->err = msg; else g_create_error = msg;
  return s;
}

iris_so_status cuda_fail(iris_so_ctx* ctx, cudaError_t e, const char* what) {
  char buf[512];
  snprintf(buf, sizeof buf, "%s: %s", what, cudaGetErrorString(e));
  return fail(ctx, e == cudaErrorMemoryAllocation ? IRIS_SO_ENOMEM : IRIS_SO_ECUDA, buf);
}

#define IRIS_CHECK_LAUNCH(ctx, name)                                         \
  do {                                                                       \
    (ctx)->launches++;                                                       \
    cudaError_t e_ = cudaGetLastError();                                     \
    if (e_ != cudaSuccess) return cuda_fail((ctx), e_, "launch of " name);   \
  } while (0)

iris_so_status ensure(iris_so_ctx* ctx, float** p, size_t bytes, const char* what) {
  if (*p) return IRIS_SO_OK;
  cudaError_t e = cudaMalloc(reinterpret_cast<void**>(p), bytes);
  if (e != cudaSuccess) { *p = nullptr; cudaGetLastError(); return cuda_fail(ctx, e, what); }
  ctx->scratch_bytes += bytes;
  return IRIS_SO_OK;
}

// Device address of g_static_coef on device `dev`, which must be current: resolved once per device (the symbol has one
// instance per device that loads the module).  Returns nullptr and the reason in *err when the runtime refuses.
float* static_scratch_of_device(int dev, std::string* err) {
  constexpr int kMaxDev = 64;
  static std::mutex mu;
  static float* ptr[kMaxDev] = {};
  static bool tried[kMaxDev] = {};
  static std::string why[kMaxDev];
  if (dev < 0 || dev >= kMaxDev) { *err = "device index beyond the table of static scratch addresses"; return nullptr; }
  std::lock_guard<std::mutex> lock(mu);
  if (!tried[dev]) {
    tried[dev] = true;
    void* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, g_static_coef);
    if (e != cudaSuccess) {
      cudaGetLastError();
      why[dev] = std::string("cudaGetSymbolAddress(static scratch): ") + cudaGetErrorString(e);
    } else {
      ptr[dev] = static_cast<float*>(p);
    }
  }
  if (!ptr[dev]) *err = why[dev];
  return ptr[dev];
}

// Brackets the kernels a stage launches with two events on the caller's stream when profiling is on.
struct ProfScope {
  iris_so_ctx* ctx; cudaStream_t st; int stage; uint64_t l0; cudaEvent_t a = nullptr;
  ProfScope(iris_so_ctx* c, int stage_, cudaStream_t s) : ctx(c), st(s), stage(stage_), l0(c->launches) {
    if (!ctx->profiling) return;
    a = take(); if (a) cudaEventRecord(a, st);
  }
  ~ProfScope() {
    if (!a) return;
    cudaEvent_t b = take();
    if (!b) return;
    cudaEventRecord(b, st);
    ctx->recs.push_back({stage, ctx->launches - l0, a, b});
  }
  cudaEvent_t take() {
    if (!ctx->event_pool.empty()) { cudaEvent_t e = ctx->event_pool.back(); ctx->event_pool.pop_back(); return e; }
    cudaEvent_t e = nullptr;
    if (cudaEventCreate(&e) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    return e;
  }
};

void prof_reset(iris_so_ctx* ctx) {
  for (auto& r : ctx->recs) { ctx->event_pool.push_back(r.a); ctx->event_pool.push_back(r.b); }
  ctx->recs.clear();
}

double planck_krj(double hnu_k, double T) { return T > 0.0 ? hnu_k / std::expm1(hnu_k / T) : 0.0; }

void host_philox(uint64_t seed, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t out[4]) {
  uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
  for (int r = 0; r < 10; ++r) {
    const uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
    const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
    c0 = n0; c1 = (uint32_t)p1; c2 = n2; c3 = (uint32_t)p0;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

iris_so_status validate(const iris_so_config* c, std::string& why) {
  auto bad = [&](const char* m) { why = m; return IRIS_SO_EINVAL; };
  if (!c) return bad("config is NULL");
  if (c->nx < 1 || c->ny < 1 || c->nz < 1) return bad("grid dimensions must be >= 1");
  if ((int64_t)c->nx * c->ny * c->nz > (int64_t)1 << 30) return bad("grid too large (> 2^30 cells)");
  if (!(c->cell_cm > 0.0)) return bad("cell_cm must be > 0");
  if (c->n_levels < 2 || c->n_levels > IRIS_SO_MAX_LEVELS) return bad("n_levels must be in [2, 10]");
  if (!c->energy_K || !c->weight || !c->einstein_A || !c->coll_down_ref) return bad("molecule arrays must not be NULL");
  const int N = c->n_levels;
  for (int i = 0; i < N; ++i) {
    if (!(c->weight[i] > 0.0)) return bad("statistical weights must be > 0");
    if (i > 0 && !(c->energy_K[i] > c->energy_K[i - 1])) return bad("energy_K must be strictly ascending");
  }
  for (int u = 0; u < N; ++u) {
    double down = 0.0;
    for (int l = 0; l < N; ++l) {
      const double a = c->einstein_A[u * N + l], k = c->coll_n_partners > 0 ? 0.0 : c->coll_down_ref[u * N + l];
      if (l >= u && (a != 0.0 || k != 0.0)) return bad("einstein_A / coll_down_ref must be 0 for u <= l");
      if (a < 0.0 || k < 0.0 || !std::isfinite(a) || !std::isfinite(k)) return bad("rates must be finite and >= 0");
      down += a + k;
    }
    if (u > 0 && !(down > 0.0) && c->coll_n_partners == 0) return bad("every excited level needs a downward rate");
  }
  if (!(c->coll_T_ref > 0.0)) return bad("coll_T_ref must be > 0");
  if (c->line_upper <= c->line_lower || c->line_lower < 0 || c->line_upper >= N) return bad("bad line levels");
  if (!(c->einstein_A[c->line_upper * N + c->line_lower] > 0.0)) return bad("observed line has no Einstein A");
  if (!(c->nu0_Hz > 0.0) || !(c->mol_mass_g > 0.0)) return bad("nu0_Hz and mol_mass_g must be > 0");
  if (!(c->abundance >= 0.0) || !(c->microturb_cms >= 0.0)) return bad("abundance and microturb_cms must be >= 0");
  if (!(c->T_bar >= 0.0) || !(c->T_cmb >= 0.0)) return bad("T_bar and T_cmb must be >= 0");
  if (std::isnan(c->T_inf)) return bad("T_inf is NaN");
  if (c->dust_on && (!(c->kappa_gas_cm2_g >= 0.0) || !(c->mass_per_H2_g > 0.0))) return bad("bad dust parameters");
  if (c->nv < 1 || c->nv > 65536) return bad("nv must be in [1, 65536]");
  if (!(c->dv_cms > 0.0) || !std::isfinite(c->v0_cms)) return bad("bad channel grid");
  if (c->subtract_space < 0 || c->subtract_space > 1 || c->out_unit < 0 || c->out_unit > 2) return bad("bad output mode");
  if (c->subtract_continuum && c->subtract_space == 1 && c->out_unit != 2)
    return bad("Planck-space subtraction yields Kelvin: out_unit must be 2");
  if (!(c->beam_fwhm_px >= 0.0)) return bad("beam_fwhm_px must be >= 0");
  if (!(c->noise_sigma >= 0.0) || !std::isfinite(c->noise_mu)) return bad("bad noise parameters");
  if (c->noise_gamma_mode < 0 || c->noise_gamma_mode > 1) return bad("bad noise_gamma_mode");
  if (c->transfer_algo < 0 || c->transfer_algo > 3) return bad("bad transfer_algo");
  if (c->coll_n_partners < 0 || c->coll_n_partners > 8) return bad("coll_n_partners must be in [0, 8]");
  if (c->coll_n_partners > 0) {
    if (c->coll_nT < 1 || c->coll_nT > 64) return bad("coll_nT must be in [1, 64]");
    if (!c->coll_T_grid || !c->coll_table || !c->coll_partner_frac) return bad("collision table arrays must not be NULL");
    for (int t = 0; t < c->coll_nT; ++t)
      if (!(c->coll_T_grid[t] > 0.0) || (t > 0 && !(c->coll_T_grid[t] > c->coll_T_grid[t - 1])))
        return bad("coll_T_grid must be positive and strictly ascending");
    for (int p = 0; p < c->coll_n_partners; ++p)
      if (!(c->coll_partner_frac[p] >= 0.0) || !std::isfinite(c->coll_partner_frac[p])) return bad("bad coll_partner_frac");
    const int64_t nt = (int64_t)c->coll_n_partners * c->coll_nT * N * N;
    for (int64_t q = 0; q < nt; ++q) {
      const int ul = (int)(q % (N * N)), u = ul / N, l = ul % N;
      const double k = c->coll_table[q];
      if (k < 0.0 || !std::isfinite(k) || (l >= u && k != 0.0)) return bad("coll_table must be finite, >= 0 and 0 for u <= l");
    }
  }
  if (c->coef_grid < 0 || c->coef_grid > 1) return bad("coef_grid must be 0 or 1");
  if (c->coef_grid == 1) {
    if (c->grid_n_density < 2 || c->grid_n_density > 4096 || c->grid_n_temp < 2 || c->grid_n_temp > 4096)
      return bad("grid_n_density and grid_n_temp must be in [2, 4096]");
    if (!(c->grid_nH2_lo > 0.0) || !(c->grid_nH2_hi > c->grid_nH2_lo) || !std::isfinite(c->grid_nH2_hi) ||
        !(c->grid_T_lo > 0.0) || !(c->grid_T_hi > c->grid_T_lo) || !std::isfinite(c->grid_T_hi))
      return bad("grid bounds must satisfy 0 < lo < hi");
  }
  if (c->dust_per_channel < 0 || c->dust_per_channel > 1) return bad("dust_per_channel must be 0 or 1");
  if (c->transfer_mode < 0 || c->transfer_mode > 2) return bad("transfer_mode must be 0 (thick), 1 (selectively thin) or 2 (thin)");
  if (c->integration < 0 || c->integration > 1) return bad("integration must be 0 (formal) or 1 (smooth)");
  if (c->subsample < 0 || c->subsample > 255 || (c->subsample > 0 && c->subsample % 2 == 0))
    return bad("subsample must be 0 or an odd number of added midpoints per channel (<= 255)");
  if (c->subsample > 0 && c->transfer_mode != 0) return bad("subsample (fine velocity grid) applies to the thick mode only");
  return IRIS_SO_OK;
}

int out_mode_of(const iris_so_config& c) {
  if (c.subtract_continuum) {
    if (c.subtract_space == 1) return iris::OUT_TB_SUB;
    return c.out_unit == 1 ? iris::OUT_TRJ_SUB : c.out_unit == 0 ? iris::OUT_I_SUB : iris::OUT_TB_OF_SUB;
  }
  return c.out_unit == 1 ? iris::OUT_TRJ_TOT : c.out_unit == 0 ? iris::OUT_I_TOT : iris::OUT_TB_OF_TOT;
}

void fold_constants(iris_so_ctx* ctx) {
  const iris_so_config& c = ctx->cfg;
  const int N = c.n_levels;
  iris::LevelConsts& lc = ctx->lc;
  std::memset(&lc, 0, sizeof lc);
  ctx->band = 1;
  for (int u = 1; u < N; ++u)
    for (int l = 0; l < u; ++l)
      if ((ctx->A[u * N + l] != 0.0 || ctx->Kd[u * N + l] != 0.0) && u - l > ctx->band) ctx->band = u - l;
  for (int i = 1; i < N; ++i) lc.ndE2[i] = (float)(-(ctx->energy[i] - ctx->energy[i - 1]) * 1.4426950408889634);
  double Amax = 0.0;
  for (double a : ctx->A) Amax = std::max(Amax, a);
  const double rs = Amax > 0.0 ? 1.0 / Amax : 1.0;              // common rate scale (fractions are invariant)
  lc.rate_scale = (float)rs;
  for (int u = 1; u < N; ++u)
    for (int l = 0; l < u; ++l) {
      const int p = iris::pair_index(u, l);
      const double A = ctx->A[u * N + l], K = ctx->Kd[u * N + l];
      const double gr = ctx->weight[u] / ctx->weight[l];
      double ngam = 0.0;
      if (A > 0.0 && c.T_bar > 0.0) {
        const double hnu_k = ctx->energy[u] - ctx->energy[l];   // h nu_ul / k
        ngam = 1.0 / std::expm1(hnu_k / c.T_bar);               // photon occupation of B_nu(T_bar), Eq. 3.6.2
      }
      lc.pr[p].x = (float)(rs * K);                             // K_ul(T_ref)
      lc.pr[p].y = (float)(rs * A * (1.0 + ngam));              // A_ul + B_ul J
      lc.pr[p].z = (float)(rs * K * gr);                        // K_ul(T_ref) g_u / g_l
      lc.pr[p].w = (float)(rs * gr * A * ngam);                 // B_lu J
    }
  lc.inv_Tref = (float)(1.0 / c.coll_T_ref);
  lc.Texp = (float)c.coll_T_exp;

  const int u = c.line_upper, l = c.line_lower;
  const double nu = c.nu0_Hz, A = ctx->A[u * N + l];
  const double gr = ctx->weight[u] / ctx->weight[l];
  const double Bul = C_LIGHT * C_LIGHT / (2.0 * H_PLANCK * nu * nu * nu) * A;   // Eq. 3.7.1
  const double KRJ = C_LIGHT * C_LIGHT / (2.0 * K_BOLTZ * nu * nu);             // Eq. 4.9.2
  const double dnuW = nu * c.dv_cms / C_LIGHT;                                  // channel width in Hz
  const double pref = H_PLANCK * nu / (4.0 * PI) * c.abundance * c.cell_cm / (2.0 * dnuW);
  iris::CoefConsts& cc = ctx->cc;
  cc.upper = u; cc.lower = l; cc.gr = (float)gr;
  for (int i = 0; i < iris::kMaxLevels; ++i) { cc.pick_upper[i] = i == u ? 1.0f : 0.0f; cc.pick_lower[i] = i == l ? 1.0f : 0.0f; }
  cc.c_e = (float)(KRJ * pref * A);
  cc.c_a = (float)(pref * Bul);
  cc.c_d = c.dust_on ? (float)(c.kappa_gas_cm2_g * c.mass_per_H2_g * c.cell_cm) : 0.0f;
  cc.hnu_k = (float)(H_PLANCK * nu / K_BOLTZ);
  cc.c_b = (float)(2.0 * K_BOLTZ / c.mol_mass_g);
  cc.xi2 = (float)(c.microturb_cms * c.microturb_cms);
  cc.dv = (float)c.dv_cms; cc.inv_dv = (float)(1.0 / c.dv_cms); cc.v0 = (float)c.v0_cms;
  cc.T_inf = std::isinf(c.T_inf) ? INFINITY : (float)c.T_inf;
  cc.dust_on = c.dust_on ? 1 : 0;

  iris::MarchConsts& mc = ctx->mc;
  mc.hnu_k = cc.hnu_k;
  mc.T_bg = (float)planck_krj(H_PLANCK * nu / K_BOLTZ, c.T_cmb);
  mc.inv_KRJ = (float)(1.0 / KRJ);
  mc.out_mode = out_mode_of(c);
  mc.fine_m = 0;
  mc.ray_simpson = 0;
  mc.sel_thin = 0;
  mc.v0_over_c = (float)(c.v0_cms / C_LIGHT);
  mc.dv_over_c = (float)(c.dv_cms / C_LIGHT);
  mc.hnu_k_over_Tcmb = c.T_cmb > 0.0 ? (float)(H_PLANCK * nu / K_BOLTZ / c.T_cmb) : 0.0f;

  iris::BeamConsts& bc = ctx->bc;
  std::memset(&bc, 0, sizeof bc);
  if (c.beam_fwhm_px > 0.0) {
    const double sigma = c.beam_fwhm_px / (2.0 * std::sqrt(2.0 * std::log(2.0)));
    const int R = (int)std::ceil(4.0 * sigma);
    bc.R = R;
    double g[2 * iris::kMaxBeamRadius + 1], s = 0.0;
    for (int d = -R; d <= R; ++d) { g[d + R] = std::exp(-0.5 * d * d / (sigma * sigma)); s += g[d + R]; }
    for (int d = 0; d <= 2 * R; ++d) bc.g[d] = (float)(g[d] / s);
  }

  iris::NoiseConsts& nc = ctx->nc;
  nc.k0 = (uint32_t)c.seed; nc.k1 = (uint32_t)(c.seed >> 32);
  double gamma = 1.0;
  if (c.noise_gamma_mode == 1) {
    uint32_t r[4];
    host_philox(c.seed, 0u, 0u, 1u, 0u, r);
    gamma = (double)(r[0] >> 8) / 16777216.0;
  }
  nc.mu = (float)(gamma * c.noise_mu);
  nc.sigma = (float)(gamma * c.noise_sigma);
  nc.on = (c.noise_sigma != 0.0 || c.noise_mu != 0.0) ? 1 : 0;

  iris::AdjointConsts& ac = ctx->ac;
  ac.c_e = cc.c_e; ac.c_a = cc.c_a; ac.c_d = cc.c_d; ac.gr = cc.gr; ac.upper = u; ac.lower = l;
  ac.T_inf = cc.T_inf;
  ac.scale = c.out_unit == 1 ? 1.0f : mc.inv_KRJ;      // dL/dD in Kelvin space
  ac.subtract = c.subtract_continuum ? 1 : 0;
}

template <int N>
void launch_levelpop(iris_so_ctx* ctx, const float* n, const float* T, float* pop, cudaStream_t st) {
  const int64_t nc = ctx->ncell;
  const unsigned grid = (unsigned)((nc + 127) / 128);
  constexpr int BN = iris::kBandNarrow < N - 1 ? iris::kBandNarrow : N - 1;
  const bool table = ctx->lc.tb.K != nullptr;
  if (ctx->band <= BN) {
    if (table) iris::levelpop_kernel<N, BN, true><<<grid, 128, 0, st>>>(ctx->lc, nc, n, T, pop);
    else iris::levelpop_kernel<N, BN, false><<<grid, 128, 0, st>>>(ctx->lc, nc, n, T, pop);
  } else {
    if (table) iris::levelpop_kernel<N, N - 1, true><<<grid, 128, 0, st>>>(ctx->lc, nc, n, T, pop);
    else iris::levelpop_kernel<N, N - 1, false><<<grid, 128, 0, st>>>(ctx->lc, nc, n, T, pop);
  }
}

template <int N>
void launch_cellcoef(iris_so_ctx* ctx, const float* n, const float* T, const float* Td, const float* v, float* coef,
                     cudaStream_t st) {
  const int64_t nc = ctx->ncell;
  const unsigned grid = (unsigned)((nc + 127) / 128);
  constexpr int BN = iris::kBandNarrow < N - 1 ? iris::kBandNarrow : N - 1;
  const bool table = ctx->lc.tb.K != nullptr;
  // two cells per thread with packed arithmetic (bit-identical results, cell_kernels.cuh) where the 8-byte accesses line up
  const bool pairs = !table && ctx->band <= BN && nc % 2 == 0 &&
                     ((reinterpret_cast<uintptr_t>(n) | reinterpret_cast<uintptr_t>(T) | reinterpret_cast<uintptr_t>(Td) |
                       reinterpret_cast<uintptr_t>(v) | reinterpret_cast<uintptr_t>(coef)) % 8 == 0);
  if (pairs) {
    iris::cellcoef2_kernel<N, BN><<<(unsigned)((nc / 2 + 127) / 128), 128, 0, st>>>(ctx->lc, ctx->cc, nc, n, T, Td, v, coef);
    return;
  }
  if (ctx->band <= BN) {
    if (table) iris::cellcoef_kernel<N, BN, true><<<grid, 128, 0, st>>>(ctx->lc, ctx->cc, nc, n, T, Td, v, coef);
    else iris::cellcoef_kernel<N, BN, false><<<grid, 128, 0, st>>>(ctx->lc, ctx->cc, nc, n, T, Td, v, coef);
  } else {
    if (table) iris::cellcoef_kernel<N, N - 1, true><<<grid, 128, 0, st>>>(ctx->lc, ctx->cc, nc, n, T, Td, v, coef);
    else iris::cellcoef_kernel<N, N - 1, false><<<grid, 128, 0, st>>>(ctx->lc, ctx->cc, nc, n, T, Td, v, coef);
  }
}

#define IRIS_DISPATCH_N(N_, CALL)                       \
  switch (N_) {                                         \
    case 2: CALL(2); break;  case 3: CALL(3); break;    \
    case 4: CALL(4); break;  case 5: CALL(5); break;    \
    case 6: CALL(6); break;  case 7: CALL(7); break;    \
    case 8: CALL(8); break;  case 9: CALL(9); break;    \
    default: CALL(10); break;                           \
  }

// K1+K2 (or K2 from caller populations) into ctx->d_coef
iris_so_status run_coefficients(iris_so_ctx* ctx, const float* n, const float* T, const float* Td, const float* v,
                                const float* pop, cudaStream_t st) {
  iris_so_status s = ensure(ctx, &ctx->d_coef, sizeof(float) * 6 * (size_t)ctx->ncell, "cudaMalloc(coefficient planes)");
  if (s != IRIS_SO_OK) return s;
  ProfScope prof(ctx, IRIS_SO_STAGE_CELL, st);
  if (pop) {
    iris::coef_from_pop_kernel<<<(unsigned)((ctx->ncell + 255) / 256), 256, 0, st>>>(ctx->cc, ctx->ncell, n, T, Td, v, pop,
                                                                                     ctx->d_coef);
    IRIS_CHECK_LAUNCH(ctx, "coef_from_pop_kernel");
  } else if (ctx->cfg.coef_grid == 1) {
    // 16-byte accesses need aligned field pointers and planes that are a multiple of 4 cells apart
    const int aligned = (ctx->ncell % 4 == 0) &&
                        ((reinterpret_cast<uintptr_t>(n) | reinterpret_cast<uintptr_t>(T) | reinterpret_cast<uintptr_t>(Td) |
                          reinterpret_cast<uintptr_t>(v)) % 16 == 0);
    iris::cellcoef_grid_kernel<<<(unsigned)(((ctx->ncell + 3) / 4 + 255) / 256), 256, 0, st>>>(ctx->cc, ctx->gc, ctx->ncell, aligned, n,
                                                                                               T, Td, v, ctx->d_coef);
    IRIS_CHECK_LAUNCH(ctx, "cellcoef_grid_kernel");
  } else {
#define CALL_(N) launch_cellcoef<N>(ctx, n, T, Td, v, ctx->d_coef, st)
    IRIS_DISPATCH_N(ctx->cfg.n_levels, CALL_)
#undef CALL_
    IRIS_CHECK_LAUNCH(ctx, "cellcoef_kernel");
  }
  return IRIS_SO_OK;
}

// Which transfer kernel the configuration selects: 1 dense, 2 window + centre-expansion profile, 3 window + erfc edges.
int resolved_algo(const iris_so_config& c) {
  int algo = c.transfer_algo;
  if (algo == IRIS_SO_ALGO_AUTO) algo = IRIS_SO_ALGO_WINDOW;
  if (algo == IRIS_SO_ALGO_WINDOW && !(c.microturb_cms > 0.0 && c.dv_cms <= (double)iris::kSeriesMaxS * c.microturb_cms))
    algo = IRIS_SO_ALGO_WINDOW_EDGE;      // b >= xi bounds dv / b only when there is microturbulence
  return algo;
}

bool hot_path_mode(const iris_so_config& c) { return c.transfer_mode == 0 && c.integration == 0 && c.subsample == 0; }

bool spectra_fit_shared(const iris_so_config& c) {
  return (size_t)(32 / 8) * ((size_t)c.nv + 32) * sizeof(float) + 2048 <= 227u * 1024u;
}

// Selectively thin and optically thin transfer with formal integration and the channel-integrated profile are identities
// outside a cell's line window too (in the dust-scaled spectrum), so they run through the line-window series kernel
// (template MODE 1 / 2) whenever it applies; transfer_algo = IRIS_SO_ALGO_DENSE keeps them on transfer_modes_kernel.
bool windowed_thin_mode(const iris_so_config& c) {
  const bool formal = (c.transfer_mode == 1 || c.transfer_mode == 2) && c.integration == 0;
  const bool thin_simpson = c.transfer_mode == 2 && c.integration == 1;     // a weighted sum along the ray: same kernel
  return (formal || thin_simpson) && c.subsample == 0 &&
         c.transfer_algo != IRIS_SO_ALGO_DENSE && c.microturb_cms > 0.0 &&
         c.dv_cms <= (double)iris::kSeriesMaxS * c.microturb_cms && spectra_fit_shared(c);
}

// Optically thick formal transfer on the fine velocity grid (subsample = f > 0): the same line-window march over the
// nv (f + 1) + 1 points of the fine grid with the point profile, Simpson's rule per channel in the epilogue (MODE 3).
bool windowed_fine_mode(const iris_so_config& c) {
  if (!(c.transfer_mode == 0 && c.integration == 0 && c.subsample > 0 && c.transfer_algo != IRIS_SO_ALGO_DENSE)) return false;
  const size_t points = (size_t)c.nv * (size_t)(c.subsample + 1) + 1;
  return (size_t)(32 / 8) * (points + 32) * sizeof(float) + 2048 <= 227u * 1024u;
}

// Optically thick transfer with the smooth integrator as a line-window march (transfer_smooth.cuh), followed by the
// dense modes kernel gated on the flag the window kernel raises when a ReLU fires where it does not look.
bool windowed_smooth_mode(const iris_so_config& c) {
  if (!((c.transfer_mode == 0 || c.transfer_mode == 1) && c.integration == 1 && c.transfer_algo != IRIS_SO_ALGO_DENSE && c.nz >= 2)) return false;
  if (c.subsample == 0 && !(c.microturb_cms > 0.0 && c.dv_cms <= (double)iris::kSeriesMaxS * c.microturb_cms)) return false;
  return iris::smooth_window_smem_per_warp(c.nv, c.subsample > 0 ? c.subsample + 1 : 0) + 1024 <= 227u * 1024u;
}

// K3 (+K4, K5) from ctx->d_coef
iris_so_status run_transfer(iris_so_ctx* ctx, const iris::MarchConsts& mc, float* out, float* out_cont, cudaStream_t st) {
  const bool dust = ctx->cfg.dust_on != 0;
  const int npix = (int)ctx->npix, nz = ctx->cfg.nz, nv = ctx->cfg.nv;
  const int algo = resolved_algo(ctx->cfg);
  ProfScope prof(ctx, IRIS_SO_STAGE_TRANSFER, st);
  if (windowed_fine_mode(ctx->cfg)) {
    iris::MarchConsts mf = mc;
    mf.fine_m = ctx->cfg.subsample + 1;
    cudaError_t e = iris::launch_transfer_series(mf, ctx->d_coef, ctx->ncell, npix, nz, nv, dust, 0.0f, out, out_cont, st, 3);
    ctx->launches++;
    if (e != cudaSuccess) return cuda_fail(ctx, e, "launch of the line-window transfer kernel (fine grid)");
    return IRIS_SO_OK;
  }
  if (windowed_thin_mode(ctx->cfg)) {
    iris::MarchConsts mt = mc;
    mt.ray_simpson = ctx->cfg.integration == 1 ? 1 : 0;
    cudaError_t e = iris::launch_transfer_series(mt, ctx->d_coef, ctx->ncell, npix, nz, nv, dust,
                                                 (float)(ctx->cfg.dv_cms / ctx->cfg.microturb_cms), out, out_cont, st,
                                                 ctx->cfg.transfer_mode);
    ctx->launches++;
    if (e != cudaSuccess) return cuda_fail(ctx, e, "launch of the line-window transfer kernel");
    return IRIS_SO_OK;
  }
  if (!hot_path_mode(ctx->cfg)) {
    iris::ModeConsts md;
    md.mode = ctx->cfg.transfer_mode; md.smooth = ctx->cfg.integration;
    md.fine_m = ctx->cfg.subsample > 0 ? ctx->cfg.subsample + 1 : 0;
    md.nx = ctx->cfg.nx;
    md.gate = nullptr;
    md.list = nullptr;
    if (windowed_smooth_mode(ctx->cfg)) {
      if (!ctx->d_gate) return fail(ctx, IRIS_SO_ECUDA, "gate flag not allocated");      // begin_call allocates it
      cudaError_t e = cudaMemsetAsync(ctx->d_gate, 0, sizeof(int), st);
      if (e != cudaSuccess) return cuda_fail(ctx, e, "cudaMemsetAsync(gate)");
      iris::MarchConsts mf = mc;
      mf.fine_m = md.fine_m;
      mf.sel_thin = ctx->cfg.transfer_mode == 1;
      e = iris::launch_transfer_smooth_window(mf, ctx->d_coef, ctx->ncell, npix, nz, nv, out, out_cont, ctx->d_gate,
                                              ctx->d_gate + 2, st);
      ctx->launches++;
      if (e != cudaSuccess) return cuda_fail(ctx, e, "launch of transfer_smooth_window_kernel");
      md.gate = ctx->d_gate;
      md.list = ctx->d_gate + 2;
    }
    cudaError_t e = iris::launch_transfer_modes(mc, md, ctx->d_coef, ctx->ncell, npix, nz, nv, out, out_cont, st);
    ctx->launches++;
    if (e != cudaSuccess) return cuda_fail(ctx, e, "launch of transfer_modes_kernel");
    return IRIS_SO_OK;
  }
  // the line-window kernels keep whole spectra in shared memory: beyond ~13000 channels they do not fit and the
  // dense kernel (spectra in registers, any nv) takes over
  const bool fits = (size_t)(32 / 8) * ((size_t)nv + 32) * sizeof(float) + 2048 <= 227u * 1024u;
  if (algo == IRIS_SO_ALGO_DENSE || !fits || ctx->cfg.dust_per_channel) {
    constexpr int CB = 16, NW = 4;
    const int nx = ctx->cfg.nx, rows = npix / nx;
    dim3 block(32, NW), grid(((nx + 7) / 8) * ((rows + 3) / 4), (nv + CB * NW - 1) / (CB * NW));
    if (ctx->cfg.dust_per_channel)      // (with the dust off its planes are zero: the same instantiation)
      iris::transfer_dense_kernel<CB, true, true><<<grid, block, 0, st>>>(mc, ctx->d_coef, ctx->ncell, npix, nx, nz, nv, out, out_cont);
    else if (dust) iris::transfer_dense_kernel<CB, true><<<grid, block, 0, st>>>(mc, ctx->d_coef, ctx->ncell, npix, nx, nz, nv, out, out_cont);
    else iris::transfer_dense_kernel<CB, false><<<grid, block, 0, st>>>(mc, ctx->d_coef, ctx->ncell, npix, nx, nz, nv, out, out_cont);
    IRIS_CHECK_LAUNCH(ctx, "transfer_dense_kernel");
    return IRIS_SO_OK;
  }
  cudaError_t e;
  if (algo == IRIS_SO_ALGO_WINDOW) {
    // reachable-range spectra (half-size circular buffers, transfer_series.cuh) while at most 3 % of the pixels of the
    // previous launch had to be handed over to the whole-spectrum variant
    if (ctx->hand_pending && cudaEventQuery(ctx->ev_hand) == cudaSuccess) {
      if ((int64_t)*ctx->h_hand * 100 > 3 * ctx->hand_npix) ctx->circ_ok = false;
      ctx->hand_pending = false;
    }
    cudaGetLastError();
    int* hand = (ctx->circ_ok && ctx->d_gate) ? ctx->d_gate : nullptr;
    if (hand && (e = cudaMemsetAsync(hand, 0, sizeof(int), st)) != cudaSuccess) return cuda_fail(ctx, e, "cudaMemsetAsync(hand-over count)");
    int used_circ = 0;
    e = iris::launch_transfer_series(mc, ctx->d_coef, ctx->ncell, npix, nz, nv, dust,
                                     (float)(ctx->cfg.dv_cms / ctx->cfg.microturb_cms), out, out_cont, st, 0, hand, &used_circ);
    if (used_circ) {
      ctx->launches++;
      if (e == cudaSuccess && ctx->h_hand && !ctx->hand_pending) {
        cudaMemcpyAsync(ctx->h_hand, hand, sizeof(int), cudaMemcpyDeviceToHost, st);
        cudaEventRecord(ctx->ev_hand, st);
        ctx->hand_pending = true;
        ctx->hand_npix = npix;
      }
    }
  } else {
    e = iris::launch_transfer_window(mc, ctx->d_coef, ctx->ncell, npix, nz, nv, dust, ctx->sm_count, out, out_cont, st);
  }
  ctx->launches++;
  if (e != cudaSuccess) return cuda_fail(ctx, e, "launch of the line-window transfer kernel");
  return IRIS_SO_OK;
}

// Kernels that hand pixels over to a second launch: the smooth window kernel, and the series kernel of the hot path with
// reachable-range spectra.
bool uses_handover(const iris_so_config& c) {
  return windowed_smooth_mode(c) ||
         (hot_path_mode(c) && !c.dust_per_channel && resolved_algo(c) == IRIS_SO_ALGO_WINDOW && spectra_fit_shared(c));
}

// Start of a public call that runs the transfer: clears the accumulated hand-over count.
iris_so_status begin_call(iris_so_ctx* ctx, cudaStream_t st) {
  if (!uses_handover(ctx->cfg)) return IRIS_SO_OK;
  cudaError_t e;
  if (!ctx->d_gate) {
    if ((e = cudaMalloc(reinterpret_cast<void**>(&ctx->d_gate), (2 + (size_t)ctx->npix) * sizeof(int))) != cudaSuccess)
      return cuda_fail(ctx, e, "cudaMalloc(gate)");
    if (cudaHostAlloc(reinterpret_cast<void**>(&ctx->h_hand), sizeof(int), cudaHostAllocDefault) != cudaSuccess ||
        cudaEventCreateWithFlags(&ctx->ev_hand, cudaEventDisableTiming) != cudaSuccess) {
      cudaGetLastError();
      if (ctx->h_hand) { cudaFreeHost(ctx->h_hand); ctx->h_hand = nullptr; }      // no feedback: the choice stays as it is
    }
  }
  if ((e = cudaMemsetAsync(ctx->d_gate, 0, 2 * sizeof(int), st)) != cudaSuccess) return cuda_fail(ctx, e, "cudaMemsetAsync(gate)");
  return IRIS_SO_OK;
}

iris_so_status run_beam(iris_so_ctx* ctx, const float* in, float* out, float* tmp, bool noise, cudaStream_t st) {
  const iris_so_config& c = ctx->cfg;
  if (!tmp) {
    iris_so_status s = ensure(ctx, &ctx->d_tmp, sizeof(float) * (size_t)ctx->nvox, "cudaMalloc(beam temporary)");
    if (s != IRIS_SO_OK) return s;
    tmp = ctx->d_tmp;
  }
  ProfScope prof(ctx, IRIS_SO_STAGE_BEAM, st);
  iris::NoiseConsts off = ctx->nc; off.on = 0;
  iris::NoiseConsts nz2 = ctx->nc; nz2.on = noise ? ctx->nc.on : 0;
  // pass 1 along x: a = x (stride nv), b = y (stride nx*nv)
  iris::launch_beam_pass(ctx->bc, off, in, tmp, c.nx, c.ny, c.nv, (int64_t)c.nv, (int64_t)c.nx * c.nv, st);
  IRIS_CHECK_LAUNCH(ctx, "beam pass (x)");
  // pass 2 along y: a = y (stride nx*nv), b = x (stride nv)
  iris::launch_beam_pass(ctx->bc, nz2, tmp, out, c.ny, c.nx, c.nv, (int64_t)c.nx * c.nv, (int64_t)c.nv, st);
  IRIS_CHECK_LAUNCH(ctx, "beam pass (y)");
  return IRIS_SO_OK;
}

iris_so_status run_noise(iris_so_ctx* ctx, float* cube, cudaStream_t st) {
  ProfScope prof(ctx, IRIS_SO_STAGE_NOISE, st);
  iris::noise_kernel<<<(unsigned)(((ctx->nvox + 3) / 4 + 255) / 256), 256, 0, st>>>(ctx->nc, cube, ctx->nvox);
  IRIS_CHECK_LAUNCH(ctx, "noise_kernel");
  return IRIS_SO_OK;
}

template <int N>
void launch_grid_nodes(iris_so_ctx* ctx, float* nodeval) {
  const int nq = ctx->gc.nn * ctx->gc.nT;
  const unsigned grid = (unsigned)((nq + 127) / 128);
  constexpr int BN = iris::kBandNarrow < N - 1 ? iris::kBandNarrow : N - 1;
  const bool table = ctx->lc.tb.K != nullptr;
  if (ctx->band <= BN) {
    if (table) iris::grid_nodes_kernel<N, BN, true><<<grid, 128>>>(ctx->lc, ctx->cc, ctx->gc, nodeval);
    else iris::grid_nodes_kernel<N, BN, false><<<grid, 128>>>(ctx->lc, ctx->cc, ctx->gc, nodeval);
  } else {
    if (table) iris::grid_nodes_kernel<N, N - 1, true><<<grid, 128>>>(ctx->lc, ctx->cc, ctx->gc, nodeval);
    else iris::grid_nodes_kernel<N, N - 1, false><<<grid, 128>>>(ctx->lc, ctx->cc, ctx->gc, nodeval);
  }
}

// Grid precomputation: node tables on the host (double), node values and cell coefficients on the device.
iris_so_status build_grid(iris_so_ctx* ctx) {
  const iris_so_config& c = ctx->cfg;
  const int nn = c.grid_n_density, nT = c.grid_n_temp;
  std::vector<float> h(2 * (size_t)(nn + nT));
  auto fill = [&](float* dst, int cnt, double lo, double hi) {
    std::vector<double> node(cnt);
    for (int i = 0; i < cnt; ++i) node[i] = (double)(float)(lo * std::pow(hi / lo, (double)i / (double)(cnt - 1)));
    for (int i = 0; i < cnt; ++i) {
      const int a = std::min(i, cnt - 2);
      dst[2 * i] = (float)node[i];
      dst[2 * i + 1] = (float)(1.0 / (node[a + 1] - node[a]));
    }
  };
  fill(h.data(), nn, c.grid_nH2_lo, c.grid_nH2_hi);
  fill(h.data() + 2 * nn, nT, c.grid_T_lo, c.grid_T_hi);
  const size_t tab_f = h.size(), node_f = 2 * (size_t)nn * nT, cell_f = 8 * (size_t)(nn - 1) * (nT - 1);
  const size_t node_off = (tab_f + 3) / 4 * 4, cell_off = (node_off + node_f + 3) / 4 * 4;      // 16-byte aligned blocks
  cudaError_t e = cudaMalloc(reinterpret_cast<void**>(&ctx->d_grid), (cell_off + cell_f) * sizeof(float));
  if (e != cudaSuccess) return cuda_fail(nullptr, e, "cudaMalloc(coefficient grid)");
  if ((e = cudaMemcpy(ctx->d_grid, h.data(), tab_f * sizeof(float), cudaMemcpyHostToDevice)) != cudaSuccess)
    return cuda_fail(nullptr, e, "upload of the grid nodes");
  iris::GridConsts& gc = ctx->gc;
  gc.nodes_n = reinterpret_cast<const float2*>(ctx->d_grid);
  gc.nodes_T = reinterpret_cast<const float2*>(ctx->d_grid + 2 * nn);
  gc.cells = reinterpret_cast<const float4*>(ctx->d_grid + cell_off);
  gc.nn = nn; gc.nT = nT;
  gc.log2_n_lo = (float)std::log2(c.grid_nH2_lo);
  gc.inv_dlog2_n = (float)((nn - 1) / std::log2(c.grid_nH2_hi / c.grid_nH2_lo));
  gc.log2_T_lo = (float)std::log2(c.grid_T_lo);
  gc.inv_dlog2_T = (float)((nT - 1) / std::log2(c.grid_T_hi / c.grid_T_lo));
  float* nodeval = ctx->d_grid + node_off;
#define CALL_(N) launch_grid_nodes<N>(ctx, nodeval)
  IRIS_DISPATCH_N(c.n_levels, CALL_)
#undef CALL_
  ctx->launches++;
  if ((e = cudaGetLastError()) != cudaSuccess) return cuda_fail(nullptr, e, "launch of grid_nodes_kernel");
  iris::grid_cells_kernel<<<(unsigned)((2 * (nn - 1) * (nT - 1) + 127) / 128), 128>>>(nn, nT, nodeval,
                                                                                    reinterpret_cast<float4*>(ctx->d_grid + cell_off));
  ctx->launches++;
  if ((e = cudaGetLastError()) != cudaSuccess) return cuda_fail(nullptr, e, "launch of grid_cells_kernel");
  if ((e = cudaDeviceSynchronize()) != cudaSuccess) return cuda_fail(nullptr, e, "grid precomputation");
  ctx->scratch_bytes += (cell_off + cell_f) * sizeof(float);
  return IRIS_SO_OK;
}

}  // namespace

extern "C" {

int iris_so_version(void) { return IRIS_SO_VERSION; }

const char* iris_so_status_string(iris_so_status s) {
  switch (s) {
    case IRIS_SO_OK: return "ok";
    case IRIS_SO_EINVAL: return "invalid argument";
    case IRIS_SO_EUNSUPPORTED: return "unsupported";
    case IRIS_SO_ECUDA: return "CUDA error";
    case IRIS_SO_ENOMEM: return "out of memory";
  }
  return "unknown";
}

const char* iris_so_last_error(const iris_so_ctx* ctx) { return ctx ? ctx->err.c_str() : g_create_error.c_str(); }

const char* iris_so_transfer_kernel(const iris_so_ctx* ctx) {
  if (!ctx) return "";
  if (windowed_thin_mode(ctx->cfg) || windowed_fine_mode(ctx->cfg)) return "transfer_series_kernel";
  if (windowed_smooth_mode(ctx->cfg)) return "transfer_smooth_window_kernel";
  if (!hot_path_mode(ctx->cfg)) return "transfer_modes_kernel";
  if (ctx->cfg.dust_per_channel) return "transfer_dense_kernel";
  if ((size_t)(32 / 8) * ((size_t)ctx->cfg.nv + 32) * sizeof(float) + 2048 > 227u * 1024u) return "transfer_dense_kernel";
  switch (resolved_algo(ctx->cfg)) {
    case IRIS_SO_ALGO_DENSE: return "transfer_dense_kernel";
    case IRIS_SO_ALGO_WINDOW: return "transfer_series_kernel";
    default: return "transfer_window_kernel";
  }
}

uint64_t iris_so_launch_count(const iris_so_ctx* ctx) { return ctx ? ctx->launches : 0; }
uint64_t iris_so_scratch_bytes(const iris_so_ctx* ctx) { return ctx ? ctx->scratch_bytes : 0; }

iris_so_status iris_so_create(const iris_so_config* cfg, iris_so_ctx** out) {
  if (!out) return fail(nullptr, IRIS_SO_EINVAL, "out is NULL");
  *out = nullptr;
  std::string why;
  iris_so_status s = validate(cfg, why);
  if (s != IRIS_SO_OK) return fail(nullptr, s, why);
  if (cfg->beam_fwhm_px > 0.0) {
    const double sigma = cfg->beam_fwhm_px / (2.0 * std::sqrt(2.0 * std::log(2.0)));
    if ((int)std::ceil(4.0 * sigma) > iris::kMaxBeamRadius)
      return fail(nullptr, IRIS_SO_EUNSUPPORTED, "beam radius ceil(4 sigma) exceeds 32 pixels");
  }
  if (cfg->dust_per_channel && !hot_path_mode(*cfg))
    return fail(nullptr, IRIS_SO_EUNSUPPORTED, "dust_per_channel = 1 is implemented for the thick / formal / channel-integrated mode only");
  int dev = 0, count = 0;
  cudaError_t e = cudaGetDeviceCount(&count);
  if (e != cudaSuccess || count == 0) {
    cudaGetLastError();
    return fail(nullptr, IRIS_SO_ECUDA, "no CUDA device: this library has no CPU fallback");
  }
  if ((e = cudaGetDevice(&dev)) != cudaSuccess) return cuda_fail(nullptr, e, "cudaGetDevice");
  iris_so_ctx* ctx = new (std::nothrow) iris_so_ctx;
  if (!ctx) return fail(nullptr, IRIS_SO_ENOMEM, "host allocation failed");
  ctx->cfg = *cfg;
  const int N = cfg->n_levels;
  ctx->energy.assign(cfg->energy_K, cfg->energy_K + N);
  ctx->weight.assign(cfg->weight, cfg->weight + N);
  ctx->A.assign(cfg->einstein_A, cfg->einstein_A + N * N);
  ctx->Kd.assign(cfg->coll_down_ref, cfg->coll_down_ref + N * N);
  ctx->cfg.energy_K = ctx->energy.data(); ctx->cfg.weight = ctx->weight.data();
  ctx->cfg.einstein_A = ctx->A.data(); ctx->cfg.coll_down_ref = ctx->Kd.data();
  if (cfg->coll_n_partners > 0) {
    const int nT = cfg->coll_nT;
    ctx->Tgrid.assign(cfg->coll_T_grid, cfg->coll_T_grid + nT);
    ctx->Keff.assign((size_t)nT * N * N, 0.0);
    for (int p = 0; p < cfg->coll_n_partners; ++p)
      for (int64_t q = 0; q < (int64_t)nT * N * N; ++q)
        ctx->Keff[q] += cfg->coll_partner_frac[p] * cfg->coll_table[(int64_t)p * nT * N * N + q];
    // the copied configuration must not point into the caller's arrays: the folded table takes their place
    ctx->cfg.coll_T_grid = ctx->Tgrid.data(); ctx->cfg.coll_table = nullptr; ctx->cfg.coll_partner_frac = nullptr;
    // Kd = the largest rate over the grid: band detection and validation of "a downward rate exists"
    for (int q = 0; q < N * N; ++q) {
      double m = 0.0;
      for (int t = 0; t < nT; ++t) m = std::max(m, ctx->Keff[(size_t)t * N * N + q]);
      ctx->Kd[q] = m;
    }
  }
  ctx->device = dev;
  cudaDeviceGetAttribute(&ctx->sm_count, cudaDevAttrMultiProcessorCount, dev);
  ctx->npix = (int64_t)cfg->nx * cfg->ny;
  ctx->ncell = ctx->npix * cfg->nz;
  ctx->nvox = ctx->npix * cfg->nv;
  fold_constants(ctx);
  if (!ctx->Keff.empty()) {
    // device table in the kernels' layout
    const int nT = cfg->coll_nT;
    std::vector<float> h((size_t)nT + (size_t)nT * iris::kMaxPairs * 2, 0.0f);
    for (int t = 0; t < nT; ++t) h[t] = (float)ctx->Tgrid[t];
    const double rs = ctx->lc.rate_scale;
    for (int t = 0; t < nT; ++t)
      for (int u = 1; u < N; ++u)
        for (int l = 0; l < u; ++l) {
          const double K = ctx->Keff[(size_t)t * N * N + u * N + l];
          const size_t o = (size_t)nT + ((size_t)t * iris::kMaxPairs + iris::pair_index(u, l)) * 2;
          h[o] = (float)(rs * K);
          h[o + 1] = (float)(rs * K * ctx->weight[u] / ctx->weight[l]);
        }
    // the float2 rows must be 8-byte aligned: pad the temperature block to an even count
    const size_t toff = (size_t)(nT + 1) / 2 * 2;
    std::vector<float> hd(toff + (size_t)nT * iris::kMaxPairs * 2, 0.0f);
    std::copy(h.begin(), h.begin() + nT, hd.begin());
    std::copy(h.begin() + nT, h.end(), hd.begin() + toff);
    cudaError_t ce = cudaMalloc(reinterpret_cast<void**>(&ctx->d_colltab), hd.size() * sizeof(float));
    if (ce == cudaSuccess) ce = cudaMemcpy(ctx->d_colltab, hd.data(), hd.size() * sizeof(float), cudaMemcpyHostToDevice);
    if (ce != cudaSuccess) {
      cudaGetLastError();
      iris_so_status st = cuda_fail(nullptr, ce, "upload of the collision table");
      iris_so_destroy(ctx);
      return st;
    }
    ctx->lc.tb.T = ctx->d_colltab;
    ctx->lc.tb.K = reinterpret_cast<const float2*>(ctx->d_colltab + toff);
    ctx->lc.tb.nT = nT;
  }
  if (cfg->coef_grid == 1) {
    iris_so_status gs = build_grid(ctx);
    if (gs != IRIS_SO_OK) { iris_so_destroy(ctx); return gs; }
  }
  // set-up for iris_so_observe_raw_static (this device is current): not fatal here, that entry point reports it
  ctx->d_static_coef = static_scratch_of_device(dev, &ctx->static_err);
  *out = ctx;
  return IRIS_SO_OK;
}

void iris_so_destroy(iris_so_ctx* ctx) {
  if (!ctx) return;
  cudaFree(ctx->d_coef); cudaFree(ctx->d_tmp); cudaFree(ctx->d_stage); cudaFree(ctx->d_adj); cudaFree(ctx->d_counter); cudaFree(ctx->d_gate); cudaFree(ctx->d_metrics); cudaFree(ctx->d_colltab); cudaFree(ctx->d_grid);
  if (ctx->h_hand) cudaFreeHost(ctx->h_hand);
  if (ctx->ev_hand) cudaEventDestroy(ctx->ev_hand);
  if (ctx->s_in) cudaStreamDestroy(ctx->s_in);
  if (ctx->s_out) cudaStreamDestroy(ctx->s_out);
  for (auto ev : ctx->slab_events) cudaEventDestroy(ev);
  prof_reset(ctx);
  for (cudaEvent_t e : ctx->event_pool) cudaEventDestroy(e);
  delete ctx;
}

iris_so_status iris_so_levelpop(iris_so_ctx* ctx, const float* d_nH2, const float* d_Tgas, float* d_pop, void* stream) {
  if (!ctx) return IRIS_SO_EINVAL;
  if (!d_nH2 || !d_Tgas || !d_pop) return fail(ctx, IRIS_SO_EINVAL, "iris_so_levelpop: NULL pointer");
  cudaStream_t st = static_cast<cudaStream_t>(stream);
#define CALL_(N) launch_levelpop<N>(ctx, d_nH2, d_Tgas, d_pop, st)
  IRIS_DISPATCH_N(ctx->cfg.n_levels, CALL_)
#undef CALL_
  IRIS_CHECK_LAUNCH(ctx, "levelpop_kernel");
  return IRIS_SO_OK;
}

iris_so_status iris_so_transfer(iris_so_ctx* ctx, const float* d_nH2, const float* d_Tgas, const float* d_Tdust,
                                const float* d_vlos, const float* d_pop, float* d_I_total, float* d_I_cont, void* stream) {
  if (!ctx) return IRIS_SO_EINVAL;
  if (!d_nH2 || !d_Tgas || !d_Tdust || !d_vlos) return fail(ctx, IRIS_SO_EINVAL, "iris_so_transfer: NULL field pointer");
  if (!d_I_total && !d_I_cont) return fail(ctx, IRIS_SO_EINVAL, "iris_so_transfer: no output requested");
  if (ctx->cfg.dust_per_channel && d_I_cont)
    return fail(ctx, IRIS_SO_EUNSUPPORTED, "iris_so_transfer: with dust_per_channel = 1 the continuum is a spectrum; pass d_I_cont = NULL");
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  iris_so_status s = begin_call(ctx, st);
  if (s != IRIS_SO_OK) return s;
  if ((s = run_coefficients(ctx, d_nH2, d_Tgas, d_Tdust, d_vlos, d_pop, st)) != IRIS_SO_OK) return s;
  iris::MarchConsts mc = ctx->mc;
  mc.out_mode = iris::OUT_I_TOT;
  return run_transfer(ctx, mc, d_I_total, d_I_cont, st);
}

iris_so_status iris_so_observe_stages(iris_so_ctx* ctx, const float* d_nH2, const float* d_Tgas, const float* d_Tdust,
                                      const float* d_vlos, int32_t stage_mask, float* d_cube, void* stream) {
  if (!ctx) return IRIS_SO_EINVAL;
  if (!d_nH2 || !d_Tgas || !d_Tdust || !d_vlos || !d_cube) return fail(ctx, IRIS_SO_EINVAL, "iris_so_observe: NULL pointer");
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  iris_so_status s = begin_call(ctx, st);
  if (s != IRIS_SO_OK) return s;
  if ((s = run_coefficients(ctx, d_nH2, d_Tgas, d_Tdust, d_vlos, nullptr, st)) != IRIS_SO_OK) return s;
  if ((s = run_transfer(ctx, ctx->mc, d_cube, nullptr, st)) != IRIS_SO_OK) return s;
  const bool beam = (stage_mask & 1) && ctx->cfg.beam_fwhm_px > 0.0;
  const bool noise = (stage_mask & 2) && ctx->nc.on;
  if (beam) return run_beam(ctx, d_cube, d_cube, nullptr, noise, st);   // x pass: cube -> tmp, y pass: tmp -> cube
  if (noise) return run_noise(ctx, d_cube, st);
  return IRIS_SO_OK;
}

iris_so_status iris_so_observe(iris_so_ctx* ctx, const float* d_nH2, const float* d_Tgas, const float* d_Tdust,
                               const float* d_vlos, float* d_cube, void* stream) {
  return iris_so_observe_stages(ctx, d_nH2, d_Tgas, d_Tdust, d_vlos, 3, d_cube, stream);
}

// K1 .. K5 of the hot-path mode with the coefficient planes in the library's static scratch (g_static_coef) instead of
// ctx->d_coef: no allocation of any kind, no event, no synchronisation.  A path of its own (the other entry points are
// untouched): K1 + K2, then the kernel resolved_algo() names -- the series kernel in its whole-spectrum variant (the
// reachable-range variant needs a hand-over list, i.e. more scratch), the window kernel or the dense kernel.
iris_so_status iris_so_observe_raw_static(iris_so_ctx* ctx, const float* d_nH2, const float* d_Tgas, const float* d_Tdust,
                                          const float* d_vlos, float* d_cube, void* stream) {
  if (!ctx) return IRIS_SO_EINVAL;
  if (!d_nH2 || !d_Tgas || !d_Tdust || !d_vlos || !d_cube)
    return fail(ctx, IRIS_SO_EINVAL, "iris_so_observe_raw_static: NULL pointer");
  const iris_so_config& c = ctx->cfg;
  if (!hot_path_mode(c) || c.coef_grid == 1 || c.dust_per_channel)
    return fail(ctx, IRIS_SO_EUNSUPPORTED,
                "iris_so_observe_raw_static serves the hot-path mode only (transfer_mode = integration = subsample = 0, "
                "coef_grid = 0, dust_per_channel = 0)");
  if (ctx->ncell > (int64_t)IRIS_SO_STATIC_MAX_CELLS) {
    char buf[256];
    snprintf(buf, sizeof buf, "iris_so_observe_raw_static: %lld cells exceed the static scratch of %d cells "
             "(IRIS_SO_STATIC_MAX_CELLS); use iris_so_observe_stages", (long long)ctx->ncell, (int)IRIS_SO_STATIC_MAX_CELLS);
    return fail(ctx, IRIS_SO_EUNSUPPORTED, buf);
  }
  if (!ctx->d_static_coef) return fail(ctx, IRIS_SO_ECUDA, "iris_so_observe_raw_static: " + ctx->static_err);
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  float* coef = ctx->d_static_coef;                    // planes at stride ncell, all 6 * ncell entries written by K1 + K2
  const bool dust = c.dust_on != 0;
  const int npix = (int)ctx->npix, nz = c.nz, nv = c.nv;
#define CALL_(N) launch_cellcoef<N>(ctx, d_nH2, d_Tgas, d_Tdust, d_vlos, coef, st)
  IRIS_DISPATCH_N(c.n_levels, CALL_)
#undef CALL_
  IRIS_CHECK_LAUNCH(ctx, "cellcoef_kernel");
  const int algo = resolved_algo(c);
  if (algo == IRIS_SO_ALGO_DENSE || !spectra_fit_shared(c)) {
    constexpr int CB = 16, NW = 4;
    const int nx = c.nx, rows = npix / nx;
    dim3 block(32, NW), grid(((nx + 7) / 8) * ((rows + 3) / 4), (nv + CB * NW - 1) / (CB * NW));
    if (dust) iris::transfer_dense_kernel<CB, true><<<grid, block, 0, st>>>(ctx->mc, coef, ctx->ncell, npix, nx, nz, nv, d_cube, nullptr);
    else iris::transfer_dense_kernel<CB, false><<<grid, block, 0, st>>>(ctx->mc, coef, ctx->ncell, npix, nx, nz, nv, d_cube, nullptr);
    IRIS_CHECK_LAUNCH(ctx, "transfer_dense_kernel");
    return IRIS_SO_OK;
  }
  cudaError_t e;
  if (algo == IRIS_SO_ALGO_WINDOW)
    e = iris::launch_transfer_series(ctx->mc, coef, ctx->ncell, npix, nz, nv, dust, (float)(c.dv_cms / c.microturb_cms), d_cube,
                                     nullptr, st, 0, nullptr, nullptr);
  else
    e = iris::launch_transfer_window(ctx->mc, coef, ctx->ncell, npix, nz, nv, dust, ctx->sm_count, d_cube, nullptr, st);
  ctx->launches++;
  if (e != cudaSuccess) return cuda_fail(ctx, e, "launch of the line-window transfer kernel (static scratch)");
  return IRIS_SO_OK;
}

// Host-buffer path.  Pixel columns are independent up to the beam, so the sky plane is cut into slabs of rows and
// the three legs are pipelined on three streams: H2D of slab k+1 (four strided field copies into a compact
// [nz][rows][nx] staging slab), K1-K5 of slab k on the caller's stream, D2H of the finished cube rows of slab k-1
// (PCIe is full duplex).  With a beam or noise configured the cube stays on the device until every slab is done, the
// post-processing runs on the whole cube and one D2H follows.
iris_so_status iris_so_observe_host(iris_so_ctx* ctx, const float* h_nH2, const float* h_Tgas, const float* h_Tdust,
                                    const float* h_vlos, float* h_cube, void* stream) {
  if (!ctx) return IRIS_SO_EINVAL;
  if (!h_nH2 || !h_Tgas || !h_Tdust || !h_vlos || !h_cube) return fail(ctx, IRIS_SO_EINVAL, "iris_so_observe_host: NULL pointer");
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const iris_so_config cfg0 = ctx->cfg;
  const int64_t ncell0 = ctx->ncell, npix0 = ctx->npix, nvox0 = ctx->nvox;
  const size_t fb = sizeof(float) * (size_t)ncell0, cb = sizeof(float) * (size_t)nvox0;
  iris_so_status s = ensure(ctx, &ctx->d_stage, 4 * fb + cb, "cudaMalloc(host-path staging)");
  if (s != IRIS_SO_OK) return s;
  float* f[4] = {ctx->d_stage, ctx->d_stage + ncell0, ctx->d_stage + 2 * ncell0, ctx->d_stage + 3 * ncell0};
  float* d_cube = ctx->d_stage + 4 * ncell0;
  const float* h[4] = {h_nH2, h_Tgas, h_Tdust, h_vlos};
  cudaError_t e;
  // slab height: 128 MB of field data per slab (a sixth of the fields for smaller cubes), at least 3 slabs, else one shot
  const size_t row_bytes = (size_t)cfg0.nz * cfg0.nx * sizeof(float) * 4;
  // (measured on the 512^3 cube, 2.1 GB of fields: 16 MB slabs 49.3 ms, 48 MB 48.5, 128 MB 43.3, 256 MB 44.8, 512 MB 47.4;
  // with the last slab tapered as below: 44.6 -> 43.6 ms)
  const size_t slab_bytes = std::min<size_t>((size_t)128 << 20, std::max<size_t>((size_t)16 << 20, 4 * fb / 6));
  int rows = (int)std::max<size_t>(1, slab_bytes / std::max<size_t>(row_bytes, 1));
  rows = std::min(rows, cfg0.ny);
  // the slabs: equal heights, the last one cut into a half, a quarter and two eighths -- what follows the last H2D (K1-K5 and
  // the D2H of that slab) is the part of the pipeline nothing overlaps with
  std::vector<int> slab_y0, slab_ny;
  for (int y = 0; y < cfg0.ny; y += rows) {
    const int h = std::min(rows, cfg0.ny - y);
    if (y + rows >= cfg0.ny && h >= 8) {
      const int parts[4] = {h / 2, h / 4, h / 8, h - h / 2 - h / 4 - h / 8};
      int yy = y;
      for (int q = 0; q < 4; ++q) { slab_y0.push_back(yy); slab_ny.push_back(parts[q]); yy += parts[q]; }
    } else {
      slab_y0.push_back(y); slab_ny.push_back(h);
    }
  }
  const int nslab = (int)slab_y0.size();
  if ((cfg0.ny + rows - 1) / rows < 3) {
    for (int i = 0; i < 4; ++i)
      if ((e = cudaMemcpyAsync(f[i], h[i], fb, cudaMemcpyHostToDevice, st)) != cudaSuccess) return cuda_fail(ctx, e, "H2D copy");
    if ((s = iris_so_observe(ctx, f[0], f[1], f[2], f[3], d_cube, stream)) != IRIS_SO_OK) return s;
    if ((e = cudaMemcpyAsync(h_cube, d_cube, cb, cudaMemcpyDeviceToHost, st)) != cudaSuccess) return cuda_fail(ctx, e, "D2H copy");
    if ((e = cudaStreamSynchronize(st)) != cudaSuccess) return cuda_fail(ctx, e, "cudaStreamSynchronize");
    return IRIS_SO_OK;
  }
  if ((s = ensure(ctx, &ctx->d_coef, sizeof(float) * 6 * (size_t)ncell0, "cudaMalloc(coefficient planes)")) != IRIS_SO_OK) return s;
  if ((s = begin_call(ctx, st)) != IRIS_SO_OK) return s;
  if (!ctx->s_in) {
    if ((e = cudaStreamCreateWithFlags(&ctx->s_in, cudaStreamNonBlocking)) != cudaSuccess) return cuda_fail(ctx, e, "cudaStreamCreate");
    if ((e = cudaStreamCreateWithFlags(&ctx->s_out, cudaStreamNonBlocking)) != cudaSuccess) return cuda_fail(ctx, e, "cudaStreamCreate");
  }
  while ((int)ctx->slab_events.size() < 2 * nslab + 1) {
    cudaEvent_t ev;
    if ((e = cudaEventCreateWithFlags(&ev, cudaEventDisableTiming)) != cudaSuccess) return cuda_fail(ctx, e, "cudaEventCreate");
    ctx->slab_events.push_back(ev);
  }
  const bool post = (cfg0.beam_fwhm_px > 0.0) || ctx->nc.on;
  cudaEvent_t ev_start = ctx->slab_events[2 * nslab];
  iris_so_status rs = IRIS_SO_OK;
  cudaError_t ce = cudaSuccess;
  const char* what = "";
#define HOSTPATH_CU(call, text) do { if (ce == cudaSuccess && rs == IRIS_SO_OK) { ce = (call); if (ce != cudaSuccess) what = (text); } } while (0)
  HOSTPATH_CU(cudaEventRecord(ev_start, st), "cudaEventRecord");
  HOSTPATH_CU(cudaStreamWaitEvent(ctx->s_in, ev_start, 0), "cudaStreamWaitEvent");      // staging may still be in use on st
  HOSTPATH_CU(cudaStreamWaitEvent(ctx->s_out, ev_start, 0), "cudaStreamWaitEvent");
  for (int k = 0; k < nslab; ++k) {
    const int y0 = slab_y0[k], ny_k = slab_ny[k];
    const int64_t cells_before = (int64_t)cfg0.nz * y0 * cfg0.nx;         // compact slabs are stored back to back
    const size_t width = (size_t)ny_k * cfg0.nx * sizeof(float), spitch = (size_t)cfg0.ny * cfg0.nx * sizeof(float);
    for (int i = 0; i < 4; ++i)
      HOSTPATH_CU(cudaMemcpy2DAsync(f[i] + cells_before, width, h[i] + (size_t)y0 * cfg0.nx, spitch, width, (size_t)cfg0.nz,
                                    cudaMemcpyHostToDevice, ctx->s_in), "H2D slab copy");
    HOSTPATH_CU(cudaEventRecord(ctx->slab_events[2 * k], ctx->s_in), "cudaEventRecord");
    HOSTPATH_CU(cudaStreamWaitEvent(st, ctx->slab_events[2 * k], 0), "cudaStreamWaitEvent");
    if (ce != cudaSuccess || rs != IRIS_SO_OK) break;
    // K1-K5 of the slab as a (nx, ny_k, nz) problem
    ctx->cfg.ny = ny_k;
    ctx->npix = (int64_t)ny_k * cfg0.nx; ctx->ncell = ctx->npix * cfg0.nz; ctx->nvox = ctx->npix * cfg0.nv;
    float* cube_k = d_cube + (int64_t)y0 * cfg0.nx * cfg0.nv;
    rs = run_coefficients(ctx, f[0] + cells_before, f[1] + cells_before, f[2] + cells_before, f[3] + cells_before, nullptr, st);
    if (rs == IRIS_SO_OK) rs = run_transfer(ctx, ctx->mc, cube_k, nullptr, st);
    ctx->cfg = cfg0; ctx->ncell = ncell0; ctx->npix = npix0; ctx->nvox = nvox0;
    if (!post) {
      HOSTPATH_CU(cudaEventRecord(ctx->slab_events[2 * k + 1], st), "cudaEventRecord");
      HOSTPATH_CU(cudaStreamWaitEvent(ctx->s_out, ctx->slab_events[2 * k + 1], 0), "cudaStreamWaitEvent");
      HOSTPATH_CU(cudaMemcpyAsync(h_cube + (size_t)y0 * cfg0.nx * cfg0.nv, cube_k, sizeof(float) * (size_t)ny_k * cfg0.nx * cfg0.nv,
                                  cudaMemcpyDeviceToHost, ctx->s_out), "D2H slab copy");
    }
  }
  if (post && ce == cudaSuccess && rs == IRIS_SO_OK) {
    if (cfg0.beam_fwhm_px > 0.0) rs = run_beam(ctx, d_cube, d_cube, nullptr, ctx->nc.on != 0, st);
    else rs = run_noise(ctx, d_cube, st);
    HOSTPATH_CU(cudaMemcpyAsync(h_cube, d_cube, cb, cudaMemcpyDeviceToHost, st), "D2H copy");
  }
#undef HOSTPATH_CU
  // always drain the three streams before returning (also on error: nothing may still be writing h_cube)
  cudaError_t e1 = cudaStreamSynchronize(ctx->s_in), e2 = cudaStreamSynchronize(st), e3 = cudaStreamSynchronize(ctx->s_out);
  if (rs != IRIS_SO_OK) return rs;
  if (ce != cudaSuccess) return cuda_fail(ctx, ce, what);
  if (e1 != cudaSuccess) return cuda_fail(ctx, e1, "cudaStreamSynchronize(copy-in)");
  if (e2 != cudaSuccess) return cuda_fail(ctx, e2, "cudaStreamSynchronize");
  if (e3 != cudaSuccess) return cuda_fail(ctx, e3, "cudaStreamSynchronize(copy-out)");
  return IRIS_SO_OK;
}

iris_so_status iris_so_profile(iris_so_ctx* ctx, int32_t enable) {
  if (!ctx) return IRIS_SO_EINVAL;
  prof_reset(ctx);
  ctx->profiling = enable != 0;
  return IRIS_SO_OK;
}

iris_so_status iris_so_profile_read(iris_so_ctx* ctx, int32_t stage, double* total_ms, uint64_t* launches) {
  if (!ctx) return IRIS_SO_EINVAL;
  if (stage < 0 || stage >= IRIS_SO_NUM_STAGES || !total_ms || !launches)
    return fail(ctx, IRIS_SO_EINVAL, "iris_so_profile_read: bad stage or NULL output");
  double ms = 0.0; uint64_t n = 0;
  for (auto& r : ctx->recs) {
    if (r.stage != stage) continue;
    cudaError_t e = cudaEventSynchronize(r.b);
    float t = 0.0f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&t, r.a, r.b);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "iris_so_profile_read");
    ms += t; n += r.launches;
  }
  *total_ms = ms; *launches = n;
  return IRIS_SO_OK;
}

iris_so_status iris_so_transfer_work(iris_so_ctx* ctx, uint64_t* window_updates, void* stream) {
  if (!ctx) return IRIS_SO_EINVAL;
  if (!window_updates) return fail(ctx, IRIS_SO_EINVAL, "iris_so_transfer_work: NULL output");
  if (!ctx->d_coef) return fail(ctx, IRIS_SO_EINVAL, "iris_so_transfer_work: no coefficient planes yet (call observe / transfer first)");
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  cudaError_t e;
  if (!ctx->d_counter && (e = cudaMalloc(reinterpret_cast<void**>(&ctx->d_counter), sizeof(unsigned long long))) != cudaSuccess)
    return cuda_fail(ctx, e, "cudaMalloc(counter)");
  if ((e = cudaMemsetAsync(ctx->d_counter, 0, sizeof(unsigned long long), st)) != cudaSuccess) return cuda_fail(ctx, e, "memset");
  const int fine_m = ctx->cfg.subsample > 0 ? ctx->cfg.subsample + 1 : 0;
  if (windowed_smooth_mode(ctx->cfg)) {
    iris::hull_work_kernel<<<(unsigned)((ctx->npix + 127) / 128), 128, 0, st>>>(ctx->d_coef, ctx->ncell, (int)ctx->npix, ctx->cfg.nz,
                                                                                ctx->cfg.nv, fine_m, iris::kSmoothKeep, ctx->d_counter);
    IRIS_CHECK_LAUNCH(ctx, "hull_work_kernel");
  } else {
    iris::window_work_kernel<<<(unsigned)((ctx->ncell + 255) / 256), 256, 0, st>>>(ctx->d_coef, ctx->ncell, ctx->cfg.nv, fine_m,
                                                                                   ctx->d_counter);
    IRIS_CHECK_LAUNCH(ctx, "window_work_kernel");
  }
  unsigned long long h = 0;
  if ((e = cudaMemcpyAsync(&h, ctx->d_counter, sizeof h, cudaMemcpyDeviceToHost, st)) != cudaSuccess) return cuda_fail(ctx, e, "D2H");
  if ((e = cudaStreamSynchronize(st)) != cudaSuccess) return cuda_fail(ctx, e, "cudaStreamSynchronize");
  *window_updates = h;
  return IRIS_SO_OK;
}

iris_so_status iris_so_smooth_fallback(iris_so_ctx* ctx, int32_t* fell_back, void* stream) {
  if (!ctx) return IRIS_SO_EINVAL;
  if (!fell_back) return fail(ctx, IRIS_SO_EINVAL, "iris_so_smooth_fallback: NULL output");
  *fell_back = 0;
  if (!ctx->d_gate || !uses_handover(ctx->cfg)) return IRIS_SO_OK;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  int h = 0;
  cudaError_t e;
  if ((e = cudaMemcpyAsync(&h, ctx->d_gate + 1, sizeof h, cudaMemcpyDeviceToHost, st)) != cudaSuccess) return cuda_fail(ctx, e, "D2H");
  if ((e = cudaStreamSynchronize(st)) != cudaSuccess) return cuda_fail(ctx, e, "cudaStreamSynchronize");
  *fell_back = h;
  return IRIS_SO_OK;
}

iris_so_status iris_so_beam(iris_so_ctx* ctx, const float* d_in, float* d_out, float* d_tmp, void* stream) {
  if (!ctx) return IRIS_SO_EINVAL;
  if (!d_in || !d_out) return fail(ctx, IRIS_SO_EINVAL, "iris_so_beam: NULL pointer");
  if (!(ctx->cfg.beam_fwhm_px > 0.0)) return fail(ctx, IRIS_SO_EINVAL, "iris_so_beam: no beam configured");
  return run_beam(ctx, d_in, d_out, d_tmp, false, static_cast<cudaStream_t>(stream));
}

iris_so_status iris_so_noise(iris_so_ctx* ctx, float* d_cube, void* stream) {
  if (!ctx) return IRIS_SO_EINVAL;
  if (!d_cube) return fail(ctx, IRIS_SO_EINVAL, "iris_so_noise: NULL pointer");
  if (!ctx->nc.on) return IRIS_SO_OK;
  return run_noise(ctx, d_cube, static_cast<cudaStream_t>(stream));
}

static iris_so_status observe_adjoint_impl(iris_so_ctx* ctx, const float* d_nH2, const float* d_Tgas, const float* d_Tdust,
                                          const float* d_vlos, const float* d_w, float* d_grad, void* stream,
                                          bool wrt_abundance) {
  if (!ctx) return IRIS_SO_EINVAL;
  if (!d_nH2 || !d_Tgas || !d_Tdust || !d_vlos || !d_w || !d_grad)
    return fail(ctx, IRIS_SO_EINVAL, "iris_so_observe_adjoint: NULL pointer");
  const iris_so_config& c = ctx->cfg;
  if ((c.subtract_continuum && c.subtract_space != 0) || c.out_unit == 2)
    return fail(ctx, IRIS_SO_EUNSUPPORTED, "adjoint needs intensity-space subtraction and out_unit 0 or 1");
  // the hot-path mode has the windowed closed-form adjoint (adjoint_kernels.cuh); the thick mode with the smooth integrator
  // and / or the fine grid the stored-state reverse sweep of adjoint_modes.cuh; the thin modes have none
  const bool modes_adjoint = c.transfer_mode == 0 && !hot_path_mode(c);
  if (c.transfer_mode != 0)
    return fail(ctx, IRIS_SO_EUNSUPPORTED, "adjoint is implemented for the optically thick transfer mode only");
  if (c.coef_grid == 1)
    return fail(ctx, IRIS_SO_EUNSUPPORTED, "adjoint differentiates the per-cell level solve: not available with coef_grid = 1");
  if (c.dust_per_channel)
    return fail(ctx, IRIS_SO_EUNSUPPORTED, "adjoint is not available with dust_per_channel = 1");
  // the adjoint march keeps five spectra per pixel in shared memory (one warp per pixel beyond 384 channels)
  if (!modes_adjoint &&
      (size_t)5 * (((size_t)c.nv + 31) / 32 * 32) * sizeof(float) + (size_t)iris::kAdjRecFields * 32 * sizeof(float4) > 227u * 1024u)
    return fail(ctx, IRIS_SO_EUNSUPPORTED, "adjoint: five spectra of this many channels do not fit the shared memory of an SM");
  // the reverse sweep of the other modes stages a column's coefficients and accumulators in shared memory
  if (modes_adjoint && iris::kAdjModesWarps * iris::adjoint_modes_smem_per_warp(c.nz) > 227u * 1024u)
    return fail(ctx, IRIS_SO_EUNSUPPORTED, "adjoint: a column of this many cells does not fit the shared memory of an SM");
  if (modes_adjoint && (size_t)c.nv * (size_t)(c.subsample + 1) + 1 > 65535u)
    return fail(ctx, IRIS_SO_EUNSUPPORTED, "adjoint: more than 65535 spectral points per pixel");
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  iris_so_status s = run_coefficients(ctx, d_nH2, d_Tgas, d_Tdust, d_vlos, nullptr, st);
  if (s != IRIS_SO_OK) return s;
  // scratch: d(e_c)/dn and d(a_c)/dn per cell, then (with a beam) what = G^T w -- the beam is symmetric and zero
  // padded, so its adjoint is the same convolution
  const size_t dcoef_floats = 2 * (size_t)ctx->ncell;
  // (other modes: + the stored states of the forward sweep, one slab per resident warp)
  const int modes_grid = modes_adjoint ? iris::adjoint_modes_grid(ctx->sm_count, c.nz) : 0;
  const size_t states_floats =
      modes_adjoint ? (size_t)modes_grid * iris::kAdjModesWarps * iris::adjoint_modes_scratch_per_warp(c.nz) / sizeof(float) : 0;
  const size_t need = sizeof(float) * (dcoef_floats + (c.beam_fwhm_px > 0.0 ? (size_t)ctx->nvox : 0) + states_floats);
  if (ctx->d_adj && ctx->adj_bytes < need) { cudaFree(ctx->d_adj); ctx->d_adj = nullptr; ctx->scratch_bytes -= ctx->adj_bytes; }
  if ((s = ensure(ctx, &ctx->d_adj, need, "cudaMalloc(adjoint scratch)")) != IRIS_SO_OK) return s;
  ctx->adj_bytes = need;
  float* dcoef = ctx->d_adj;
  const float* what = d_w;
  if (c.beam_fwhm_px > 0.0) {
    float* wb = ctx->d_adj + dcoef_floats;
    if ((s = run_beam(ctx, d_w, wb, nullptr, false, st)) != IRIS_SO_OK) return s;
    what = wb;
  }
  ProfScope prof(ctx, IRIS_SO_STAGE_ADJOINT, st);
  iris::AdjointConsts ac = ctx->ac;
  if (wrt_abundance) ac.c_d = 0.0f;                    // the dust does not depend on the tracer abundance
  if (modes_adjoint) {
    cudaError_t e = cudaSuccess;
    if (!wrt_abundance) {
      e = iris::launch_coef_grad_levels(ctx->lc, ac, c.n_levels, ctx->band, ctx->ncell, d_nH2, d_Tgas, dcoef, st);
      if (e != cudaSuccess) return cuda_fail(ctx, e, "launch of coef_grad_kernel");
      ++ctx->launches;
    }
    float* states = ctx->d_adj + dcoef_floats + (c.beam_fwhm_px > 0.0 ? (size_t)ctx->nvox : 0);
    e = iris::launch_adjoint_modes(ctx->mc, ac, c.integration == 1, c.subsample > 0 ? c.subsample + 1 : 0, ctx->d_coef,
                                   wrt_abundance ? ctx->d_coef : dcoef, ctx->ncell, (int)ctx->npix, c.nz, c.nv, what, states,
                                   d_grad, modes_grid, st);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "launch of adjoint_modes_kernel");
    ++ctx->launches;
    return IRIS_SO_OK;
  }
  cudaError_t e = iris::launch_adjoint(ctx->mc, ac, ctx->lc, c.n_levels, ctx->band, ctx->d_coef, dcoef, ctx->ncell, (int)ctx->npix,
                                       c.nz, c.nv, c.dust_on != 0, resolved_algo(c) == IRIS_SO_ALGO_WINDOW, d_nH2, d_Tgas, what,
                                       d_grad, st, &ctx->launches, wrt_abundance);
  if (e != cudaSuccess) return cuda_fail(ctx, e, "launch of adjoint kernels");
  return IRIS_SO_OK;
}

iris_so_status iris_so_observe_adjoint(iris_so_ctx* ctx, const float* d_nH2, const float* d_Tgas, const float* d_Tdust,
                                       const float* d_vlos, const float* d_w, float* d_grad, void* stream) {
  return observe_adjoint_impl(ctx, d_nH2, d_Tgas, d_Tdust, d_vlos, d_w, d_grad, stream, false);
}

iris_so_status iris_so_observe_adjoint_abundance(iris_so_ctx* ctx, const float* d_nH2, const float* d_Tgas,
                                                 const float* d_Tdust, const float* d_vlos, const float* d_w,
                                                 float* d_grad, void* stream) {
  return observe_adjoint_impl(ctx, d_nH2, d_Tgas, d_Tdust, d_vlos, d_w, d_grad, stream, true);
}

iris_so_status iris_so_density_trace(iris_so_ctx* ctx, const float* d_nH2, const float* d_vlos, float* d_cube, void* stream) {
  if (!ctx) return IRIS_SO_EINVAL;
  if (!d_nH2 || !d_vlos || !d_cube) return fail(ctx, IRIS_SO_EINVAL, "iris_so_density_trace: NULL pointer");
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const iris_so_config& c = ctx->cfg;
  cudaError_t e = cudaMemsetAsync(d_cube, 0, sizeof(float) * (size_t)ctx->nvox, st);
  if (e != cudaSuccess) return cuda_fail(ctx, e, "cudaMemsetAsync(cube)");
  iris::density_trace_kernel<<<(unsigned)((ctx->npix + 127) / 128), 128, 0, st>>>(
      d_nH2, d_vlos, (int)ctx->npix, c.nz, c.nv, c.v0_cms, c.dv_cms, (float)(c.cell_cm / c.dv_cms), d_cube);
  IRIS_CHECK_LAUNCH(ctx, "density_trace_kernel");
  return IRIS_SO_OK;
}

iris_so_status iris_so_metrics(iris_so_ctx* ctx, const float* d_T1, const float* d_T2, double T_min, double* h_out, void* stream) {
  if (!ctx) return IRIS_SO_EINVAL;
  if (!d_T1 || !d_T2 || !h_out) return fail(ctx, IRIS_SO_EINVAL, "iris_so_metrics: NULL pointer");
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const iris_so_config& c = ctx->cfg;
  if (!(T_min > 0.0)) T_min = 5.0e-2;
  cudaError_t e;
  if (!ctx->d_metrics && (e = cudaMalloc(reinterpret_cast<void**>(&ctx->d_metrics), 9 * sizeof(double))) != cudaSuccess)
    return cuda_fail(ctx, e, "cudaMalloc(metrics)");
  double init[9] = {0, 0, 0, 0, 0, -INFINITY, -INFINITY, 0, 0};
  if ((e = cudaMemcpyAsync(ctx->d_metrics, init, sizeof init, cudaMemcpyHostToDevice, st)) != cudaSuccess) return cuda_fail(ctx, e, "H2D");
  if ((e = cudaStreamSynchronize(st)) != cudaSuccess) return cuda_fail(ctx, e, "cudaStreamSynchronize");   // init is a stack array
  iris::metrics_pixel_kernel<<<(unsigned)((ctx->npix * 32 + 255) / 256), 256, 0, st>>>(d_T1, d_T2, (int)ctx->npix, c.nv, T_min,
                                                                                   ctx->d_metrics);
  IRIS_CHECK_LAUNCH(ctx, "metrics_pixel_kernel");
  const int64_t nlv = (int64_t)c.nx * c.nv;
  iris::metrics_lv_kernel<<<(unsigned)((nlv + 255) / 256), 256, 0, st>>>(d_T1, d_T2, c.ny, c.nx, c.nv, T_min, ctx->d_metrics);
  IRIS_CHECK_LAUNCH(ctx, "metrics_lv_kernel");
  double r[9];
  if ((e = cudaMemcpyAsync(r, ctx->d_metrics, sizeof r, cudaMemcpyDeviceToHost, st)) != cudaSuccess) return cuda_fail(ctx, e, "D2H");
  if ((e = cudaStreamSynchronize(st)) != cudaSuccess) return cuda_fail(ctx, e, "cudaStreamSynchronize");
  h_out[0] = r[0] / (double)ctx->nvox;
  h_out[1] = r[1] / (double)ctx->npix;
  h_out[2] = r[2] / (double)nlv;
  h_out[3] = r[7] > 0.0 ? r[3] / r[7] : 0.0;
  h_out[4] = r[8] > 0.0 ? r[4] / r[8] : 0.0;
  h_out[5] = r[5]; h_out[6] = r[6]; h_out[7] = r[7]; h_out[8] = r[8];
  return IRIS_SO_OK;
}

}  // extern "C"
