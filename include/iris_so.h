/* iris_so.h -- C ABI of the B200-native (sm_100a) IRIS-SO hot path.
 *
 * The library computes, entirely in hand-written CUDA kernels, the synthetic-observation hot path of
 * arxiv/paper_2607_01338 (IRIS-SO, PAPER.md sections 3-4):
 *
 *   per cell   optically-thin level balance  (Eq. 3.6.1-3.6.3, 3.7.1-3.7.2)
 *   per cell   line + dust coefficients      (Eq. 3.3.1-3.3.4, 3.2.1-3.2.2)
 *   per ray    formal solution of the transfer equation for every velocity channel with the
 *              channel-integrated (erf) profile (Eq. 4.8.5-4.8.7, 4.6.3-4.6.4, 4.4.1)
 *   per voxel  continuum subtraction and unit conversion (section 4.9-4.10)
 *   per cube   Gaussian beam (section 4.11) and seeded noise (Eq. 4.12.1)
 *   optional   reverse-scan adjoint d(sum w * cube) / d n_H2 (section 4 intro)
 *
 * Conventions
 *   - Pointers named d_* are CUDA DEVICE pointers, pointers named h_* are HOST pointers; all are owned
 *     by the caller.  The library never allocates or frees caller buffers.  A context owns only its
 *     private scratch (per-cell coefficient planes, one cube-sized temporary when the beam is on).
 *   - All field arrays are float32 [nz][ny][nx] (x fastest); rays march along z and k = 0 is the FAR
 *     side (the background enters there), k = nz-1 is nearest the observer.
 *   - All cube arrays are float32 [ny][nx][nv] (velocity channel fastest).
 *   - Units are CGS.  v_los > 0 means receding gas; a cell emits at channel velocity v = v_los
 *     (radio convention; velocity-space reading of Eq. 4.3.1).
 *   - Every d_* call is asynchronous on `cuda_stream` (a cudaStream_t passed as void*; NULL = the
 *     legacy default stream) and never synchronises the device.  h_* calls synchronise the stream
 *     before returning.
 *   - Argument errors return IRIS_SO_EINVAL before any launch; CUDA failures return IRIS_SO_ECUDA /
 *     IRIS_SO_ENOMEM.  iris_so_last_error() gives the text.  No exception crosses the ABI.
 *   - There is no CPU fallback: without a CUDA device iris_so_create fails with IRIS_SO_ECUDA.
 *   - A context is not thread-safe; use one per host thread / stream.
 */
#ifndef IRIS_SO_H_
#define IRIS_SO_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define IRIS_SO_VERSION 100     /* 0.1.0 */
#define IRIS_SO_MAX_LEVELS 10

typedef struct iris_so_ctx iris_so_ctx; /* opaque */

typedef enum {
  IRIS_SO_OK = 0,
  IRIS_SO_EINVAL = 1,        /* bad argument or configuration */
  IRIS_SO_EUNSUPPORTED = 2,  /* valid but not implemented combination */
  IRIS_SO_ECUDA = 3,         /* CUDA runtime / launch failure, or no device */
  IRIS_SO_ENOMEM = 4         /* device or host allocation failed */
} iris_so_status;

/* transfer_algo */
#define IRIS_SO_ALGO_AUTO 0     /* = IRIS_SO_ALGO_WINDOW */
#define IRIS_SO_ALGO_DENSE 1    /* every (cell, channel) update evaluated; register-resident channel blocks */
#define IRIS_SO_ALGO_WINDOW 2   /* only channels inside each cell's line window are updated; exact in fp32.
                                 * Profile from the channel-centre expansion when dv / xi <= 0.55 (every cell then
                                 * has dv / b <= 0.55), otherwise from erfc at the channel edges */
#define IRIS_SO_ALGO_WINDOW_EDGE 3 /* line window with the erfc-at-the-edges profile for any channel width */

typedef struct {
  /* grid: rays = z columns.  The paper's observer-centred spherical lattice (l, b, r) with r sampled "at regular
   * intervals" IS this layout: x = l, y = b, z = r with k = 0 the far end of the ray and cell_cm the
   * radial step (every ray of the lattice is a column with a constant step; the cube comes out as [b][l][v]). */
  int32_t nx, ny, nz;
  double cell_cm;               /* step h along the ray (Eq. 4.8.7) */
  /* molecule (the paper reads these from a LAMDA file); host arrays, copied by create */
  int32_t n_levels;             /* 2 .. IRIS_SO_MAX_LEVELS */
  const double *energy_K;       /* [n_levels]  E_i / k, ascending */
  const double *weight;         /* [n_levels]  statistical weights g_i */
  const double *einstein_A;     /* [n_levels * n_levels]  A[u*n + l] (1/s) for u > l, else 0 */
  const double *coll_down_ref;  /* [n_levels * n_levels]  K_ul(T_ref) (cm^3/s) for u > l, else 0 */
  double coll_T_ref, coll_T_exp;/* K_ul(T) = K_ul(T_ref) (T / T_ref)^coll_T_exp; upward by Eq. 3.7.2 */
  int32_t line_upper, line_lower;
  double nu0_Hz;                /* frequency of the observed transition */
  double mol_mass_g;            /* m_a of Eq. 3.3.4 */
  double abundance;             /* tracer molecules per H2 (Eq. 4.2.1) */
  double microturb_cms;         /* xi: b^2 = 2 k T / m_a + xi^2; 0 = thermal only */
  double T_bar;                 /* level-balance radiation temperature (Eq. 3.6.2); 0 = none */
  double T_cmb;                 /* transfer background temperature */
  double T_inf;                 /* no line above this gas temperature; +inf = off */
  /* dust (Eq. 3.2.1-3.2.2) */
  int32_t dust_on;
  double kappa_gas_cm2_g;       /* opacity per gram of GAS (gas-to-dust ratio folded in) */
  double mass_per_H2_g;         /* rho_gas = mass_per_H2_g * n_H2 */
  /* channel grid: channel k has centre v0 + k dv and width dv (Eq. 4.4.1) */
  int32_t nv;
  double v0_cms, dv_cms;
  /* post-processing */
  int32_t subtract_continuum;   /* 1: cube = total - continuum (section 4.10) */
  int32_t subtract_space;       /* 0: intensity / Rayleigh-Jeans space, 1: Planck brightness-temperature space */
  int32_t out_unit;             /* 0: intensity (cgs), 1: T_RJ (Eq. 4.9.2), 2: Planck T_B (Eq. 4.9.1) */
  double beam_fwhm_px;          /* Gaussian beam FWHM in pixels; 0 = off (section 4.11) */
  double noise_mu, noise_sigma; /* Eq. 4.12.1, in the output unit; both 0 = off */
  int32_t noise_gamma_mode;     /* 0: gamma = 1; 1: one gamma ~ U[0,1) per cube */
  uint64_t seed;                /* noise seed (Philox4x32-10 key) */
  /* implementation choice, does not change the mathematics */
  int32_t transfer_algo;        /* IRIS_SO_ALGO_* */
  /* The paper's other transfer / integration modes (sections 4.4 - 4.8).  All three 0 = the hot
   * path above (optically thick, formal integration, channel-integrated profile).  Any other combination runs a
   * line-window kernel of its own or transfer_modes_kernel (iris_so_transfer_kernel names it).  The gradient entry
   * points serve transfer_mode = 0 with every integration / subsample; transfer_mode 1 and 2: IRIS_SO_EUNSUPPORTED. */
  int32_t transfer_mode;        /* 0 optically thick (4.5), 1 selectively thin (4.6, Eq. 4.8.13-4.8.15),
                                 * 2 optically thin (4.7, Eq. 4.7.3-4.7.5) */
  int32_t integration;          /* 0 formal (Eq. 4.8.5 / 4.7.6), 1 smooth (trapezoidal first step Eq. 4.8.12 + BDF2
                                 * Eq. 4.8.10 with the ReLU of PAPER.md:709; Simpson along the ray Eq. 4.7.7 in thin mode) */
  int32_t subsample;            /* thick mode only: 0 = channel-integrated profile (Eq. 4.6.3); odd f >= 1 = point
                                 * profile (Eq. 3.3.3) on a fine velocity grid with f added midpoints per channel,
                                 * averaged over the channel by Simpson's rule (Eq. 4.5.1) */
  /* Tabulated collision rates of several partners (LAMDA tables interpolated in temperature; H,
   * para-H2, ortho-H2 at 3:1, He at 0.1 per H).  coll_n_partners = 0: the power law coll_down_ref (T / T_ref)^exp above.
   * Otherwise K_ul(T) = sum_p coll_partner_frac[p] * K^p_ul(T) per unit n_H2, every table interpolated linearly in T
   * between its grid points and held constant outside the grid; coll_down_ref / coll_T_ref / coll_T_exp are ignored.
   * Host arrays, copied by create. */
  int32_t coll_n_partners;          /* 0 .. 8 */
  int32_t coll_nT;                  /* 1 .. 64 grid temperatures */
  const double *coll_T_grid;        /* [coll_nT] strictly ascending, > 0 */
  const double *coll_table;         /* [coll_n_partners][coll_nT][n_levels * n_levels] K_ul (cm^3/s) for u > l, else 0 */
  const double *coll_partner_frac;  /* [coll_n_partners] number density of the partner per n_H2, >= 0 */
  /* Grid precomputation (section 4.2) and lookup (section 4.3).  coef_grid = 0: the
   * level balance is solved per cell (K1).  coef_grid = 1: iris_so_create tabulates the line coefficients per tracer
   * abundance (Eq. 4.2.1) on grid_n_density x grid_n_temp nodes, spaced geometrically from grid_nH2_lo to grid_nH2_hi and
   * from grid_T_lo to grid_T_hi, with their finite-difference gradients, and observe / transfer interpolate them:
   * multilinear in n_H2 and T_gas inside the grid cell that holds the point, the edge cell's form continued outside
   * the grid; abundance and the T_inf mask are applied after the lookup.  (The paper's third axis, the H2 abundance,
   * has one node here: the fields carry n_H2 and the partner fractions are configuration constants.)  The lookup
   * replaces K1 only in calls that solve the populations internally; iris_so_levelpop is unaffected, and the adjoint
   * entry points return IRIS_SO_EUNSUPPORTED. */
  int32_t coef_grid;
  int32_t grid_n_density, grid_n_temp;   /* 2 .. 4096 nodes each (paper: 128, 64) */
  double grid_nH2_lo, grid_nH2_hi;       /* 0 < lo < hi, cm^-3 */
  double grid_T_lo, grid_T_hi;           /* 0 < lo < hi, K */
  /* 0: the dust source B_nu(T_dust), the background B_nu(T_cmb) and the unit conversion are taken at nu0 (the continuum
   * is one value per pixel).  1: at every channel's own frequency ("the Doppler-shifted Planck source
   * function"): channel k is observed at nu_k = nu0 (1 - v_k / c) and the dust of a cell moving with v_los emits at
   * nu_k (1 + v_los / c) in its own frame; the dust opacity stays constant over the band.  Hot-path mode only
   * (transfer_mode = integration = subsample = 0; else create returns IRIS_SO_EUNSUPPORTED); runs through the dense
   * kernel; iris_so_transfer then takes d_I_cont = NULL only (the continuum is a spectrum), the adjoint entry points
   * return IRIS_SO_EUNSUPPORTED. */
  int32_t dust_per_channel;
} iris_so_config;

/* Validates and copies the configuration (including the host arrays), selects the current CUDA device.
 * On failure *out is NULL; the text is available through iris_so_last_error(NULL). */
iris_so_status iris_so_create(const iris_so_config *cfg, iris_so_ctx **out);
void iris_so_destroy(iris_so_ctx *ctx);

/* Text of the last error of this context (or of the last failed create if ctx is NULL).
 * Valid until the next call on the same context. */
const char *iris_so_last_error(const iris_so_ctx *ctx);
const char *iris_so_status_string(iris_so_status s);
int iris_so_version(void);

/* Number of kernels this context has launched so far (for launch accounting in benchmarks). */
uint64_t iris_so_launch_count(const iris_so_ctx *ctx);

/* Bytes of device scratch the context holds after its first observe / transfer call. */
uint64_t iris_so_scratch_bytes(const iris_so_ctx *ctx);

/* K1.  Level fractions x_i (sum_i x_i = 1) of every cell: Eq. 3.6.1 with the ground-state row replaced
 * by the conservation equation, radiation field B_nu(T_bar), collisions with H2 only (Eq. 3.6.3).
 * d_pop is [n_levels][n_cells] float32, n_cells = nx*ny*nz. */
iris_so_status iris_so_levelpop(iris_so_ctx *ctx, const float *d_nH2, const float *d_Tgas, float *d_pop,
                                void *cuda_stream);

/* K2 + K3 + K4.  Coefficients and formal transfer.  d_pop may be NULL (populations solved internally,
 * never written) or the output of iris_so_levelpop.  Outputs are specific intensities in CGS
 * (erg s^-1 cm^-2 Hz^-1 sr^-1): d_I_total [ny][nx][nv] is the channel-averaged total intensity
 * (Eq. 3.1.2), d_I_cont [ny][nx] the continuum baseline (Eq. 3.1.3); either may be NULL. */
iris_so_status iris_so_transfer(iris_so_ctx *ctx, const float *d_nH2, const float *d_Tgas,
                                const float *d_Tdust, const float *d_vlos, const float *d_pop,
                                float *d_I_total, float *d_I_cont, void *cuda_stream);

/* K1 .. K7.  Whole path: cube [ny][nx][nv] in `out_unit`, continuum-subtracted if configured, then beam
 * and noise if configured (stage order of PAPER.md:467). */
iris_so_status iris_so_observe(iris_so_ctx *ctx, const float *d_nH2, const float *d_Tgas,
                               const float *d_Tdust, const float *d_vlos, float *d_cube, void *cuda_stream);

/* Same as iris_so_observe with `stage_mask` overriding the configured post-processing:
 * bit 0 = apply the beam, bit 1 = apply the noise (each only if configured). */
iris_so_status iris_so_observe_stages(iris_so_ctx *ctx, const float *d_nH2, const float *d_Tgas,
                                      const float *d_Tdust, const float *d_vlos, int32_t stage_mask,
                                      float *d_cube, void *cuda_stream);

/* K1 .. K5 without any allocation, for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid it): the raw cube of iris_so_observe_stages(..., stage_mask = 0, ...) -- no beam, no noise
 * -- for the hot-path mode (transfer_mode = integration = subsample = 0, coef_grid = 0, dust_per_channel = 0).  The six
 * coefficient planes K1 + K2 hand to K3 live in a file-scope `static __device__` array of the library instead of the
 * context's cudaMalloc'ed scratch: 6 * IRIS_SO_STATIC_MAX_CELLS floats = 12 MiB, held by every GPU that loads the library
 * until the process exits.  nx * ny * nz > IRIS_SO_STATIC_MAX_CELLS returns IRIS_SO_EUNSUPPORTED (message in
 * iris_so_last_error).  The call makes no cudaMalloc / cudaFree / cudaHostAlloc and no allocating library call; it launches
 * K1 + K2 and one transfer kernel on `cuda_stream` and returns without synchronising.  The array is shared by EVERY call
 * of every context on that GPU and keeps the last call's planes: each call overwrites all 6 * ncell entries it reads
 * before reading them (nothing has to start at zero), but two calls that overlap on the GPU (different streams, or
 * different contexts / host threads) race on it -- serialise them.  The device of the context must be current, as for
 * every other call.  Same layouts as iris_so_observe. */
#define IRIS_SO_STATIC_MAX_CELLS (1 << 19)
iris_so_status iris_so_observe_raw_static(iris_so_ctx *ctx, const float *d_nH2, const float *d_Tgas,
                                          const float *d_Tdust, const float *d_vlos, float *d_cube,
                                          void *cuda_stream);

/* Whole path with HOST buffers (pinned or pageable): copies the four fields to the device, runs
 * iris_so_observe, copies the cube back and synchronises.  h_* fields [nz][ny][nx], h_cube [ny][nx][nv]. */
iris_so_status iris_so_observe_host(iris_so_ctx *ctx, const float *h_nH2, const float *h_Tgas,
                                    const float *h_Tdust, const float *h_vlos, float *h_cube,
                                    void *cuda_stream);

/* K8 + K9.  Gradient of L = sum_{y,x,v} w * cube (noise-free cube, beam applied if configured) with
 * respect to n_H2 of every cell, by a reverse scan along every ray (the pipeline is
 * differentiable end to end).  Requires subtract_space = 0, out_unit 0 or 1 and the optically thick transfer mode
 * (transfer_mode = 0), with either integration and any subsample: the hot-path mode has a closed-form windowed
 * adjoint, the smooth integrator (Eq. 4.8.10 / 4.8.12 with the ReLU) and the fine grid (Eq. 4.5.1) a stored-state
 * reverse sweep whose scratch is sized by the resident warps, not by the cube.  Not available with coef_grid = 1 or
 * dust_per_channel = 1 (IRIS_SO_EUNSUPPORTED).  d_w [ny][nx][nv], d_grad_nH2 [nz][ny][nx]. */
iris_so_status iris_so_observe_adjoint(iris_so_ctx *ctx, const float *d_nH2, const float *d_Tgas,
                                       const float *d_Tdust, const float *d_vlos, const float *d_w,
                                       float *d_grad_nH2, void *cuda_stream);

/* Abundance-only gradient: d L / d ln X_c of the same L for a per-cell factor X_c on the tracer abundance
 * (the level fractions do not depend on it, Eq. 4.2.1); the sum over cells is the derivative with respect to the
 * logarithm of the global abundance.  Same requirements and layouts as iris_so_observe_adjoint. */
iris_so_status iris_so_observe_adjoint_abundance(iris_so_ctx *ctx, const float *d_nH2, const float *d_Tgas,
                                                 const float *d_Tdust, const float *d_vlos, const float *d_w,
                                                 float *d_grad_lnX, void *cuda_stream);

/* Measurement support.  iris_so_profile(ctx, 1) makes every later call bracket each stage's kernels with
 * CUDA events on the caller's stream (no synchronisation); iris_so_profile(ctx, 0) switches it off; both
 * discard what was recorded.  iris_so_profile_read waits for the recorded events and returns the summed
 * device time and the number of kernel launches of one stage since profiling was switched on. */
#define IRIS_SO_STAGE_CELL 0      /* K1 + K2 */
#define IRIS_SO_STAGE_TRANSFER 1  /* K3 + K4 + K5 */
#define IRIS_SO_STAGE_BEAM 2      /* K6 (+ K7 fused) */
#define IRIS_SO_STAGE_NOISE 3     /* K7 alone */
#define IRIS_SO_STAGE_ADJOINT 4   /* K8 + K9 */
#define IRIS_SO_NUM_STAGES 5
iris_so_status iris_so_profile(iris_so_ctx *ctx, int32_t enable);
iris_so_status iris_so_profile_read(iris_so_ctx *ctx, int32_t stage, double *total_ms, uint64_t *launches);

/* Work counter for roofline accounting: number of (cell, channel) updates inside the line windows of the
 * coefficient planes left in the context by the last transfer / observe call (the updates the line-window
 * algorithm evaluates; the dense algorithm evaluates nx*ny*nz*nv).  With subsample > 0 the windows are counted in
 * points of the fine velocity grid; with the smooth integrator on its line-window kernel (integration = 1, thick mode)
 * the count is that of the points the kernel steps: per cell the hull of the windows of the last 12 cells.
 * Synchronises the stream. */
iris_so_status iris_so_transfer_work(iris_so_ctx *ctx, uint64_t *window_updates, void *cuda_stream);

/* Name of the LOS transfer kernel this context launches ("transfer_series_kernel", "transfer_window_kernel",
 * "transfer_dense_kernel", "transfer_modes_kernel" or "transfer_smooth_window_kernel"); static storage. */
const char *iris_so_transfer_kernel(const iris_so_ctx *ctx);

/* The optically thick mode with the smooth integrator (integration = 1; trapezoidal + BDF2 steps with the ReLU of
 * PAPER.md:709) is marched over line windows; the march of a pixel is exact unless a ReLU fires outside its windows or
 * the dust is so opaque per cell (a sustained tau_d above ~0.1) that a point the windows have left has not yet settled
 * on the dominant solution of the homogeneous BDF2 step (Eq. 4.8.10), both of which the kernel detects per
 * pixel: it lists the pixel, and the dense kernel, launched right after it and driven by that list, recomputes the
 * listed pixels.  *fell_back = the number of pixels that were handed over in the last transfer / observe call of this
 * context (for iris_so_observe_host: summed over the slabs of pixel rows of that call).
 * The hot path hands pixels over too: its line-window kernel keeps, per pixel, a circular buffer of half the band
 * ("reachable-range spectra": a pixel's lines only touch the channels its line-of-sight velocities reach) whenever that
 * lets more warps stay resident, and a pixel whose lines span more than the buffer is recomputed by the same kernel with
 * whole spectra; the count is reported here as well (the library stops using the buffers once more than 3 % of the
 * pixels of a launch had to be recomputed).  0 for every other mode.  Synchronises the stream. */
iris_so_status iris_so_smooth_fallback(iris_so_ctx *ctx, int32_t *fell_back, void *cuda_stream);

/* Stand-alone post-processing stages (also used inside iris_so_observe). */
/* K6: separable Gaussian beam of FWHM beam_fwhm_px on d_in -> d_out (must not alias), zero padding,
 * radius ceil(4 sigma), weights normalised to sum 1.  d_tmp is a cube-sized temporary or NULL (context
 * scratch is used). */
iris_so_status iris_so_beam(iris_so_ctx *ctx, const float *d_in, float *d_out, float *d_tmp,
                            void *cuda_stream);
/* K7: d_cube += gamma (mu + sigma z), z = Box-Muller of Philox4x32-10(key = seed, counter = voxel index). */
iris_so_status iris_so_noise(iris_so_ctx *ctx, float *d_cube, void *cuda_stream);

/* Diagnostics of PAPER.md section 5.
 * Density tracing ("simple observation", section 5.10): d_cube [ny][nx][nv] = column density per
 * unit velocity, cm^-2 per (cm/s): every cell adds n_H2 * cell_cm / dv_cms to the channel that contains its v_los
 * (channel k covers [v0 + (k - 1/2) dv, v0 + (k + 1/2) dv)); cells outside the band add nothing.  Asynchronous. */
iris_so_status iris_so_density_trace(iris_so_ctx *ctx, const float *d_nH2, const float *d_vlos, float *d_cube,
                                     void *cuda_stream);
/* Error metrics of section 5.1 (Eq. 5.1.1 - 5.1.5) of two cubes [ny][nx][nv] (l = x, b = y):
 * h_out[9] = { mean-TSRE over voxels, mean-TSRE of the l-b images (cube means over v), mean-TSRE of the l-v images
 * (cube means over y), TAM(T1), TAM(T2), max T1, max T2, active voxels of T1, of T2 }; TSRE counts 0 where either
 * |T| <= T_min, the means run over all elements, TAM of a cube without active voxels is 0.  T_min <= 0 selects the
 * paper's 5e-2 K.  Synchronises the stream. */
iris_so_status iris_so_metrics(iris_so_ctx *ctx, const float *d_T1, const float *d_T2, double T_min, double *h_out,
                               void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* IRIS_SO_H_ */
