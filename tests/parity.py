"""Parity criteria between the CUDA path and the oracle (BASELINE.json north_star).

* level populations: component-wise relative error <= 1e-5 wherever x_oracle >= 1e-30, absolute 1e-35 below;
* spectra: per pixel, max_v |dT| <= 1e-4 * max_v |T_oracle| + 1e-6 K  (in the cube's unit; for intensity
  cubes the 1e-6 K floor is converted with the Rayleigh-Jeans factor);
* totals that are not continuum-subtracted additionally allow the fp32 storage rounding of the value itself;
* noise: + 8e-6 * sigma (fp32 log / sqrt / cospi of the Box-Muller transform at |z| <= 5.5).
"""
import numpy as np

KB, CL = 1.380649e-16, 2.99792458e10


def krj(nu0):
    """Kelvin per unit CGS intensity (Eq. 4.9.2)."""
    return CL ** 2 / (2.0 * KB * nu0 ** 2)


def pop_errors(pop_gpu, pop_ora):
    g = np.asarray(pop_gpu, dtype=np.float64)
    o = np.asarray(pop_ora, dtype=np.float64)
    big = o >= 1e-30
    rel = np.zeros_like(o)
    rel[big] = np.abs(g[big] / o[big] - 1.0)
    absmax = float(np.abs(g[~big] - o[~big]).max()) if (~big).any() else 0.0
    return float(rel.max()), absmax


def assert_pops(pop_gpu, pop_ora, rel_tol=1e-5):
    rel, absmax = pop_errors(pop_gpu, pop_ora)
    assert rel <= rel_tol, "max component-wise relative population error %.3g > %.1g" % (rel, rel_tol)
    assert absmax <= 1e-35, "absolute error %.3g on populations below 1e-30" % absmax
    return rel


def spectrum_excess(gpu, ora, floor=1e-6, rel=1e-4, extra=0.0, peak_of=None):
    """Per-pixel max_v(|gpu - ora| - extra) / (rel * peak + floor); <= 1 passes.  Arrays [..., nv]."""
    g = np.asarray(gpu, dtype=np.float64)
    o = np.asarray(ora, dtype=np.float64)
    peak = np.abs(o if peak_of is None else np.asarray(peak_of, dtype=np.float64)).max(axis=-1)
    err = (np.abs(g - o) - extra).max(axis=-1)
    return err / (rel * peak + floor)


def assert_spectra(gpu, ora, floor=1e-6, rel=1e-4, extra=0.0, peak_of=None, what="spectra"):
    assert np.all(np.isfinite(np.asarray(gpu))), "%s: non-finite values in the CUDA result" % what
    ex = spectrum_excess(gpu, ora, floor, rel, extra, peak_of)
    worst = float(ex.max())
    assert worst <= 1.0, "%s: worst pixel is at %.3g x the tolerance (1e-4 peak + floor)" % (what, worst)
    return worst


def selthin_source_allowance(cfg, fields):
    """Float32 rounding allowance [npix, nv] (Kelvin) of the selectively thin mode (derived for
    the smooth integrator, the formal step D' = E_d D + (E - A C') w(tau_d) is unsaturated in the same way).
    The step  D_n = [2 (E_n - A_n C_n) + 4 D_n-1 - D_n-2] / (3 + 2 tau_d)  has no line opacity
    in the denominator (Eq. 4.8.13 - 4.8.15: the line does not absorb itself), so the products E_n = e p and A_n C_n
    enter at full size whatever the optical depth, each formed by up to four float32 roundings (2^-22 relative), and the
    root 1 of the BDF2 recurrence keeps every one of them: |error| <= 2^-22 sum_n (E_n + A_n C_n) beside the usual
    1e-4 peak + 1e-6 K.  The sum is bounded with the oracle alone: C_n <= C_max = max(I_bg, max_n S_d,n) (a continuum never
    exceeds its largest source), and sum_n h p (j0 + kappa0 C_max) is the optically thin formal march (Eq. 4.7.6) of the
    column with j0 replaced by j0 + kappa0 C_max, minus its continuum.  A factor 2 covers the worst-case sign pattern."""
    from oracle import Oracle
    plane = cfg.nx * cfg.ny
    c_thin = cfg.with_(transfer_mode=2, integration=0, subsample=0, subtract_continuum=False, out_unit=0)
    o = Oracle(c_thin)
    coef = o.coefficients(fields["nH2"], fields["Tgas"], fields["Tdust"])
    I_bg = o.planck(cfg.nu0_Hz, cfg.T_cmb)
    C_max = np.maximum(I_bg, coef[4].reshape(cfg.nz, plane).max(axis=0))
    c2 = coef.copy()
    c2[0] = coef[0] + coef[1] * np.tile(C_max, cfg.nz)
    S, S_cont = o.march(c2, fields["vlos"])
    return 2.0 ** -21 * krj(cfg.nu0_Hz) * (S - S_cont[:, None])


# ---- allowances of the randomised campaign (tests/test_gpu_random.py) -------------------------------
def total_allowance(ora_total, ora_subtracted):
    """[..., 1] Kelvin.  The CUDA path marches D = I_T - I_C next to the continuum C, so a value that is printed as a
    total (or a line seen in absorption against a bright continuum) carries the float32 rounding of max(|total|, C):
    3e-7 of it (storage rounding of both, and of their sum)."""
    cont = np.abs(np.asarray(ora_total) - np.asarray(ora_subtracted)).max(axis=-1, keepdims=True)
    return 3e-7 * np.maximum(np.abs(ora_total).max(axis=-1, keepdims=True), cont)


def line_centre_allowance(cfg, ora_subtracted, saturated=None):
    """[..., 1] Kelvin.  The line-centre plane c_los = (v_los - v0) / dv + 1/2 is a float32 in channel units: its rounding
    (6e-8 nv channels) times the channel width in Doppler widths (<= dv / xi) moves the profile of a cell by that much of a
    Doppler width; negligible for resolved lines (dv < b), 1e-4 of the peak for 200 channels 6 Doppler widths wide.
    `saturated` (saturated_source of the same configuration, thick modes): a pixel that shows only the WINGS of opaque cells
    (a 1 K spectrum out of cells with S_L = 26 K at 2 - 3 Doppler widths, where d ln(profile) / dx = -2 x) answers to the
    shift with the source function of those cells, not with its own peak: the scale is then the larger of the two."""
    scale = np.abs(ora_subtracted).max(axis=-1, keepdims=True)
    if saturated is not None:
        scale = np.maximum(scale, np.asarray(saturated).reshape(ora_subtracted.shape).max(axis=-1, keepdims=True))
    return 1.2e-7 * cfg.nv * (cfg.dv_cms / cfg.microturb_cms) * scale


def saturated_source(cfg, fields):
    """[npix, nv] Kelvin: sum_n (S_L,n + C_max) (1 - e^-tau_n) e^-tau_beyond, the formal thick solution (oracle, hot-path
    mode) of the column with j0 replaced by j0 + kappa0 C_max, no dust and no background -- what every cell can put into a
    channel at most, the scale the allowances below are proportional to."""
    from oracle import Oracle
    plane = cfg.nx * cfg.ny
    c0 = cfg.with_(transfer_mode=0, integration=0, subsample=0, subtract_continuum=False, out_unit=0, T_cmb=0.0, coef_grid=0,
                   dust_per_channel=0)
    coef = Oracle(cfg.with_(coef_grid=0)).coefficients(fields["nH2"], fields["Tgas"], fields["Tdust"])
    I_bg = Oracle(cfg).planck(cfg.nu0_Hz, cfg.T_cmb) if cfg.T_cmb > 0 else 0.0
    C_max = np.maximum(I_bg, coef[4].reshape(cfg.nz, plane).max(axis=0))
    c2 = coef.copy()
    c2[0] = coef[0] + np.abs(coef[1]) * np.tile(C_max, cfg.nz)
    c2[1] = np.abs(coef[1])
    c2[3] = 0.0
    c2[4] = 0.0
    I, _ = Oracle(c0).march(c2, fields["vlos"])
    return krj(cfg.nu0_Hz) * I


def cancellation_allowance(cfg, fields, delta=2.0e-6, saturated=None):
    """[npix, nv] Kelvin.  K1's level fractions are within 1.2e-6 relative of the oracle's (north_star asks 1e-5), so the
    emission and the absorption of every cell carry ~2e-6 relative each.  Where the line source function S_L is close to
    the continuum the line is seen against (excitation temperature ~ background temperature), D = sum_n (S_L,n - C)
    (1 - e^-tau_n) e^-tau_beyond is a small difference of terms that do not share that error: the bound is delta times the
    same sum with S_L,n + C_max (saturated_source)."""
    return delta * (saturated_source(cfg, fields) if saturated is None else saturated)
