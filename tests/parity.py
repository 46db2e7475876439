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
