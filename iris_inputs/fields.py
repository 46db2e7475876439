"""Seeded synthetic CMZ-shaped cell fields and the five BASELINE.json workloads.

These stand in for the paper's AREPO-derived physical tensors (Table 1),
which are not in the container.  Recipe: SURVEY.md section 8(d) / BASELINE.json "configs":

* G(x): white N(0,1) -> rfftn -> x |k|^(-11/6) (P(k) ~ k^(-11/3), k = 0 mode zeroed) -> irfftn ->
  rescaled to zero mean, unit variance.
* n_H2 = exp(mu_ln + sigma_ln G1), mu_ln = ln(mean) - sigma_ln^2 / 2   (lognormal with given mean).
* T_gas = T_dust ~ U[T_lo, T_hi) iid per cell.
* v_los = V_edge (x - x_c) / (L_x / 2) + sigma_t G2   (solid-body rotation seen along z + turbulence).
* optional uniform foreground / background layers of cells along z (config "medium").

All arrays are float32, C-contiguous, shape (nz, ny, nx) (x fastest; k = 0 is the far side), and are
consumed unchanged by both the oracle and the CUDA path.  Nothing here computes any part of the method.
"""
import math
import numpy as np
from scipy import fft as _fft

from .config import ObsConfig
from .molecule import rigid_rotor, line_frequency

PC_CM = 3.0856775814913673e18
KMS = 1.0e5


def gaussian_random_field(shape, seed, index=-11.0 / 3.0, stream=0):
    """Zero-mean unit-variance Gaussian random field with power spectrum P(k) ~ k^index."""
    nz, ny, nx = (int(s) for s in shape)
    rng = np.random.default_rng([int(seed), int(stream)])
    white = rng.standard_normal((nz, ny, nx), dtype=np.float32)
    fk = _fft.rfftn(white, workers=-1)
    del white
    kz = np.fft.fftfreq(nz).astype(np.float32)[:, None, None]
    ky = np.fft.fftfreq(ny).astype(np.float32)[None, :, None]
    kx = np.fft.rfftfreq(nx).astype(np.float32)[None, None, :]
    k2 = kz * kz + ky * ky + kx * kx
    k2[0, 0, 0] = 1.0
    amp = k2 ** np.float32(index / 4.0)        # |k|^(index/2)
    amp[0, 0, 0] = 0.0
    fk *= amp
    del amp, k2
    g = _fft.irfftn(fk, s=(nz, ny, nx), workers=-1).astype(np.float32, copy=False)
    del fk
    g -= g.mean(dtype=np.float64)
    rms = math.sqrt(float(np.mean(np.square(g, dtype=np.float64))))
    if rms > 0.0:                      # a single-cell grid has no fluctuating mode: the field is zero
        g /= np.float32(rms)
    else:
        g[...] = 0.0
    return np.ascontiguousarray(g)


# name -> recipe.  Index in BASELINE.json "configs": tiny 0, small 1, medium 2, large 3, batch 4.
WORKLOADS = {
    "tiny": dict(n=32, cell_pc=3.0, n_levels=5, nv=64, dv_kms=0.5, mean_n=1.0e3, sigma_ln=1.5,
                 T_lo=30.0, T_hi=120.0, v_edge_kms=100.0, sigma_t_kms=10.0, dust=False, layers=0,
                 beam_fwhm_px=0.0, noise_sigma=0.0, seed=0),
    "small": dict(n=128, cell_pc=1.0, n_levels=10, nv=256, dv_kms=0.5, mean_n=1.0e3, sigma_ln=1.5,
                  T_lo=30.0, T_hi=120.0, v_edge_kms=100.0, sigma_t_kms=10.0, dust=True, layers=0,
                  beam_fwhm_px=0.0, noise_sigma=0.0, seed=1),
    "medium": dict(n=256, cell_pc=1.0, n_levels=10, nv=512, dv_kms=0.25, mean_n=3.0e3, sigma_ln=2.0,
                   T_lo=30.0, T_hi=120.0, v_edge_kms=100.0, sigma_t_kms=10.0, dust=True, layers=16,
                   beam_fwhm_px=3.0, noise_sigma=0.25, seed=2),
    "large": dict(n=512, cell_pc=0.5, n_levels=10, nv=1024, dv_kms=0.25, mean_n=3.0e3, sigma_ln=2.0,
                  T_lo=30.0, T_hi=120.0, v_edge_kms=200.0, sigma_t_kms=20.0, dust=True, layers=0,
                  beam_fwhm_px=0.0, noise_sigma=0.0, seed=3),
    # one cube of the batch; cube i uses seed 1000 + i and draws its own v_edge / sigma_t
    "batch": dict(n=128, cell_pc=1.0, n_levels=10, nv=256, dv_kms=0.5, mean_n=1.0e3, sigma_ln=1.5,
                  T_lo=30.0, T_hi=150.0, v_edge_kms=None, sigma_t_kms=None, dust=True, layers=0,
                  beam_fwhm_px=3.0, noise_sigma=0.25, seed=1000, n_cubes=64),
}

LAYER_N, LAYER_T, LAYER_V = 1.0e2, 20.0, 0.0   # config "medium" foreground / background cells


def _recipe(name, overrides):
    r = dict(WORKLOADS[name])
    r.update(overrides)
    return r


def make_workload(name, **overrides):
    """ObsConfig + recipe for one of the BASELINE.json workloads (optionally resized, e.g. n=64)."""
    r = _recipe(name, overrides)
    n = int(r["n"])
    nx = int(r.get("nx", n)); ny = int(r.get("ny", n)); nz = int(r.get("nz", n)) + 2 * int(r["layers"])
    mol = rigid_rotor(r["n_levels"])
    up = min(2, int(r["n_levels"]) - 1)   # J = 2-1 (1-0 for a two-level table)
    lo = up - 1
    nu0 = line_frequency(mol["energy_K"], up, lo)
    nv = int(r["nv"]); dv = r["dv_kms"] * KMS
    kappa = 0.9 * (nu0 / 230.0e9) ** 1.8 / 100.0 if r["dust"] else 0.0   # per gram of gas
    cfg = ObsConfig(
        nx=nx, ny=ny, nz=nz, cell_cm=r["cell_pc"] * PC_CM,
        line_upper=up, line_lower=lo, nu0_Hz=nu0, abundance=2.0e-6,
        microturb_cms=1.0 * KMS, T_bar=2.725, T_cmb=2.725,
        dust_on=bool(r["dust"]), kappa_gas_cm2_g=kappa,
        nv=nv, v0_cms=(0.5 - nv / 2.0) * dv, dv_cms=dv,
        subtract_continuum=True, subtract_space=0, out_unit=1,
        beam_fwhm_px=float(r["beam_fwhm_px"]), noise_mu=0.0, noise_sigma=float(r["noise_sigma"]),
        noise_gamma_mode=0, seed=int(r["seed"]), name=name, **mol)
    return cfg, r


def make_fields(cfg, recipe, seed=None):
    """Seeded cell fields for a workload: dict(nH2, Tgas, Tdust, vlos), float32 (nz, ny, nx)."""
    r = recipe
    seed = int(r["seed"] if seed is None else seed)
    L = int(r["layers"])
    nzc = cfg.nz - 2 * L
    shape = (nzc, cfg.ny, cfg.nx)
    rng = np.random.default_rng([seed, 7])
    v_edge, sigma_t = r["v_edge_kms"], r["sigma_t_kms"]
    if v_edge is None:
        v_edge = float(rng.uniform(50.0, 150.0))
    if sigma_t is None:
        sigma_t = float(rng.uniform(5.0, 20.0))
    g1 = gaussian_random_field(shape, seed, stream=1)
    mu_ln = math.log(r["mean_n"]) - 0.5 * r["sigma_ln"] ** 2
    nH2 = np.exp(np.float32(mu_ln) + np.float32(r["sigma_ln"]) * g1).astype(np.float32)
    del g1
    T = rng.uniform(r["T_lo"], r["T_hi"], size=shape).astype(np.float32)
    g2 = gaussian_random_field(shape, seed, stream=2)
    xc = 0.5 * (cfg.nx - 1)
    ramp = ((np.arange(cfg.nx, dtype=np.float32) - np.float32(xc)) / np.float32(0.5 * cfg.nx))
    vlos = (np.float32(v_edge * KMS) * ramp[None, None, :] + np.float32(sigma_t * KMS) * g2).astype(np.float32)
    del g2
    if L > 0:
        def pad(a, val):
            slab = np.full((L, cfg.ny, cfg.nx), val, dtype=np.float32)
            return np.concatenate([slab, a, slab], axis=0)
        nH2, T, vlos = pad(nH2, LAYER_N), pad(T, LAYER_T), pad(vlos, LAYER_V)
    out = dict(nH2=np.ascontiguousarray(nH2), Tgas=np.ascontiguousarray(T),
               Tdust=np.ascontiguousarray(T.copy()), vlos=np.ascontiguousarray(vlos))
    out["meta"] = dict(seed=seed, v_edge_kms=v_edge, sigma_t_kms=sigma_t)
    return out


def lattice_to_columns(t_lbr):
    """A physical tensor on the paper's observer-centred spherical lattice, indexed (l, b, r) with r sampled at regular
    intervals outward from the observer, as the [nz][ny][nx] column layout of this path: z = r with
    k = 0 the FAR end of the ray, y = b, x = l.  A pure change of index order; cell_cm is the radial step."""
    t = np.asarray(t_lbr)
    return np.ascontiguousarray(np.transpose(t, (2, 1, 0))[::-1])


def weight_cube(cfg, seed=2000):
    """Seeded weight cube w ~ U[0,1), float32 (ny, nx, nv), for L = sum(w * cube) (config "batch")."""
    rng = np.random.default_rng([int(seed), 11])
    return rng.random((cfg.ny, cfg.nx, cfg.nv), dtype=np.float32)
