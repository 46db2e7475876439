"""Observation parameter record (pure data; no arithmetic of the method).

Field meanings follow the paper's parameter list (Table 3) and
SURVEY.md section 8(b).  Units are CGS.  Both the oracle wrapper and the CUDA binding marshal
this record into their own, separately declared, C structs.
"""
from dataclasses import dataclass, field, replace
import math
import numpy as np


@dataclass
class ObsConfig:
    # grid: rays march along z; memory index (k*ny + j)*nx + i, k = 0 is the FAR side
    nx: int
    ny: int
    nz: int
    cell_cm: float
    # molecule (stands in for a LAMDA file)
    energy_K: np.ndarray          # [n_levels] E_i / k
    weight: np.ndarray            # [n_levels] g_i
    einstein_A: np.ndarray        # [n_levels, n_levels] A[u, l] (1/s), 0 where u <= l
    coll_down_ref: np.ndarray     # [n_levels, n_levels] K_ul at coll_T_ref (cm^3/s), 0 where u <= l
    coll_T_ref: float
    coll_T_exp: float
    line_upper: int
    line_lower: int
    nu0_Hz: float
    mol_mass_g: float
    abundance: float              # tracer molecules per H2
    microturb_cms: float = 0.0    # xi; 0 = thermal only
    T_bar: float = 2.725          # level-balance background temperature
    T_cmb: float = 2.725          # transfer background temperature
    T_inf: float = math.inf       # cutoff above which the tracer is absent
    # dust; kappa per gram of GAS
    dust_on: bool = False
    kappa_gas_cm2_g: float = 0.0
    mass_per_H2_g: float = 2.8 * 1.6735575e-24
    # channel grid: centre of channel k is v0 + k*dv
    nv: int = 64
    v0_cms: float = 0.0
    dv_cms: float = 0.5e5
    # post-processing
    subtract_continuum: bool = True
    subtract_space: int = 0       # 0 = intensity / Rayleigh-Jeans, 1 = Planck brightness temperature
    out_unit: int = 1             # 0 = intensity (cgs), 1 = T_RJ (K), 2 = Planck T_B (K)
    beam_fwhm_px: float = 0.0     # 0 = no beam
    noise_mu: float = 0.0
    noise_sigma: float = 0.0      # 0 (with mu = 0) = no noise
    noise_gamma_mode: int = 0     # 0: gamma = 1; 1: one gamma ~ U[0,1) per cube (Eq. 4.12.1)
    seed: int = 0
    # transfer / integration modes (PAPER.md sections 4.4 - 4.8); all 0 = the hot path
    transfer_mode: int = 0        # 0 optically thick, 1 selectively thin, 2 optically thin
    integration: int = 0          # 0 formal, 1 smooth (TR + BDF2; Simpson in thin mode)
    subsample: int = 0            # thick mode: 0 = channel-integrated profile; odd f = fine grid + Simpson (Eq. 4.5.1)
    # tabulated collision rates of several partners; None = the power law coll_down_ref (T/T_ref)^p
    coll_T_grid: np.ndarray = None        # [nT] ascending temperatures (K)
    coll_table: np.ndarray = None         # [P, nT, n_levels, n_levels] K_ul of partner p at T_grid[t], 0 where u <= l
    coll_partner_frac: np.ndarray = None  # [P] number density of partner p per n_H2
    # grid precomputation + interpolation of the line coefficients; 0 = level balance solved per cell
    coef_grid: int = 0
    grid_n_density: int = 128     # nodes along n_H2 (paper: 128)
    grid_n_temp: int = 64         # nodes along T_gas (paper: 64)
    grid_nH2_lo: float = 1.0e-2
    grid_nH2_hi: float = 1.0e9
    grid_T_lo: float = 5.0
    grid_T_hi: float = 3000.0
    # 0: dust source, background and unit conversion at nu0; 1: at every channel's own frequency
    dust_per_channel: int = 0
    # free-form label, ignored by both implementations
    name: str = field(default="", compare=False)

    @property
    def n_levels(self) -> int:
        return int(len(self.energy_K))

    @property
    def n_cells(self) -> int:
        return self.nx * self.ny * self.nz

    def with_(self, **kw) -> "ObsConfig":
        return replace(self, **kw)
