"""Analytic rigid-rotor molecule table (an INPUT: stands in for the LAMDA 13CO file, which is
not in the container -- PAPER.md:471, SURVEY.md section 8(c) O2 / BASELINE.json config 1).

Levels J = 0..N-1:  E_J = h B J(J+1),  g_J = 2J+1,  nu_{J->J-1} = 2 B J,
A_{J->J-1} = 64 pi^4 nu^3 mu^2 J / (3 h c^3 (2J+1))   (only Delta J = 1 radiative),
collisional de-excitation K_ul(T) = k_ref (T/T_ref)^p for Delta J = 1, half that for Delta J = 2,
zero otherwise (upward rates come from detailed balance inside each implementation).
"""
import math
import numpy as np

# CODATA-2018 exact SI values in CGS; used only to build the input table
_H = 6.62607015e-27      # erg s
_K = 1.380649e-16        # erg / K
_C = 2.99792458e10       # cm / s
_AMU = 1.66053906660e-24  # g
_DEBYE = 1.0e-18         # esu cm


def rigid_rotor(n_levels, B_Hz=55.101e9, mu_debye=0.11, k_ref=1.0e-11, T_ref=100.0, T_exp=0.2,
                dj2_factor=0.5, mass_amu=29.0):
    """Return a dict with the molecule arrays of ObsConfig for a linear rigid rotor."""
    n = int(n_levels)
    J = np.arange(n, dtype=np.float64)
    energy_K = _H * B_Hz * J * (J + 1.0) / _K
    weight = 2.0 * J + 1.0
    A = np.zeros((n, n))
    Kd = np.zeros((n, n))
    mu = mu_debye * _DEBYE
    for u in range(1, n):
        nu = 2.0 * B_Hz * u
        A[u, u - 1] = 64.0 * math.pi ** 4 * nu ** 3 * mu ** 2 * u / (3.0 * _H * _C ** 3 * (2.0 * u + 1.0))
        Kd[u, u - 1] = k_ref
        if u >= 2:
            Kd[u, u - 2] = dj2_factor * k_ref
    return dict(energy_K=energy_K, weight=weight, einstein_A=A, coll_down_ref=Kd,
                coll_T_ref=float(T_ref), coll_T_exp=float(T_exp), mol_mass_g=mass_amu * _AMU)


def line_frequency(energy_K, upper, lower):
    """nu_ul = k (E_u - E_l) / h for a table given as E/k."""
    return _K * (float(energy_K[upper]) - float(energy_K[lower])) / _H
