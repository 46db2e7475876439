"""Pins for the float64 oracle (oracle/iris_oracle.cpp): closed forms, limits, invariants, brute force.

None of these compares the oracle with itself through the same formula, and none involves the CUDA
path.  Citations are PAPER.md line + equation; the pin list is SURVEY.md section 8(c).
"""
import json
import math
import os
from fractions import Fraction

import numpy as np
import pytest
from scipy import integrate, special

from iris_inputs import ObsConfig, make_fields, make_workload, rigid_rotor
from iris_inputs.fields import KMS, PC_CM
from oracle import Oracle

H, KB, CL = 6.62607015e-27, 1.380649e-16, 2.99792458e10


def base_cfg(n_levels=5, **kw):
    cfg, _ = make_workload("tiny", n_levels=n_levels)
    return cfg.with_(**kw) if kw else cfg


def boltzmann(cfg, T):
    x = cfg.weight * np.exp(-cfg.energy_K / T)
    return x / x.sum()


@pytest.fixture(scope="module")
def anchors(golden_dir):
    with open(os.path.join(golden_dir, "survey_anchors.json")) as f:
        return json.load(f)


# ------------------------------------------------------------------------------------------------
# input table (not the oracle, but everything downstream depends on it)
def test_rotor_table_matches_anchors(anchors):
    m = rigid_rotor(10)
    a = anchors["rotor"]
    nu = KB * np.diff(m["energy_K"]) / H
    assert np.allclose(nu[:4] / 1e9, a["nu_GHz"], rtol=1e-6, atol=0.0)
    assert np.allclose(m["energy_K"][1:5], a["E_over_k_K"], rtol=2e-6, atol=0.0)
    A = m["einstein_A"]
    for k, (u, l) in {"A_10": (1, 0), "A_21": (2, 1), "A_32": (3, 2), "A_43": (4, 3), "A_98": (9, 8)}.items():
        assert A[u, l] == pytest.approx(a[k], rel=2e-6, abs=0.0)
    assert np.count_nonzero(A) == 9 and np.all(np.triu(A) == 0)
    K = m["coll_down_ref"]
    assert K[3, 2] == 1e-11 and K[3, 1] == 0.5e-11 and K[3, 0] == 0.0 and np.all(np.triu(K) == 0)


# ------------------------------------------------------------------------------------------------
# Pins 1-4: level balance, Eq. 3.6.1-3.6.3 / 3.7.1-3.7.2
@pytest.mark.parametrize("n_levels", [2, 5, 10])
@pytest.mark.parametrize("nH2,T", [(1.0, 30.0), (1e3, 50.0), (3e5, 119.0), (1e8, 20.0)])
def test_pop_sum_and_stationarity(n_levels, nH2, T):
    o = Oracle(base_cfg(n_levels))
    x = o.levelpop_cell(nH2, T)
    assert abs(x.sum() - 1.0) < 1e-14
    assert np.all(x > 0)
    # stationarity via flux balance written from the RATES (not from the oracle's matrix):
    # inflow to level i equals outflow from level i, Eq. 3.6.1
    R = o.rates(nH2, T)
    inflow = x @ R - x * np.diag(R)
    outflow = x * (R.sum(axis=1) - np.diag(R))
    assert np.allclose(inflow[1:], outflow[1:], rtol=1e-10, atol=0)


def test_pop_exact_rational_solve():
    """Component-wise accuracy of the float64 GE solve over 30 decades: exact rational arithmetic on
    the same (double-valued) rates, by the subtraction-free state-elimination recursion."""
    for nH2, T, Tbar in [(1.0, 30.0, 2.725), (1.0, 30.0, 0.0), (1e3, 50.0, 2.725), (2e6, 117.0, 2.725), (0.05, 25.0, 0.0)]:
        o = Oracle(base_cfg(10, T_bar=Tbar))
        x = o.levelpop_cell(nH2, T)
        R = [[Fraction(v) for v in row] for row in o.rates(nH2, T)]
        N = 10
        for n in range(N - 1, 0, -1):       # eliminate state n (censored Markov chain)
            s = sum(R[n][j] for j in range(n))
            for i in range(n):
                R[i][n] = R[i][n] / s
            for i in range(n):
                for j in range(n):
                    if i != j:
                        R[i][j] += R[i][n] * R[n][j]
        y = [Fraction(1)] + [Fraction(0)] * (N - 1)
        for j in range(1, N):
            y[j] = sum(y[i] * R[i][j] for i in range(j))
        tot = sum(y)
        exact = np.array([float(v / tot) for v in y])
        assert np.max(np.abs(x / exact - 1.0)) < 1e-11, (nH2, T, Tbar)


def test_pop_lte_limit_is_boltzmann():
    """n_H2 -> large: collisions dominate and detailed balance (Eq. 3.7.2) forces Boltzmann at T_gas."""
    cfg = base_cfg(10)
    o = Oracle(cfg)
    for T in (20.0, 50.0, 120.0):
        x = o.levelpop_cell(1e14, T)
        assert np.allclose(x, boltzmann(cfg, T), rtol=1e-6, atol=0.0)


def test_pop_tbar_equals_tgas_is_boltzmann_at_any_density():
    """Radiation field at T_bar = T_gas: every process obeys detailed balance at one temperature
    (Eq. 3.6.2 + 3.7.1 + 3.7.2), so the solution is Boltzmann whatever the density."""
    for T in (15.0, 40.0):
        cfg = base_cfg(10, T_bar=T)
        o = Oracle(cfg)
        for n in (1e-2, 1e2, 1e5):
            assert np.allclose(o.levelpop_cell(n, T), boltzmann(cfg, T), rtol=1e-9, atol=0.0)


def test_pop_radiative_limit():
    """n_H2 -> 0: Boltzmann at T_bar (Einstein relations, Eq. 3.7.1); all in the ground state if T_bar = 0."""
    cfg = base_cfg(5, T_bar=8.0)
    x = Oracle(cfg).levelpop_cell(1e-12, 60.0)
    assert np.allclose(x, boltzmann(cfg, 8.0), rtol=1e-6, atol=0.0)
    x0 = Oracle(base_cfg(5, T_bar=0.0)).levelpop_cell(1e-14, 60.0)
    assert x0[0] == pytest.approx(1.0, abs=1e-9) and np.all(x0[1:] < 1e-9)


def test_pop_two_level_closed_form(anchors):
    """x_1/x_0 = (C_01 + B_01 J) / (A_10 + B_10 J + C_10) with the rates typed out here."""
    m = rigid_rotor(2)
    for Tbar in (0.0, 2.725):
        cfg = base_cfg(2, T_bar=Tbar)
        n, T = 1e3, 50.0
        nu = KB * (m["energy_K"][1] - m["energy_K"][0]) / H
        A10 = m["einstein_A"][1, 0]
        ngam = 0.0 if Tbar == 0 else 1.0 / math.expm1(H * nu / (KB * Tbar))
        K10 = 1e-11 * (T / 100.0) ** 0.2
        C10 = K10 * n
        C01 = K10 * 3.0 * math.exp(-m["energy_K"][1] / T) * n
        ratio = (C01 + 3.0 * A10 * ngam) / (A10 * (1.0 + ngam) + C10)
        x = Oracle(cfg).levelpop_cell(n, T)
        assert x[1] / x[0] == pytest.approx(ratio, rel=1e-12, abs=0.0)
        if Tbar == 0.0:
            assert x[1] == pytest.approx(anchors["two_level_n1e3_T50_Tbar0_x1"], rel=2e-6, abs=0.0)


def test_pop_anchors(anchors):
    x0 = Oracle(base_cfg(5, T_bar=0.0)).levelpop_cell(1e3, 50.0)
    x1 = Oracle(base_cfg(5, T_bar=2.725)).levelpop_cell(1e3, 50.0)
    assert np.allclose(x0, anchors["pop5_n1e3_T50_Tbar0"], rtol=6e-6, atol=0.0)      # anchors are printed to 6 digits
    assert np.allclose(x1, anchors["pop5_n1e3_T50_Tbar2p725"], rtol=6e-6, atol=0.0)
    assert Oracle(base_cfg(10, T_bar=2.725)).levelpop_cell(1.0, 30.0)[9] == pytest.approx(
        anchors["pop10_n1_T30_x9_Tbar2p725"], rel=5e-3, abs=0.0)
    assert Oracle(base_cfg(10, T_bar=0.0)).levelpop_cell(1.0, 30.0)[9] == pytest.approx(
        anchors["pop10_n1_T30_x9_Tbar0"], rel=5e-3, abs=0.0)


# ------------------------------------------------------------------------------------------------
# Pin 10: Planck / Rayleigh-Jeans, Eq. 4.9.1-4.9.2
def test_planck_and_rj(anchors):
    cfg = base_cfg()
    o = Oracle(cfg)
    nu = cfg.nu0_Hz
    assert H * nu / KB == pytest.approx(anchors["h_nu21_over_k_K"], rel=1e-6, abs=0.0)
    B = o.planck(nu, 2.725)
    assert B == pytest.approx(2 * H * nu ** 3 / CL ** 2 / (math.exp(H * nu / (KB * 2.725)) - 1), rel=1e-13, abs=0.0)
    assert B == pytest.approx(anchors["B_nu_2p725_cgs"], rel=2e-6, abs=0.0)
    assert o.rayleigh_jeans_T(nu, B) == pytest.approx(anchors["T_RJ_of_B_2p725"], rel=2e-6, abs=0.0)
    for T in (0.5, 2.725, 40.0, 3000.0):
        assert o.planck_TB(nu, o.planck(nu, T)) == pytest.approx(T, rel=1e-12, abs=0.0)
    # Rayleigh-Jeans limit: h nu << k T  =>  T_RJ(B_nu(T)) -> T - h nu / 2k
    T = 1e5
    assert o.rayleigh_jeans_T(nu, o.planck(nu, T)) == pytest.approx(T - H * nu / (2 * KB), rel=1e-8, abs=0.0)
    assert o.planck(nu, 0.0) == 0.0 and o.planck_TB(nu, 0.0) == 0.0
    assert o.planck_TB(nu, -B) == -o.planck_TB(nu, B)


# ------------------------------------------------------------------------------------------------
# Pin 5: integrated profile, Eq. 4.6.3 = channel average (Eq. 4.4.1) of Eq. 3.3.3
def test_profile_equals_quadrature_of_point_profile():
    cfg = base_cfg()
    o = Oracle(cfg)
    nu0, dv = cfg.nu0_Hz, cfg.dv_cms
    dnuW = nu0 * dv / CL
    for vlos, b in [(0.0, 1.0e5), (3.3e5, 0.4e5), (-7.77e5, 2.5e5), (0.1e5, 0.05e5)]:
        dnuD = nu0 * b / CL
        for k in range(0, cfg.nv, 5):
            vk = cfg.v0_cms + k * dv
            # frequency offsets (from the Doppler-shifted line centre) of the channel edges
            lo = nu0 * (vk - dv / 2 - vlos) / CL
            hi = nu0 * (vk + dv / 2 - vlos) / CL
            f = lambda x: math.exp(-(x / dnuD) ** 2) / (dnuD * math.sqrt(math.pi))   # Eq. 3.3.3
            pts = [p for p in (0.0,) if lo < p < hi]
            q, _ = integrate.quad(f, lo, hi, points=pts or None, epsabs=0, epsrel=1e-13, limit=200)
            # erf differences carry the absolute rounding of erf near 1 (a few 1e-16 of probability mass)
            assert o.phibar(k, vlos, b) * dnuW == pytest.approx(q, rel=1e-10, abs=5e-16)


def test_profile_normalisation_and_sign_convention():
    cfg = base_cfg()
    o = Oracle(cfg)
    dnuW = cfg.nu0_Hz * cfg.dv_cms / CL
    pb = np.array([o.phibar(k, 2.2e5, 1.3e5) for k in range(cfg.nv)])
    assert pb.sum() * dnuW == pytest.approx(1.0, abs=1e-12)          # probability mass over a wide band
    vk = cfg.v0_cms + np.arange(cfg.nv) * cfg.dv_cms
    assert abs(vk[np.argmax(pb)] - 2.2e5) <= cfg.dv_cms / 2            # receding gas -> positive channel velocity
    assert (pb * vk).sum() / pb.sum() == pytest.approx(2.2e5, rel=1e-9, abs=0.0)
    # point profile: value at line centre is 1 / (Delta nu_D sqrt(pi)), Eq. 3.3.3-3.3.4
    assert o.phi_point(2.2e5, 2.2e5, 1.3e5) == pytest.approx(1.0 / (cfg.nu0_Hz * 1.3e5 / CL * math.sqrt(math.pi)), rel=1e-14, abs=0.0)
    # channel grid (reading S12): band is symmetric about 0 with edges +- nv dv / 2
    assert vk[0] - cfg.dv_cms / 2 == pytest.approx(-cfg.nv * cfg.dv_cms / 2)
    assert vk[-1] + cfg.dv_cms / 2 == pytest.approx(cfg.nv * cfg.dv_cms / 2)


# ------------------------------------------------------------------------------------------------
# helpers for slab / small-grid tests
def uniform_fields(cfg, n=1e3, T=50.0, v=0.0, Td=None):
    shape = (cfg.nz, cfg.ny, cfg.nx)
    return dict(nH2=np.full(shape, n, np.float32), Tgas=np.full(shape, T, np.float32),
                Tdust=np.full(shape, T if Td is None else Td, np.float32), vlos=np.full(shape, v, np.float32))


def small_cfg(nx=2, ny=2, nz=32, **kw):
    return base_cfg(**kw).with_(nx=nx, ny=ny, nz=nz)


# Pin 6: uniform slab, closed form of Eq. 3.1.1 with constant coefficients
def test_uniform_slab_closed_form_and_anchors(anchors):
    cfg = small_cfg()
    o = Oracle(cfg)
    f = uniform_fields(cfg)
    coef = o.coefficients(f["nH2"], f["Tgas"], f["Tdust"])
    s = anchors["slab"]
    assert coef[0, 0] == pytest.approx(s["j0"], rel=3e-6, abs=0.0)
    assert coef[1, 0] == pytest.approx(s["kappa0"], rel=3e-6, abs=0.0)
    assert coef[2, 0] / KMS == pytest.approx(s["b_kms"], rel=2e-6, abs=0.0)
    It, Ic = o.march(coef, f["vlos"])
    Ibg = o.planck(cfg.nu0_Hz, cfg.T_cmb)
    L = cfg.nz * cfg.cell_cm
    dnuW = cfg.nu0_Hz * cfg.dv_cms / CL
    vk = cfg.v0_cms + np.arange(cfg.nv) * cfg.dv_cms
    b = coef[2, 0]
    pb = (special.erf((vk + cfg.dv_cms / 2) / b) - special.erf((vk - cfg.dv_cms / 2) / b)) / (2 * dnuW)
    tau = coef[1, 0] * pb * L
    S = coef[0, 0] / coef[1, 0]
    expect = S * (1 - np.exp(-tau)) + Ibg * np.exp(-tau)
    assert np.allclose(It[0], expect, rtol=1e-12, atol=0.0)
    assert Ic[0] == pytest.approx(Ibg, rel=1e-15, abs=0.0)
    # anchors: line optical depths and subtracted T_RJ at v = +0.25 ... +2.75 km/s
    idx = [int(round((v * KMS - cfg.v0_cms) / cfg.dv_cms)) for v in s["v_kms"]]
    assert np.allclose(tau[idx], s["tau_line"], rtol=2e-5, atol=0.0)        # anchors are printed to 5-6 digits
    T = o.convert(It, Ic)[0]
    assert T[idx[0]] == pytest.approx(s["T_RJ_first"], rel=3e-6, abs=0.0)
    assert np.allclose(T[idx[3:]], s["T_RJ_last3"], rtol=5e-6, atol=0.0)
    # S = j0 / kappa0 = B_nu(T_ex) with T_ex defined by x_u / x_l = (g_u / g_l) exp(-h nu / k T_ex)
    # (Eq. 3.3.1-3.3.2 with the Einstein relations Eq. 3.7.1).  The surveyor's "T_ex_21" anchor (4.5444 K)
    # contradicts the surveyor's own saturated T_RJ anchor checked above and is not used.
    x = o.levelpop_cell(1e3, 50.0)
    Tex = -(H * cfg.nu0_Hz / KB) / math.log(x[2] / x[1] * 3.0 / 5.0)
    assert o.planck_TB(cfg.nu0_Hz, S) == pytest.approx(Tex, rel=1e-12, abs=0.0)
    assert T[idx[0]] == pytest.approx((H * cfg.nu0_Hz / KB) * (1 / math.expm1(H * cfg.nu0_Hz / (KB * Tex))
                                      - 1 / math.expm1(H * cfg.nu0_Hz / (KB * cfg.T_cmb))), rel=1e-9, abs=0.0)


def test_substep_invariance():
    """Semigroup property of Eq. 4.8.5: splitting every cell into m sub-cells of h/m changes nothing."""
    cfg, r = make_workload("tiny", n=4, nv=32)
    cfg = cfg.with_(dust_on=True, kappa_gas_cm2_g=5.0)
    f = make_fields(cfg, r)
    f["Tdust"] = (f["Tdust"] * 0.5).astype(np.float32)
    o = Oracle(cfg)
    I1, C1 = o.march(o.coefficients(f["nH2"], f["Tgas"], f["Tdust"]), f["vlos"])
    m = 5
    cfg_m = cfg.with_(nz=cfg.nz * m, cell_cm=cfg.cell_cm / m)
    fm = {k: np.repeat(f[k], m, axis=0) for k in ("nH2", "Tgas", "Tdust", "vlos")}
    om = Oracle(cfg_m)
    Im, Cm = om.march(om.coefficients(fm["nH2"], fm["Tgas"], fm["Tdust"]), fm["vlos"])
    assert np.allclose(Im, I1, rtol=1e-12, atol=0.0) and np.allclose(Cm, C1, rtol=1e-12, atol=0.0)
    assert np.max(np.abs(I1 / C1[:, None] - 1)) > 0.1     # the test has a line in it


# Pin 7: optically thin limit, Eq. 4.7.3
def test_optically_thin_limit():
    cfg0, r = make_workload("tiny", n=4, nv=64)
    f = make_fields(cfg0, r)
    f["vlos"] = (0.1 * f["vlos"]).astype(np.float32)          # keep the lines inside the band
    X = 1e-12                      # tau ~ 1e-6 per cell: first order in tau is exact to ~1e-6
    cfg = cfg0.with_(abundance=X)
    o = Oracle(cfg)
    coef = o.coefficients(f["nH2"], f["Tgas"], f["Tdust"])
    It, Ic = o.march(coef, f["vlos"])
    Ibg = o.planck(cfg.nu0_Hz, cfg.T_cmb)
    plane = cfg.nx * cfg.ny
    j0 = coef[0].reshape(cfg.nz, plane)
    k0 = coef[1].reshape(cfg.nz, plane)
    # velocity-integrated: sum_v (I - I_bg) dnu_W = sum_cells (j0 - kappa0 I_bg) h  as tau -> 0
    dnuW = cfg.nu0_Hz * cfg.dv_cms / CL
    lhs = (It - Ibg).sum(axis=1) * dnuW
    rhs = ((j0 - k0 * Ibg) * cfg.cell_cm).sum(axis=0)
    assert np.allclose(lhs, rhs, rtol=2e-5, atol=0.0)
    # per channel: I - I_bg = sum_k (j0 - kappa0 I_bg) phibar_k h, with phibar from scipy's erf
    vk = cfg.v0_cms + np.arange(cfg.nv) * cfg.dv_cms
    vl = f["vlos"].reshape(cfg.nz, plane).astype(np.float64)
    b = coef[2].reshape(cfg.nz, plane)
    p = 5
    pb = (special.erf((vk[None] + cfg.dv_cms / 2 - vl[:, p, None]) / b[:, p, None])
          - special.erf((vk[None] - cfg.dv_cms / 2 - vl[:, p, None]) / b[:, p, None])) / (2 * dnuW)
    expect = (((j0[:, p] - k0[:, p] * Ibg) * cfg.cell_cm)[:, None] * pb).sum(axis=0)
    assert np.allclose(It[p] - Ibg, expect, rtol=2e-5, atol=1e-8 * np.abs(expect).max())
    # linear in abundance (Eq. 4.2.1)
    o2 = Oracle(cfg0.with_(abundance=2 * X))
    It2, _ = o2.march(o2.coefficients(f["nH2"], f["Tgas"], f["Tdust"]), f["vlos"])
    assert np.allclose(It2 - Ibg, 2 * (It - Ibg), rtol=2e-5, atol=1e-8 * np.abs(It - Ibg).max())


# Pin 8: brute-force monochromatic integration on 4^3 grids (Eq. 3.1.2 + 3.3.3, averaged by Eq. 4.4.2)
def test_brute_force_fine_frequency_integration():
    cfg0, r = make_workload("tiny", n=4, nv=48)
    f = make_fields(cfg0, r)
    f["vlos"] = (0.05 * f["vlos"]).astype(np.float32)
    gaps = []
    for X in (2e-10, 2e-8, 2e-6):
        cfg = cfg0.with_(abundance=X, dust_on=True, kappa_gas_cm2_g=0.5)
        o = Oracle(cfg)
        coef = o.coefficients(f["nH2"], f["Tgas"], f["Tdust"])
        It, Ic = o.march(coef, f["vlos"])
        gap = 0.0
        for pix in (0, 7, 13):
            br = o.brute_column(coef, f["vlos"], pix, 400)
            gap = max(gap, np.max(np.abs(br - It[pix])) / np.max(np.abs(It[pix] - Ic[pix])))
        gaps.append(gap)
    # converges to the method as tau -> 0; the remaining gap at large tau is the model difference of
    # reading R1 (channel-mean profile inside the exponential), documented in DESIGN.md
    assert gaps[0] < 1e-5 and gaps[1] < 1e-3 and gaps[0] < gaps[1] < gaps[2] < 0.2


# Pin 9: dust only
def test_dust_only():
    cfg = small_cfg(nz=16, dust_on=True, kappa_gas_cm2_g=0.5, abundance=0.0)
    o = Oracle(cfg)
    f = uniform_fields(cfg, n=3e3, T=50.0, Td=35.0)
    cube = o.observe(f)
    assert np.all(cube == 0.0)
    coef = o.coefficients(f["nH2"], f["Tgas"], f["Tdust"])
    It, Ic = o.march(coef, f["vlos"])
    alpha = 0.5 * cfg.mass_per_H2_g * 3e3
    assert coef[3, 0] == pytest.approx(alpha, rel=1e-14, abs=0.0)
    tau = alpha * cfg.nz * cfg.cell_cm
    assert 0.05 < tau < 5
    Bd, Ibg = o.planck(cfg.nu0_Hz, 35.0), o.planck(cfg.nu0_Hz, cfg.T_cmb)
    assert Ic[0] == pytest.approx(Bd * (1 - math.exp(-tau)) + Ibg * math.exp(-tau), rel=1e-13, abs=0.0)
    # dust at the background temperature leaves the background untouched, whatever tau
    f2 = uniform_fields(cfg, n=3e3, T=50.0, Td=cfg.T_cmb)
    _, Ic2 = o.march(o.coefficients(f2["nH2"], f2["Tgas"], f2["Tdust"]), f2["vlos"])
    # (the field is float32: the dust sees T = float32(T_cmb), 3.5e-8 away, and d ln B / d ln T = 4 here)
    Bd2 = o.planck(cfg.nu0_Hz, float(np.float32(cfg.T_cmb)))
    assert Ic2[0] == pytest.approx(Bd2 * (1 - math.exp(-tau)) + Ibg * math.exp(-tau), rel=1e-13, abs=0.0)
    assert Ic2[0] == pytest.approx(Ibg, rel=5e-7, abs=0.0)
    # dust_on = 0 switches it off
    o3 = Oracle(cfg.with_(dust_on=False))
    assert np.all(o3.coefficients(f["nH2"], f["Tgas"], f["Tdust"])[3:] == 0.0)


def test_kappa_dust_anchor(anchors):
    cfg, _ = make_workload("small")
    assert cfg.kappa_gas_cm2_g * 100.0 == pytest.approx(anchors["kappa_dust_220p404GHz_per_g_dust"], rel=2e-6, abs=0.0)


def test_T_inf_cutoff_and_no_subtraction_modes():
    cfg = small_cfg(nz=8, T_inf=60.0)
    o = Oracle(cfg)
    f = uniform_fields(cfg, T=50.0)
    f["Tgas"][3:5] = 80.0
    coef = o.coefficients(f["nH2"], f["Tgas"], f["Tdust"]).reshape(5, cfg.nz, -1)
    assert np.all(coef[:2, 3:5] == 0.0) and np.all(coef[:2, :3] > 0.0)
    # conversion modes
    It, Ic = o.march(coef.reshape(5, -1), f["vlos"])
    nu = cfg.nu0_Hz
    K = CL ** 2 / (2 * KB * nu ** 2)
    assert np.allclose(Oracle(cfg.with_(out_unit=0)).convert(It, Ic), It - Ic[:, None], rtol=1e-15, atol=0.0)
    assert np.allclose(Oracle(cfg.with_(out_unit=1)).convert(It, Ic), K * (It - Ic[:, None]), rtol=1e-14, atol=0.0)
    assert np.allclose(Oracle(cfg.with_(out_unit=1, subtract_continuum=False)).convert(It, Ic), K * It, rtol=1e-14, atol=0.0)
    tb = lambda I: (H * nu / KB) / np.log1p(2 * H * nu ** 3 / (CL ** 2 * I))
    assert np.allclose(Oracle(cfg.with_(out_unit=2, subtract_space=1)).convert(It, Ic), tb(It) - tb(Ic)[:, None], rtol=1e-12, atol=0.0)


# ------------------------------------------------------------------------------------------------
# Pin 11: beam (reading S8)
def test_beam():
    o = Oracle(base_cfg())
    g = o.beam_weights(2.0)
    R = (len(g) - 1) // 2
    assert R == math.ceil(4 * 2.0 / (2 * math.sqrt(2 * math.log(2))))
    assert g.sum() == pytest.approx(1.0, abs=1e-15) and np.allclose(g, g[::-1])
    assert g[R + 1] / g[R] == pytest.approx(0.5, rel=1e-14, abs=0.0)          # half maximum at FWHM / 2 = 1 px
    g3 = o.beam_weights(3.0)
    assert len(g3) == 2 * 6 + 1                                       # sigma = 1.274 px, R = ceil(5.1) = 6
    ny, nx, nv = 21, 19, 3
    rng = np.random.default_rng(1)
    # constant image unchanged in the interior, attenuated at the zero-padded edge
    c = o.beam(np.ones((ny, nx, nv)), 3.0)
    assert np.allclose(c[6:-6, 6:-6], 1.0, atol=1e-14) and c[0, 0, 0] < 0.5
    # delta -> outer product of the 1-D weights
    d = np.zeros((ny, nx, nv)); d[10, 9, 1] = 1.0
    out = o.beam(d, 3.0)
    assert np.allclose(out[4:17, 3:16, 1], np.outer(g3, g3), atol=1e-16)
    assert np.all(out[:, :, 0] == 0) and np.all(out[:, :, 2] == 0)      # channels do not mix
    # direct 2-D sum equals two separable 1-D passes (scipy, independent code)
    from scipy.ndimage import convolve1d
    img = rng.standard_normal((ny, nx, nv))
    sep = convolve1d(convolve1d(img, g3, axis=0, mode="constant"), g3, axis=1, mode="constant")
    assert np.allclose(o.beam(img, 3.0), sep, atol=1e-13)


# ------------------------------------------------------------------------------------------------
# Pin 12: noise (Eq. 4.12.1; reading S10)
def test_philox_known_answers():
    """Philox4x32-10 known-answer vectors published with the Random123 library (Salmon et al. 2011)."""
    o = Oracle(base_cfg())
    assert o.philox(0, 0, 0) == [0x6627e8d5, 0xe169c58d, 0xbc57ac4c, 0x9b00dbd8]
    assert o.philox(0xffffffffffffffff, 0xffffffffffffffff, 0xffffffffffffffff) == [0x408f276d, 0x41c83b0e, 0xa20bc7c6, 0x6d5451fd]
    assert o.philox(0x299f31d0a4093822, 0x85a308d3243f6a88, 0x0370734413198a2e) == [0xd16cfe09, 0x94fdcceb, 0x5001e420, 0x24126ea1]


def test_noise_statistics_and_definition():
    cfg = base_cfg(noise_sigma=0.25, noise_mu=0.1, seed=12345)
    o = Oracle(cfg)
    n = 200_000
    z = (o.noise(np.zeros(n)) - 0.1) / 0.25
    assert abs(z.mean()) < 4 / math.sqrt(n)
    assert abs(z.std() - 1.0) < 4 / math.sqrt(2 * n)
    assert abs(np.mean(z[1:] * z[:-1])) < 4 / math.sqrt(n)            # lag-1 correlation
    assert abs(np.mean(z ** 3)) < 0.03 and abs(np.mean(z ** 4) - 3.0) < 0.08
    for lag in (2, 3, 4):                                              # the four voxels of one Philox call, and beyond
        assert abs(np.mean(z[lag:] * z[:-lag])) < 4 / math.sqrt(n)
    z2sq = z ** 2 - 1.0                                                # cos / sin partners share a radius only
    assert abs(np.mean(z2sq[0::2] * z2sq[1::2])) < 6 / math.sqrt(n / 2)
    # voxel i depends only on (seed, i): one Philox call per four voxels, Box-Muller cos / sin per word pair
    for i in (776, 777, 778, 779):
        r = o.philox(12345, i // 4)
        p = (i // 2) % 2
        u1, u2 = ((r[2 * p] >> 8) + 0.5) / 2 ** 24, ((r[2 * p + 1] >> 8) + 0.5) / 2 ** 24
        trig = math.sin if i % 2 else math.cos
        assert z[i] == pytest.approx(math.sqrt(-2 * math.log(u1)) * trig(2 * math.pi * u2), rel=1e-9, abs=1e-12)
        assert o.normal(12345, i) == pytest.approx(z[i], rel=1e-9, abs=1e-12)
    # different seed -> different field; gamma mode 1 scales the whole cube by one U[0,1) draw
    z2 = Oracle(cfg.with_(seed=12346)).noise(np.zeros(1000))
    assert abs(np.corrcoef(z2, o.noise(np.zeros(1000)))[0, 1]) < 0.15
    og = Oracle(cfg.with_(noise_gamma_mode=1))
    gam = og.noise_gamma()
    assert 0.0 <= gam < 1.0
    assert np.allclose(og.noise(np.zeros(100)), gam * o.noise(np.zeros(100)), rtol=1e-13, atol=0.0)


# ------------------------------------------------------------------------------------------------
# whole path = the stages chained (stage list PAPER.md:467)
def test_observe_equals_chained_stages():
    cfg, r = make_workload("tiny", n=8, nv=32)
    cfg = cfg.with_(dust_on=True, kappa_gas_cm2_g=0.3, beam_fwhm_px=3.0, noise_sigma=0.25, seed=5)
    f = make_fields(cfg, r)
    o = Oracle(cfg)
    pop = o.levelpop(f["nH2"], f["Tgas"])
    coef = o.coefficients(f["nH2"], f["Tgas"], f["Tdust"], pop)
    It, Ic = o.march(coef, f["vlos"])
    raw = o.convert(It, Ic).reshape(cfg.ny, cfg.nx, cfg.nv)
    assert np.array_equal(o.observe(f, beam=False, noise=False), raw)
    assert np.allclose(o.observe(f, beam=True, noise=False), o.beam(raw), rtol=0, atol=0)
    assert np.array_equal(o.observe(f), o.noise(o.beam(raw)))
    # a subset of columns equals the same columns of the full march
    pix = np.array([3, 17, 40], dtype=np.int64)
    Is, Cs = o.march(coef, f["vlos"], pix)
    assert np.array_equal(Is, It[pix]) and np.array_equal(Cs, Ic[pix])


# ------------------------------------------------------------------------------------------------
# Pin 13: gradient
def test_adjoint_matches_finite_differences_and_is_linear_in_w():
    cfg, r = make_workload("tiny", n=6, nv=32)
    cfg = cfg.with_(dust_on=True, kappa_gas_cm2_g=0.05, beam_fwhm_px=3.0)
    f = make_fields(cfg, r)
    f["vlos"] = (0.2 * f["vlos"]).astype(np.float32)
    o = Oracle(cfg)
    rng = np.random.default_rng(3)
    w = rng.random((cfg.ny, cfg.nx, cfg.nv))
    what = o.beam(w)                                  # beam adjoint = same symmetric zero-padded conv
    g = o.grad_adjoint(f, what)
    cells = rng.choice(cfg.n_cells, size=40, replace=False)
    gfd = o.grad_fd(f, what, cells, eps=1e-5)
    assert np.allclose(g.ravel()[cells], gfd, rtol=2e-6, atol=1e-9 * np.abs(gfd).max())
    # whole-pipeline directional derivative: L(n + t d) through observe() (beam applied to the cube)
    d = rng.standard_normal(f["nH2"].shape) * f["nH2"] * 1e-3
    def L(nH2):
        ff = dict(f); ff["nH2"] = nH2
        return float((w * o.observe(ff, beam=True, noise=False)).sum())
    # fields are float32 inputs: build +- perturbations that are exactly representable
    np_ = (f["nH2"].astype(np.float64) + d).astype(np.float32)
    nm_ = (f["nH2"].astype(np.float64) - d).astype(np.float32)
    dd = np_.astype(np.float64) - nm_.astype(np.float64)
    assert (L(np_) - L(nm_)) == pytest.approx(float((g * dd).sum()), rel=1e-4, abs=0.0)
    # linear in w
    w2 = rng.random(w.shape)
    g2 = o.grad_adjoint(f, o.beam(w2))
    g12 = o.grad_adjoint(f, o.beam(w + 3 * w2))
    assert np.allclose(g12, g + 3 * g2, rtol=1e-10, atol=1e-12 * np.abs(g12).max())


def test_abundance_gradient_pins():
    """Abundance-only gradient: dL / d ln X_c for a per-cell factor on the tracer abundance."""
    cfg, r = make_workload("tiny", n=6, nv=32)
    cfg = cfg.with_(dust_on=True, kappa_gas_cm2_g=0.05)
    f = make_fields(cfg, r)
    f["vlos"] = (0.2 * f["vlos"]).astype(np.float32)
    o = Oracle(cfg)
    rng = np.random.default_rng(4)
    w = rng.random((cfg.ny, cfg.nx, cfg.nv))
    g = o.grad_adjoint(f, w, wrt="abundance")
    cells = rng.choice(cfg.n_cells, size=40, replace=False)
    gfd = o.grad_fd(f, w, cells, eps=1e-5, wrt="abundance")
    assert np.allclose(g.ravel()[cells], gfd, rtol=2e-6, atol=1e-9 * np.abs(gfd).max())
    # the sum over cells is the derivative w.r.t. the logarithm of the GLOBAL abundance: two whole observations
    def L(X):
        return float((w * Oracle(cfg.with_(abundance=X)).observe(f, beam=False, noise=False)).sum())
    X, e = cfg.abundance, 1e-5
    assert (L(X * (1 + e)) - L(X * (1 - e))) / (2 * e) == pytest.approx(g.sum(), rel=1e-5, abs=0.0)
    # optically thin limit, no dust, no background: cell c adds K_RJ j0 h phibar_k to channel k, so
    # dL / d ln X_c = sum_k w_k K_RJ j0_c h phibar_k(c)  -- a closed form per cell
    cfg_t = cfg.with_(abundance=2e-13, dust_on=False, T_cmb=0.0)
    ot = Oracle(cfg_t)
    gt = ot.grad_adjoint(f, w, wrt="abundance").reshape(cfg.nz, -1)
    coef = ot.coefficients(f["nH2"], f["Tgas"], f["Tdust"])
    plane = cfg.nx * cfg.ny
    KRJ = CL ** 2 / (2 * KB * cfg.nu0_Hz ** 2)
    dnuW = cfg.nu0_Hz * cfg.dv_cms / CL
    vk = cfg.v0_cms + np.arange(cfg.nv) * cfg.dv_cms
    p = 14
    vl = f["vlos"].reshape(cfg.nz, plane).astype(np.float64)[:, p, None]
    b = coef[2].reshape(cfg.nz, plane)[:, p, None]
    pb = (special.erf((vk[None] + cfg.dv_cms / 2 - vl) / b) - special.erf((vk[None] - cfg.dv_cms / 2 - vl) / b)) / (2 * dnuW)
    expect = KRJ * coef[0].reshape(cfg.nz, plane)[:, p] * cfg.cell_cm * (pb * w.reshape(plane, cfg.nv)[p][None]).sum(axis=1)
    assert np.allclose(gt[:, p], expect, rtol=1e-4, atol=1e-9 * np.abs(expect).max())


# ------------------------------------------------------------------------------------------------
# tabulated collision rates of several partners
def _power_law_table(cfg, T_grid, split=(1.0,)):
    """The configuration's own power law K_ul(T_ref) (T / T_ref)^p sampled on T_grid, split over partners whose
    fractions times tables add up to it."""
    T_grid = np.asarray(T_grid, dtype=np.float64)
    base = cfg.coll_down_ref[None] * (T_grid[:, None, None] / cfg.coll_T_ref) ** cfg.coll_T_exp
    frac = np.asarray([0.75, 0.25, 0.2][: len(split)], dtype=np.float64)
    table = np.stack([base * sh / fr for sh, fr in zip(split, frac)])
    return cfg.with_(coll_T_grid=T_grid, coll_table=table, coll_partner_frac=frac)


def test_tabulated_rates_reduce_to_the_power_law_and_add_over_partners():
    cfg = base_cfg(10)
    o = Oracle(cfg)
    # at the grid points the table IS the power law; between them linear interpolation of T^0.2 on a 1 K grid is off by <= 1e-5
    grid = np.arange(5.0, 200.5, 1.0)
    ot = Oracle(_power_law_table(cfg, grid))
    for nH2, T in ((1e3, 50.0), (3e5, 119.0), (10.0, 20.0)):
        assert np.allclose(ot.rates(nH2, T), o.rates(nH2, T), rtol=1e-12, atol=0.0)
        # level J is reached through J collisional steps, each off by the interpolation error of its rate (5e-5 at 20 K)
        gap = np.abs(ot.levelpop_cell(nH2, T + 0.37) / o.levelpop_cell(nH2, T + 0.37) - 1.0)
        assert np.all(gap <= 2e-5 * (1 + np.arange(gap.size)))
    # three partners (para-H2, ortho-H2, He) whose weighted tables add up to the same total: identical rates
    o3 = Oracle(_power_law_table(cfg, grid, split=(0.2, 0.5, 0.3)))
    assert np.allclose(o3.rates(2e4, 77.3), ot.rates(2e4, 77.3), rtol=1e-13, atol=0.0)
    # linear interpolation between two grid points, constant outside the grid (reading S30)
    coarse = _power_law_table(cfg, [20.0, 100.0])
    oc = Oracle(coarse)
    K = lambda T: cfg.coll_down_ref[3, 2] * (T / cfg.coll_T_ref) ** cfg.coll_T_exp
    R = oc.rates(1.0, 60.0) - Oracle(cfg.with_(coll_down_ref=0 * cfg.coll_down_ref)).rates(1.0, 60.0)
    # (R is a difference of total rates ~1e-6 s^-1: its rounding is 1e-22 absolute, 1e-11 of this collisional rate)
    assert R[3, 2] == pytest.approx(0.5 * (K(20.0) + K(100.0)), rel=1e-9, abs=0.0)
    Rlo = oc.rates(1.0, 7.0) - Oracle(cfg.with_(coll_down_ref=0 * cfg.coll_down_ref)).rates(1.0, 7.0)
    Rhi = oc.rates(1.0, 500.0) - Oracle(cfg.with_(coll_down_ref=0 * cfg.coll_down_ref)).rates(1.0, 500.0)
    assert Rlo[3, 2] == pytest.approx(K(20.0), rel=1e-9, abs=0.0) and Rhi[3, 2] == pytest.approx(K(100.0), rel=1e-9, abs=0.0)
    # detailed balance survives (Eq. 3.7.2): LTE limit is Boltzmann at the gas temperature
    x = oc.levelpop_cell(1e13, 63.0)
    assert np.allclose(x, boltzmann(cfg, 63.0), rtol=1e-6, atol=0.0)
