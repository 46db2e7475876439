"""Pins for the oracle's other transfer / integration modes (PAPER.md sections 4.5 - 4.8): optically thin
(Eq. 4.7.3 - 4.7.7), selectively thin (Eq. 4.6.1 - 4.6.2, 4.8.13 - 4.8.15), smooth integration (TR + BDF2,
Eq. 4.8.10 - 4.8.12, with the ReLU of PAPER.md:709) and the fine velocity grid with Simpson's rule (Eq. 4.5.1).

Closed forms, limits, convergence orders and cross-mode identities -- none retypes the oracle's step formula
against itself, and none involves the CUDA path."""
import numpy as np
import pytest
from scipy import special

from iris_inputs import make_fields, make_workload
from iris_inputs.fields import KMS
from oracle import Oracle

H, KB, CL = 6.62607015e-27, 1.380649e-16, 2.99792458e10


def grid_case(n=4, nv=64, vscale=0.1, **kw):
    cfg, r = make_workload("tiny", n=n, nv=nv)
    f = make_fields(cfg, r)
    f["vlos"] = (vscale * f["vlos"]).astype(np.float32)
    return (cfg.with_(**kw) if kw else cfg), f


def march(cfg, f):
    o = Oracle(cfg)
    coef = o.coefficients(f["nH2"], f["Tgas"], f["Tdust"])
    It, Ic = o.march(coef, f["vlos"])
    return o, coef, It, Ic


def slab(cfg, n=1e3, T=50.0, Td=None):
    shape = (cfg.nz, cfg.ny, cfg.nx)
    return dict(nH2=np.full(shape, n, np.float32), Tgas=np.full(shape, T, np.float32),
                Tdust=np.full(shape, T if Td is None else Td, np.float32), vlos=np.zeros(shape, np.float32))


# ------------------------------------------------------------------------------------------------
# optically thin mode, formal integration: Eq. 4.7.3 - 4.7.6
def test_thin_formal_is_the_emission_integral():
    cfg, f = grid_case(dust_on=True, kappa_gas_cm2_g=0.5, transfer_mode=2)
    o, coef, It, Ic = march(cfg, f)
    Ibg = o.planck(cfg.nu0_Hz, cfg.T_cmb)
    plane = cfg.nx * cfg.ny
    j0, ad, Sd = (coef[i].reshape(cfg.nz, plane) for i in (0, 3, 4))
    # continuum: I_bg + sum h alpha_d S_d (no absorption at all, Eq. 4.7.5)
    assert np.allclose(Ic, Ibg + (ad * Sd).sum(axis=0) * cfg.cell_cm, rtol=1e-13, atol=0.0)
    # velocity-integrated line: sum_v (I_T - I_C) dnu_W = sum_cells j0 h, since the channel-integrated profile sums to 1
    dnuW = cfg.nu0_Hz * cfg.dv_cms / CL
    assert np.allclose((It - Ic[:, None]).sum(axis=1) * dnuW, j0.sum(axis=0) * cfg.cell_cm, rtol=1e-9, atol=0.0)
    # per channel, with the profile from scipy's erf
    p = int(np.argmax((It - Ic[:, None]).max(axis=1)))               # a pixel whose line is inside the band
    vk = cfg.v0_cms + np.arange(cfg.nv) * cfg.dv_cms
    vl = f["vlos"].reshape(cfg.nz, plane).astype(np.float64)[:, p, None]
    b = coef[2].reshape(cfg.nz, plane)[:, p, None]
    pb = (special.erf((vk[None] + cfg.dv_cms / 2 - vl) / b) - special.erf((vk[None] - cfg.dv_cms / 2 - vl) / b)) / (2 * dnuW)
    expect = (j0[:, p, None] * pb).sum(axis=0) * cfg.cell_cm
    assert expect.max() > 1e-3 * Ic[p]
    assert np.allclose(It[p] - Ic[p], expect, rtol=1e-9, atol=4e-16 * Ic[p])


def test_thick_formal_tends_to_thin_as_everything_becomes_transparent():
    """Eq. 4.7.1: dropping the absorption term is exact to first order in tau.  With the background switched off
    (no stimulated absorption of I_bg) the thick and thin cubes differ by O(tau)."""
    gaps = []
    for X in (2e-12, 2e-11):
        cfg, f = grid_case(abundance=X, T_cmb=0.0, T_bar=2.725)
        _, _, I_thick, _ = march(cfg, f)
        _, _, I_thin, _ = march(cfg.with_(transfer_mode=2), f)
        gaps.append(np.max(np.abs(I_thick - I_thin)) / np.max(I_thin))
    assert gaps[0] < 1e-4 and 8.0 < gaps[1] / gaps[0] < 12.0          # the gap is first order in the abundance


# optically thin mode, smooth integration: Simpson, Eq. 4.7.7 -- exact for cubics along the ray
@pytest.mark.parametrize("nz", [9, 10])
def test_thin_smooth_simpson_is_exact_for_a_cubic_emissivity(nz):
    cfg, _ = make_workload("tiny", n=2, nv=8)
    cfg = cfg.with_(nz=nz, abundance=0.0, dust_on=True, kappa_gas_cm2_g=0.3, transfer_mode=2, integration=1)
    z = np.arange(nz, dtype=np.float64)
    poly = 40.0 + 3.0 * z - 0.7 * z ** 2 + 0.05 * z ** 3            # n_H2(z), cubic, positive on the grid
    f = slab(cfg, Td=35.0)
    f["nH2"] = np.broadcast_to(poly[:, None, None], f["nH2"].shape).astype(np.float32)
    o, coef, It, Ic = march(cfg, f)
    Ibg = o.planck(cfg.nu0_Hz, cfg.T_cmb)
    Sd = o.planck(cfg.nu0_Hz, 35.0)
    kr = cfg.kappa_gas_cm2_g * cfg.mass_per_H2_g
    nn = f["nH2"][:, 0, 0].astype(np.float64)                        # what the oracle actually saw (float32 inputs)
    P = np.polynomial.Polynomial.fit(z, nn, 3).integ()
    if nz % 2 == 1:      # whole Simpson panels: exact integral of the cubic over [x_0, x_{R-1}]
        exact = P(z[-1]) - P(z[0])
    else:                # reading S25: the left-over last interval by the trapezoidal rule
        exact = P(z[-2]) - P(z[0]) + 0.5 * (nn[-2] + nn[-1])
    assert Ic[0] == pytest.approx(Ibg + kr * Sd * cfg.cell_cm * exact, rel=1e-6, abs=0.0)
    assert np.allclose(It[0], Ic[0], rtol=1e-14, atol=0.0)


# ------------------------------------------------------------------------------------------------
# selectively thin mode: Eq. 4.6.1 - 4.6.2, 4.8.13 - 4.8.15
def test_selectively_thin_without_dust_is_a_direct_integral():
    """alpha_T = alpha_D = 0 and I_C = I_bg everywhere: dI/ds = (j0 - kappa0 I_bg) phibar, for both integrations
    the formal sum is exact (Eq. 4.8.5 with tau = 0)."""
    cfg, f = grid_case(transfer_mode=1)
    o, coef, It, Ic = march(cfg, f)
    Ibg = o.planck(cfg.nu0_Hz, cfg.T_cmb)
    assert np.allclose(Ic, Ibg, rtol=1e-15, atol=0.0)
    plane = cfg.nx * cfg.ny
    j0, k0 = coef[0].reshape(cfg.nz, plane), coef[1].reshape(cfg.nz, plane)
    dnuW = cfg.nu0_Hz * cfg.dv_cms / CL
    net = ((j0 - k0 * Ibg) * cfg.cell_cm).sum(axis=0)
    clipped = (It <= 0).any(axis=1)                                   # ReLU (reading S26) never binds here
    assert not clipped.any()
    assert np.allclose((It - Ibg).sum(axis=1) * dnuW, net, rtol=1e-9, atol=0.0)


def test_selectively_thin_agrees_with_thick_to_first_order_in_tau():
    """Eq. 4.6.2 drops the line's self-interaction: (thick - selectively thin) / line = O(tau_L) once the dust is
    transparent per cell (with opaque cells the two also differ by O(tau_d): reading S23 pairs the line absorption
    with the continuum AFTER the cell, the thick step with its in-cell evolution)."""
    gaps = []
    for X in (2e-9, 2e-8):
        cfg, f = grid_case(abundance=X, dust_on=True, kappa_gas_cm2_g=1e-6)
        _, _, I0, C0 = march(cfg, f)
        _, _, I1, C1 = march(cfg.with_(transfer_mode=1), f)
        assert np.allclose(C0, C1, rtol=1e-13, atol=0.0)                        # same continuum recurrence
        gaps.append(np.max(np.abs(I0 - I1)) / np.max(np.abs(I0 - C0[:, None])))
    assert gaps[0] < 0.03 and 8.0 < gaps[1] / gaps[0] < 12.0           # relative gap first order, absolute gap second order


def test_selectively_thin_dust_absorbs_the_line():
    """A transparent emitting layer behind an absorbing dust screen: the line is attenuated by exp(-tau_screen)."""
    cfg, _ = make_workload("tiny", n=2, nv=16)
    cfg = cfg.with_(nz=12, dust_on=True, kappa_gas_cm2_g=40.0, transfer_mode=1, abundance=2e-9, T_cmb=0.0)
    f = slab(cfg, n=200.0, T=60.0, Td=1e-3)                           # cold dust: absorbs, does not emit
    o, coef, It, Ic = march(cfg, f)
    # emission only from the far half: zero the tracer in the near half through T_inf is not available per cell,
    # so compare two runs instead: all cells emit vs. the analytic attenuation of each cell's contribution
    tau_cell = coef[3, 0] * cfg.cell_cm
    dnuW = cfg.nu0_Hz * cfg.dv_cms / CL
    vk = cfg.v0_cms + np.arange(cfg.nv) * cfg.dv_cms
    pb = (special.erf((vk + cfg.dv_cms / 2) / coef[2, 0]) - special.erf((vk - cfg.dv_cms / 2) / coef[2, 0])) / (2 * dnuW)
    # cell k (0 = far) emits j0 pb h w(tau_cell) and is then attenuated by the nz - 1 - k cells in front of it
    w = -np.expm1(-tau_cell) / tau_cell
    att = np.exp(-tau_cell * (cfg.nz - 1 - np.arange(cfg.nz))).sum()
    assert tau_cell * cfg.nz > 0.5
    assert np.allclose(It[0], coef[0, 0] * pb * cfg.cell_cm * w * att, rtol=1e-6, atol=1e-40)


# ------------------------------------------------------------------------------------------------
# smooth integration of the thick mode: TR first step + BDF2, Eq. 4.8.10 - 4.8.12
def test_smooth_thick_converges_at_second_order_to_the_slab_solution():
    errs = []
    for nz in (16, 32, 64, 128):
        cfg, _ = make_workload("tiny", n=1, nv=8)
        L = 16 * cfg.cell_cm
        cfg = cfg.with_(nz=nz + 1, cell_cm=L / nz, integration=1, abundance=3e-8)   # R - 1 = nz steps cover L (reading S24)
        f = slab(cfg)
        o, coef, It, Ic = march(cfg, f)
        Ibg = o.planck(cfg.nu0_Hz, cfg.T_cmb)
        dnuW = cfg.nu0_Hz * cfg.dv_cms / CL
        vk = cfg.v0_cms + np.arange(cfg.nv) * cfg.dv_cms
        b = coef[2, 0]
        pb = (special.erf((vk + cfg.dv_cms / 2) / b) - special.erf((vk - cfg.dv_cms / 2) / b)) / (2 * dnuW)
        tau = coef[1, 0] * pb * L
        exact = coef[0, 0] / coef[1, 0] * (1 - np.exp(-tau)) + Ibg * np.exp(-tau)
        assert 0.5 < tau.max() < 20.0
        errs.append(np.max(np.abs(It[0] - exact) / exact))
    ratios = np.array(errs[:-1]) / np.array(errs[1:])
    assert errs[-1] < 2e-4 and np.all(ratios > 3.3) and np.all(ratios < 4.6)      # halving h divides the error by ~4


def quadratic_column(cfg, o, R, mode, seed):
    """Hand-made coefficient planes of one column whose exact smooth-integration answer is known: a method of order two is
    exact when the solution is a quadratic polynomial (TR: the trapezoid of the LINEAR function y' is exact; BDF2: the
    backward difference (3 y_{n+2} - 4 y_{n+1} + y_n) / 2h of a quadratic is its derivative at x_{n+2}).  With absorption
    coefficients alpha_n that differ from cell to cell and sources j_n = y'(x_n) + alpha_n y(x_n), Eq. 4.8.12 followed by
    Eq. 4.8.10 must return y(x_n) at every point -- a swapped alpha_n / alpha_{n+1}, a backward-Euler first step, a shifted
    source index or a continuum taken at the wrong grid point does not.  Returns coef[5, R], the channel the total
    intensity was built for, and the two quadratics (continuum, total) at the grid points."""
    rng = np.random.default_rng(seed)
    h = cfg.cell_cm
    x = np.arange(R) * h
    Ibg = o.planck(cfg.nu0_Hz, cfg.T_cmb)
    L = (R - 1) * h

    def quad(c1, c2):                                   # y(0) = I_bg, positive on the grid
        return Ibg * (1 + c1 * x / L + c2 * (x / L) ** 2), Ibg * (c1 / L + 2 * c2 * x / L ** 2)

    yC, dC = quad(0.8, 1.7)
    yT, dT = quad(2.5, -0.9)
    ad = rng.uniform(0.1, 1.5, R) / h                   # dust optical depth per step 0.1 .. 1.5, different in every cell
    Sd = (dC + ad * yC) / ad                            # j_D = alpha_d S_d = y_C' + alpha_d y_C
    k = cfg.nv // 2
    b = np.full(R, 1.3e5)
    p = o.phibar(k, 0.0, 1.3e5)                         # v_los = 0 and one Doppler width: the same profile value in every cell
    k0 = rng.uniform(0.2, 2.0, R) / (h * p)             # line optical depth per step 0.2 .. 2 in channel k
    if mode == 0:                                       # thick: alpha_T = kappa0 p + alpha_d, j_T = j0 p + alpha_d S_d
        j0 = (dT + (k0 * p + ad) * yT - ad * Sd) / p
    else:                                               # selectively thin (Eq. 4.8.14 - 4.8.15, reading S23: I_C at x_n)
        j0 = (dT + ad * yT - ad * Sd + k0 * p * yC) / p
    return np.stack([j0, k0, b, ad, Sd]), k, yC, yT


@pytest.mark.parametrize("mode", [0, 1])
@pytest.mark.parametrize("R", [2, 3, 4, 9])
def test_smooth_integrator_is_exact_for_quadratic_solutions(R, mode):
    """Pins the trapezoidal first step (Eq. 4.8.12; R = 2 is that step alone) and the BDF2 steps
    (Eq. 4.8.10) with non-uniform absorption, for the continuum and for the total intensity."""
    cfg, _ = make_workload("tiny", n=1, nv=8)
    cfg = cfg.with_(nz=R, integration=1, transfer_mode=mode, dust_on=True)
    o = Oracle(cfg)
    coef, k, yC, yT = quadratic_column(cfg, o, R, mode, seed=10 * R + mode)
    assert yC.min() > 0 and yT.min() > 0                # the ReLU (reading S26) does not act
    It, Ic = o.march(coef, np.zeros(R, np.float32))
    assert Ic[0] == pytest.approx(yC[-1], rel=1e-12, abs=0.0)
    assert It[0, k] == pytest.approx(yT[-1], rel=1e-12, abs=0.0)
    # the same column through the formal integrator is NOT exact (it assumes stepwise-constant coefficients), so the
    # agreement above is a property of TR + BDF2 and not of the construction
    Itf, Icf = Oracle(cfg.with_(integration=0)).march(coef, np.zeros(R, np.float32))
    assert abs(Icf[0] / yC[-1] - 1) > 1e-3 and abs(Itf[0, k] / yT[-1] - 1) > 1e-3


def test_trapezoidal_first_step_has_third_order_local_error():
    """One TR step (R = 2) over a medium whose absorption varies linearly along the ray, constant source function S:
    exact answer S + (I_bg - S) exp(-integral of alpha).  Halving h divides the one-step error by ~8 (a backward-Euler
    first step would give ~4)."""
    cfg, _ = make_workload("tiny", n=1, nv=8)
    errs = []
    for m in (2, 4, 8, 16):
        c = cfg.with_(nz=2, integration=1, dust_on=True, cell_cm=cfg.cell_cm / m)
        o = Oracle(c)
        Ibg = o.planck(c.nu0_Hz, c.T_cmb)
        S = 7.0 * Ibg
        a0, slope = 0.3 / cfg.cell_cm, 0.9 / cfg.cell_cm ** 2          # alpha(x) = a0 + slope x
        ad = np.array([a0, a0 + slope * c.cell_cm])
        coef = np.stack([np.zeros(2), np.zeros(2), np.full(2, 1e5), ad, np.full(2, S)])
        _, Ic = o.march(coef, np.zeros(2, np.float32))
        tau = a0 * c.cell_cm + 0.5 * slope * c.cell_cm ** 2
        errs.append(abs(Ic[0] - (S + (Ibg - S) * np.exp(-tau))))
    ratios = np.array(errs[:-1]) / np.array(errs[1:])
    assert np.all(ratios > 7.0) and np.all(ratios < 9.0)


def test_selectively_thin_formal_continuum_pairing_is_a_reading_bounded_by_the_dust_depth():
    """Reading S23 (NOT fixed by the paper, "solve for the continuum step first, and then use the continuum
    intensity"): in the formal selectively thin step the line absorbs the continuum AFTER its own step of that cell.  The
    other reading (the continuum BEFORE the cell) is marched here in numpy next to it; the oracle is the first one, and
    the two differ by O(tau_d) of the absorbed continuum: the gap is proportional to the dust opacity."""
    gaps = []
    for kappa in (0.25, 0.5):
        cfg, f = grid_case(n=6, nv=32, abundance=3e-9, dust_on=True, kappa_gas_cm2_g=kappa, transfer_mode=1, T_cmb=30.0)
        f["Tdust"] = np.full_like(f["Tdust"], 5.0)                      # continuum changes along the ray: absorbed background
        o, coef, It, Ic = march(cfg, f)
        plane, R, h = cfg.nx * cfg.ny, cfg.nz, cfg.cell_cm
        j0, k0, b, ad, Sd = (coef[i].reshape(R, plane) for i in range(5))
        vl = f["vlos"].reshape(R, plane).astype(np.float64)
        Ibg = o.planck(cfg.nu0_Hz, cfg.T_cmb)
        pix = 17
        res = {}
        for which in ("after", "before"):
            I = np.full(cfg.nv, Ibg)
            C = Ibg
            for n in range(R):
                tau = ad[n, pix] * h
                w = -np.expm1(-tau) / tau
                Cn = C * np.exp(-tau) + ad[n, pix] * Sd[n, pix] * h * w
                pb = np.array([o.phibar(k, vl[n, pix], b[n, pix]) for k in range(cfg.nv)])
                jT = j0[n, pix] * pb + ad[n, pix] * Sd[n, pix] - k0[n, pix] * pb * (Cn if which == "after" else C)
                I = np.maximum(I * np.exp(-tau) + jT * h * w, 0.0)
                C = Cn
            res[which] = I
        assert np.allclose(It[pix], res["after"], rtol=1e-12, atol=0.0)
        assert res["after"].min() > 0.3 * Ic[pix]                       # absorption line on the continuum, far from the ReLU
        line = np.abs(res["after"] - Ic[pix]).max()
        tau_d = (ad[:, pix] * h).max()
        gap = np.abs(res["after"] - res["before"]).max() / line
        # per cell the two readings absorb kappa0 p h w (C_n - C_{n-1}) differently, and |C_n - C_{n-1}| <= tau_d C
        assert 0.05 * tau_d < gap < tau_d
        gaps.append(gap)
    assert 1.8 < gaps[1] / gaps[0] < 2.2


def test_smooth_thick_is_stable_and_clamped_for_huge_optical_depth():
    """A-stability: tau per step >> 1 regresses to the source function instead of diverging; the ReLU
    keeps a dark, absorbing column at exactly zero."""
    cfg, _ = make_workload("tiny", n=1, nv=8)
    cfg = cfg.with_(nz=24, integration=1, abundance=2e-2)
    f = slab(cfg)
    o, coef, It, Ic = march(cfg, f)
    S = coef[0, 0] / coef[1, 0]
    k = cfg.nv // 2
    assert coef[1, 0] * o.phibar(k, 0.0, coef[2, 0]) * cfg.cell_cm > 1e3
    assert It[0, k] == pytest.approx(S, rel=1e-3, abs=0.0)
    # ReLU: bright background, no emission, strong absorption switched on abruptly -> BDF2 overshoots below zero
    cfg2 = cfg.with_(abundance=0.0, dust_on=True, kappa_gas_cm2_g=1.0, T_cmb=50.0)
    f2 = slab(cfg2, n=1.0, Td=1e-3)
    f2["nH2"][3:] = 3e5                                                # tau_d per step ~ 1.3 from cell 3 on
    o2, coef2, It2, Ic2 = march(cfg2, f2)
    free = march(cfg2.with_(integration=0), f2)[3]
    assert Ic2[0] >= 0.0 and free[0] > 0.0 and Ic2[0] < 1e-3 * o2.planck(cfg2.nu0_Hz, 50.0)


def test_smooth_selectively_thin_converges_to_its_formal_solution():
    errs = []
    for m in (1, 2, 4):
        cfg, f = grid_case(n=6, nv=32, abundance=2e-7, dust_on=True, kappa_gas_cm2_g=2.0, transfer_mode=1)
        fm = {k: np.repeat(f[k], m, axis=0) for k in f}
        cfg_m = cfg.with_(nz=cfg.nz * m, cell_cm=cfg.cell_cm / m)
        _, _, If, Cf = march(cfg_m, fm)
        _, _, Is, Cs = march(cfg_m.with_(integration=1), fm)
        errs.append(np.max(np.abs(Is - If)) / np.max(np.abs(If)))
    assert errs[2] < errs[1] < errs[0] and errs[2] < 0.1


# ------------------------------------------------------------------------------------------------
# fine velocity grid + Simpson's rule over frequency, Eq. 4.5.1 (thick mode)
def test_fine_grid_simpson_converges_to_brute_force_frequency_integration():
    cfg, f = grid_case(n=4, nv=48, vscale=0.05, abundance=2e-6, dust_on=True, kappa_gas_cm2_g=0.5)
    o, coef, I_r1, Ic = march(cfg, f)
    gaps = []
    for sub in (1, 3, 7):
        _, _, It, Ic2 = march(cfg.with_(subsample=sub), f)
        assert np.allclose(Ic2, Ic, rtol=1e-13, atol=0.0)
        gap = 0.0
        for pix in (0, 7, 13):
            br = o.brute_column(coef, f["vlos"], pix, 400)           # midpoint rule, 400 points per channel
            gap = max(gap, np.max(np.abs(br - It[pix])) / np.max(np.abs(br - Ic[pix])))
        gaps.append(gap)
    # channel width 0.5 km/s against b ~ 1 km/s: even one midpoint per channel is within 1e-3; converges fast
    assert gaps[0] < 2e-3 and gaps[2] < gaps[1] < gaps[0] and gaps[2] < 2e-5
    # and the hot path's channel-integrated profile (reading R1) is the tau -> 0 limit of the same thing
    cfg_thin = cfg.with_(abundance=2e-11)
    _, _, A, CA = march(cfg_thin, f)
    _, _, B, CB = march(cfg_thin.with_(subsample=7), f)
    assert np.max(np.abs(A - B)) / np.max(np.abs(A - CA[:, None])) < 1e-5


def test_fine_grid_undersampling_failure_mode():
    """PAPER.md:893 ("shotgun" failure): with lines much narrower than a channel and no subsampling (centre value
    only = subsample 1's Simpson midpoint weight 4/6) emission is missed or over-counted; enough midpoints fix it."""
    cfg, f = grid_case(n=4, nv=24, vscale=0.3, abundance=2e-12, microturb_cms=0.0, dv_cms=2.0 * KMS,
                       v0_cms=-23.0 * KMS)
    o, coef, I_int, Ic = march(cfg, f)                               # integrated profile: exact in the thin limit
    line = np.abs(I_int - Ic[:, None]).max()
    coarse = march(cfg.with_(subsample=1), f)[2]
    fine = march(cfg.with_(subsample=63), f)[2]
    assert np.max(np.abs(coarse - I_int)) / line > 0.2
    assert np.max(np.abs(fine - I_int)) / line < 2e-4


# ------------------------------------------------------------------------------------------------
# diagnostics: density tracing (section 5.10) and the error metrics of section 5.1
def test_density_trace_conserves_column_density_and_bins_by_velocity():
    cfg, r = make_workload("tiny", n=6, nv=64)
    f = make_fields(cfg, r)
    f["vlos"] = (0.4 * f["vlos"]).astype(np.float32)
    o = Oracle(cfg)
    cube = o.density_trace(f)
    plane = cfg.nx * cfg.ny
    n = f["nH2"].reshape(cfg.nz, plane).astype(np.float64)
    v = f["vlos"].reshape(cfg.nz, plane).astype(np.float64)
    lo, hi = cfg.v0_cms - cfg.dv_cms / 2, cfg.v0_cms + (cfg.nv - 0.5) * cfg.dv_cms
    inband = (v >= lo) & (v < hi)
    assert inband.mean() > 0.2 and (~inband).any()
    # total column density of the in-band cells: sum_v cube dv = sum_z n h
    assert np.allclose(cube.reshape(plane, cfg.nv).sum(axis=1) * cfg.dv_cms, (n * inband).sum(axis=0) * cfg.cell_cm, rtol=1e-12, atol=0.0)
    # against numpy's histogram of one column
    p = int(np.argmax(inband.sum(axis=0)))
    edges = lo + cfg.dv_cms * np.arange(cfg.nv + 1)
    hist, _ = np.histogram(v[:, p], bins=edges, weights=n[:, p] * cfg.cell_cm / cfg.dv_cms)
    assert np.allclose(cube.reshape(plane, cfg.nv)[p], hist, rtol=1e-12, atol=0.0)


def test_density_trace_is_the_thin_observation_of_an_isothermal_cold_cloud():
    """Section 5.10 / Eq. 5.10.1: with one temperature, no dust and no absorption the optically thin line cube is
    proportional to the density-tracing cube.  Lines much narrower than a channel and velocities at channel centres make
    the channel-integrated profile an indicator of the channel, so the proportionality is exact: the constant is
    (h nu0 / 4 pi) X x_u(T) A_ul dv / dnu_W  with x_u from the LTE limit (high density)."""
    cfg, r = make_workload("tiny", n=4, nv=32)
    cfg = cfg.with_(transfer_mode=2, microturb_cms=0.0, dv_cms=4.0 * KMS, v0_cms=-62.0 * KMS, subtract_continuum=True, out_unit=0)
    rng = np.random.default_rng(3)
    shape = (cfg.nz, cfg.ny, cfg.nx)
    f = dict(nH2=(1e12 * rng.uniform(0.5, 2.0, shape)).astype(np.float32), Tgas=np.full(shape, 15.0, np.float32),
             Tdust=np.full(shape, 15.0, np.float32),
             vlos=(cfg.v0_cms + cfg.dv_cms * rng.integers(0, cfg.nv, shape)).astype(np.float32))
    o = Oracle(cfg)
    line = o.observe(f, beam=False, noise=False)              # I_T - I_C in cgs
    trace = o.density_trace(f)
    x = cfg.weight * np.exp(-cfg.energy_K / 15.0)
    x /= x.sum()
    A = cfg.einstein_A[cfg.line_upper, cfg.line_lower]
    const = H * cfg.nu0_Hz / (4 * np.pi) * cfg.abundance * x[cfg.line_upper] * A * cfg.dv_cms / (cfg.nu0_Hz * cfg.dv_cms / CL)
    assert trace.max() > 0
    assert np.allclose(line, const * trace, rtol=2e-5, atol=1e-12 * (const * trace).max())


def test_tsre_and_tam_definitions():
    o = Oracle(make_workload("tiny", n=2, nv=4)[0])
    rng = np.random.default_rng(0)
    T1 = rng.normal(0.0, 0.2, (5, 7, 6))
    T2 = T1 * rng.uniform(0.5, 1.5, T1.shape) + rng.normal(0.0, 0.02, T1.shape)
    m = o.metrics(T1, T2)
    Tmin = 5e-2
    act = (np.abs(T1) > Tmin) & (np.abs(T2) > Tmin)
    ts = np.where(act, 2 * np.abs(T1 - T2) / (np.abs(T1) + np.abs(T2) + 1e-300), 0.0)
    assert m["tsre_lbv"] == pytest.approx(ts.mean(), rel=1e-12, abs=0.0)
    def img(a, b):
        ok = (np.abs(a) > Tmin) & (np.abs(b) > Tmin)
        return np.where(ok, 2 * np.abs(a - b) / (np.abs(a) + np.abs(b) + 1e-300), 0.0).mean()
    assert m["tsre_lb"] == pytest.approx(img(T1.mean(axis=2), T2.mean(axis=2)), rel=1e-12, abs=0.0)
    assert m["tsre_lv"] == pytest.approx(img(T1.mean(axis=0), T2.mean(axis=0)), rel=1e-12, abs=0.0)
    assert m["tam1"] == pytest.approx(T1[np.abs(T1) > Tmin].mean(), rel=1e-12, abs=0.0) and m["active1"] == (np.abs(T1) > Tmin).sum()
    assert m["max2"] == T2.max()
    # properties the paper states: identical cubes -> 0; opposite signs -> 200 %; capped at 200 %
    assert o.metrics(T1, T1)["tsre_lbv"] == 0.0
    big = np.full((2, 2, 2), 1.0)
    assert o.metrics(big, -big)["tsre_lbv"] == pytest.approx(2.0)
    assert o.metrics(big, 1e9 * big)["tsre_lbv"] == pytest.approx(2.0, rel=1e-8, abs=0.0)
    assert o.metrics(big, 1e-3 * big)["tsre_lbv"] == 0.0 and o.metrics(1e-3 * big, big)["tam1"] == 0.0


# ------------------------------------------------------------------------------------------------
# dust source, background and unit conversion at every channel's own frequency (reading S32)
def _planck(nu, T):
    return 2 * H * nu ** 3 / CL ** 2 / np.expm1(H * nu / (KB * T))


def test_per_channel_dust_slab_closed_form_and_doppler_shift():
    """Dust only, uniform slab: I_cont,k = B_nu'(T_d) (1 - e^-tau) + B_nu_k(T_cmb) e^-tau with nu_k = nu0 (1 - v_k / c) and,
    for dust moving with v_los, nu' = nu_k (1 + v_los / c).  A dropped or mis-signed shift changes the answer by
    3e-4 relative (v / c times d ln B / d ln nu), far above the 1e-12 asked here."""
    cfg, _ = make_workload("tiny", n=2, nv=16)
    cfg = cfg.with_(nz=7, abundance=0.0, dust_on=True, kappa_gas_cm2_g=0.8, dust_per_channel=1, dv_cms=8.0 * KMS, v0_cms=-60.0 * KMS)
    o = Oracle(cfg)
    for vl in (0.0, 3.1e6):
        f = slab(cfg, n=2.0e3, T=40.0, Td=33.0)
        f["vlos"] = np.full_like(f["vlos"], vl)
        coef = o.coefficients(f["nH2"], f["Tgas"], f["Tdust"])
        It, Ic = o.march_perchannel(coef, f["vlos"], f["Tdust"])
        tau = coef[3, 0] * cfg.nz * cfg.cell_cm
        assert 0.05 < tau < 5
        vk = cfg.v0_cms + np.arange(cfg.nv) * cfg.dv_cms
        nuk = cfg.nu0_Hz * (1 - vk / CL)
        assert np.allclose([o.channel_frequency(k) for k in range(cfg.nv)], nuk, rtol=1e-15, atol=0.0)
        vl32 = float(np.float32(vl))
        expect = _planck(nuk * (1 + vl32 / CL), 33.0) * -np.expm1(-tau) + _planck(nuk, cfg.T_cmb) * np.exp(-tau)
        assert np.allclose(Ic[0], expect, rtol=1e-12, atol=0.0) and np.allclose(It[0], Ic[0], rtol=1e-14, atol=0.0)
        # against the channel-constant reading (S6): first order in v / c
        _, Ic0 = Oracle(cfg.with_(dust_per_channel=0)).march(coef, f["vlos"])
        gap = np.abs(Ic[0] / Ic0[0] - 1)
        assert 1e-5 < gap.max() < 2e-3 and gap[np.argmin(np.abs(vk - vl))] < gap.max()


def test_per_channel_dust_in_equilibrium_with_the_background_and_opaque_isothermal_slab():
    cfg, _ = make_workload("tiny", n=2, nv=12)
    cfg = cfg.with_(nz=5, abundance=0.0, dust_on=True, kappa_gas_cm2_g=2.0, dust_per_channel=1, dv_cms=5.0 * KMS, v0_cms=-27.5 * KMS)
    # dust at rest at the background temperature: nothing changes, whatever tau, in every channel
    f = slab(cfg, n=5.0e3, T=40.0, Td=cfg.T_cmb)
    o = Oracle(cfg)
    It, Ic = o.march_perchannel(o.coefficients(f["nH2"], f["Tgas"], f["Tdust"]), f["vlos"], f["Tdust"])
    Td32 = float(np.float32(cfg.T_cmb))
    for k in range(cfg.nv):
        lo, hi = sorted((_planck(o.channel_frequency(k), Td32), _planck(o.channel_frequency(k), cfg.T_cmb)))
        assert lo * (1 - 1e-13) <= Ic[0, k] <= hi * (1 + 1e-13)
    # an opaque isothermal slab is a black body at every channel: Planck brightness temperature = T_d in all channels
    c2 = cfg.with_(kappa_gas_cm2_g=400.0, out_unit=2, subtract_continuum=False)
    f2 = slab(c2, n=5.0e3, T=40.0, Td=57.0)
    cube = Oracle(c2).observe(f2, beam=False, noise=False)
    assert np.allclose(cube, 57.0, rtol=1e-10, atol=0.0)
    # ... which the channel-constant conversion does not give
    It2, Ic2 = Oracle(c2).march_perchannel(Oracle(c2).coefficients(f2["nH2"], f2["Tgas"], f2["Tdust"]), f2["vlos"], f2["Tdust"])
    assert abs(Oracle(c2).planck_TB(c2.nu0_Hz, It2[0, 0]) - 57.0) > 1e-3


def test_per_channel_dust_leaves_the_line_terms_alone():
    """Dust off: the per-channel background B_nu_k(T_cmb) is all that differs; with T_cmb = 0 the two readings agree."""
    cfg, f = grid_case(n=4, nv=48, T_cmb=0.0, T_bar=2.725)
    o = Oracle(cfg.with_(dust_per_channel=1))
    coef = o.coefficients(f["nH2"], f["Tgas"], f["Tdust"])
    It, Ic = o.march_perchannel(coef, f["vlos"], f["Tdust"])
    It0, Ic0 = Oracle(cfg).march(coef, f["vlos"])
    assert np.all(Ic == 0.0) and np.allclose(It, It0, rtol=1e-14, atol=0.0) and It0.max() > 0


# ------------------------------------------------------------------------------------------------
# Gradient outside the hot-path mode (the pipeline is differentiable end to end, and its production mode
# is thick + smooth + f = 1): the oracle's reverse-mode adjoint of the thick mode with the smooth integrator and / or the
# fine grid, against (a) central differences of the oracle's OWN forward march of that mode, cell by cell, and (b) the
# directional derivative of the whole observation (beam included) through observe().
ADJ_MODES = {"thick_smooth": (1, 0), "thick_smooth_sub1": (1, 1), "thick_smooth_sub3": (1, 3), "thick_formal_sub1": (0, 1),
             "thick_formal_sub3": (0, 3)}


@pytest.mark.parametrize("regime", ["plain", "relu_active"])
@pytest.mark.parametrize("mode", ADJ_MODES)
def test_adjoint_of_the_thick_modes_matches_finite_differences(mode, regime):
    integ, sub = ADJ_MODES[mode]
    cfg, r = make_workload("tiny", nx=3, ny=2, nz=9, nv=24)
    cfg = cfg.with_(integration=integ, subsample=sub, dust_on=True, kappa_gas_cm2_g=0.05, beam_fwhm_px=2.0)
    f = make_fields(cfg, r)
    f["vlos"] = (0.2 * f["vlos"]).astype(np.float32)
    if regime == "relu_active":
        if integ == 0:
            pytest.skip("the formal thick step has no ReLU")
        # bright background behind cold dust that turns opaque abruptly: the BDF2 continuum and the line points overshoot
        # below zero and are clamped (the regime of test_gpu_modes.py "opaque_dust_clamp")
        cfg = cfg.with_(T_cmb=60.0, kappa_gas_cm2_g=3.0)
        f["Tdust"] = np.full_like(f["Tdust"], 3.0)
        f["nH2"][: cfg.nz // 2] *= 1e-3
        f["nH2"][cfg.nz // 2:] *= 30.0
        # the clamp did fire: a column cut short after cell n ends in the state the full march passes through at n
        fired = False
        for cut in range(cfg.nz // 2 + 1, cfg.nz + 1):
            fc = {k: np.ascontiguousarray(f[k][:cut]) for k in ("nH2", "Tgas", "Tdust", "vlos")}
            tot = Oracle(cfg.with_(nz=cut, subtract_continuum=False, out_unit=0)).observe(fc, beam=False, noise=False)
            fired = fired or bool((tot == 0.0).any())
        assert fired
    o = Oracle(cfg)
    rng = np.random.default_rng(11)
    w = rng.random((cfg.ny, cfg.nx, cfg.nv)) - 0.3
    what = o.beam(w)
    g = o.grad_adjoint(f, what)
    assert np.all(np.isfinite(g)) and np.abs(g).max() > 0
    cells = np.arange(cfg.n_cells)
    # (behind the 60 K background of the clamped regime L is ~1e7 times a cell's contribution: the rounding of the
    # difference quotient asks for a wider bracket there; measured: the gap to the adjoint falls as 1 / eps down to 4e-6 at
    # eps = 1e-3.  A ReLU kink inside a bracket would show up as one outlier; none for this seed)
    gfd = o.grad_fd(f, what, cells, eps=1e-3 if regime == "relu_active" else 1e-5)
    scale = np.abs(gfd).max()
    assert np.allclose(g.ravel(), gfd, rtol=2e-5 if regime == "relu_active" else 5e-6, atol=1e-8 * scale)
    # whole-pipeline directional derivative through observe(), beam applied to the cube
    d = rng.standard_normal(f["nH2"].shape) * f["nH2"] * 1e-3
    np_ = (f["nH2"].astype(np.float64) + d).astype(np.float32)
    nm_ = (f["nH2"].astype(np.float64) - d).astype(np.float32)
    dd = np_.astype(np.float64) - nm_.astype(np.float64)

    def L(nH2):
        ff = dict(f)
        ff["nH2"] = nH2
        return float((w * o.observe(ff, beam=True, noise=False)).sum())
    assert (L(np_) - L(nm_)) == pytest.approx(float((g * dd).sum()), rel=2e-4, abs=0.0)


def test_adjoint_of_the_fine_grid_tends_to_the_hot_path_adjoint_for_resolved_lines():
    """For an optically thin line the intensity is linear in the profile, so the Simpson average of the point profile over
    a channel (Eq. 4.5.1) IS the channel-integrated profile of Eq. 4.6.3 to O((dv / (m b))^4): the gradient of the thick
    formal mode on the fine grid tends to the hot-path gradient, which round 1 pinned on its own (test_oracle_pins.py,
    pin 13).  (A thick line does not: averaging intensities and averaging the profile inside the exponent differ.)"""
    cfg, r = make_workload("tiny", nx=2, ny=2, nz=8, nv=48)
    cfg = cfg.with_(dust_on=True, kappa_gas_cm2_g=0.05, dv_cms=0.25 * cfg.dv_cms, v0_cms=0.25 * cfg.v0_cms,
                    abundance=1e-6 * cfg.abundance)
    f = make_fields(cfg, r)
    f["vlos"] = (0.05 * f["vlos"]).astype(np.float32)
    rng = np.random.default_rng(12)
    w = rng.random((cfg.ny, cfg.nx, cfg.nv))
    g0 = Oracle(cfg).grad_adjoint(f, w)
    errs = []
    for sub in (1, 3):
        g = Oracle(cfg.with_(subsample=sub)).grad_adjoint(f, w)
        errs.append(np.abs(g - g0).max() / np.abs(g0).max())
    assert errs[0] < 1e-3 and errs[1] < errs[0] / 8.0, errs


def test_adjoint_of_the_other_transfer_modes_is_not_claimed():
    cfg, r = make_workload("tiny", nx=2, ny=1, nz=4, nv=8)
    f = make_fields(cfg, r)
    w = np.ones((cfg.ny, cfg.nx, cfg.nv))
    for m in (1, 2):
        assert np.all(np.isnan(Oracle(cfg.with_(transfer_mode=m)).grad_adjoint(f, w)))
