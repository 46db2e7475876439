"""Randomised parity campaign: seeded random shapes (ragged, degenerate), channel grids (resolved to badly unresolved
lines, band offsets), molecules (2 - 10 levels), physics (density, abundance over four decades, dust opacity over 3.5
decades, background 0 / 2.7 / 30 K) and every transfer mode / integration / velocity grid / kernel choice, each cube
compared element by element with the float64 oracle.

The bar is the spectrum tolerance of north_star (1e-4 of the pixel's peak + 1e-6 K) plus the allowances DESIGN.md section 6
derives for the regimes a fixed workload never reaches (tests/parity.py): the rounding of the continuum a total or an
absorption line is seen against, the float32 line-centre plane for unresolved lines, the 1.2e-6 accuracy of the level
fractions where emission and absorption cancel, the unsaturated source of the selectively thin mode.  A first run of this
campaign (6000 cases) is where those four limits were found; it found no kernel error."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from iris_inputs import make_fields, make_workload
from oracle import Oracle
from parity import (cancellation_allowance, line_centre_allowance, saturated_source, selthin_source_allowance,
                    spectrum_excess, total_allowance)

pytestmark = pytest.mark.gpu

KMS = 1.0e5
# (transfer_mode, integration, subsample); the hot path gets 6 of 15 draws
MODES = [(0, 0, 0)] * 6 + [(0, 0, 1), (0, 0, 3), (0, 1, 0), (0, 1, 1), (0, 1, 3), (1, 0, 0), (1, 1, 0), (2, 0, 0), (2, 1, 0)]


def draw(seed, case):
    rng = np.random.default_rng(100000 * seed + case)
    nx, ny = int(rng.integers(1, 28)), int(rng.integers(1, 20))
    nz = int(rng.choice([1, 2, 3, 5, 8, 9, 15, 16, 17, 24, 31, 33, 40, 64]))
    nv = int(rng.choice([1, 2, 3, 7, 8, 15, 16, 17, 31, 32, 45, 64, 96, 129, 200, 256]))
    dv = float(rng.choice([0.1, 0.2, 0.25, 0.5, 0.55, 0.6, 1.0, 2.0]))
    m, integ, sub = MODES[int(rng.integers(len(MODES)))]
    dust = bool(rng.integers(2))
    cfg, r = make_workload("small", nx=nx, ny=ny, nz=nz, nv=nv, n_levels=int(rng.integers(2, 11)), dv_kms=dv,
                           seed=int(rng.integers(1 << 30)), mean_n=float(10 ** rng.uniform(1.5, 4.5)),
                           sigma_ln=float(rng.uniform(0.5, 2.5)), sigma_t_kms=float(rng.choice([1.0, 3.0, 10.0])),
                           v_edge_kms=float(rng.choice([0.0, 20.0, 100.0])), dust=dust)
    kw = dict(beam_fwhm_px=0.0, noise_sigma=0.0, transfer_mode=m, integration=integ, subsample=sub,
              abundance=float(10 ** rng.uniform(-8.5, -4.5)), T_cmb=float(rng.choice([0.0, 2.725, 2.725, 30.0])),
              v0_cms=float((0.5 - nv / 2.0) * dv * KMS + rng.uniform(-0.3, 0.3) * nv * dv * KMS),
              microturb_cms=float(rng.choice([0.3, 1.0, 1.0, 3.0])) * KMS,
              subtract_continuum=bool(rng.integers(4) > 0))
    if dust:
        kw["kappa_gas_cm2_g"] = cfg.kappa_gas_cm2_g * float(10 ** rng.uniform(-1.5, 2.0))
    cfg = cfg.with_(**kw)
    algo = int(rng.choice([0, 0, 0, 1, 2, 3]))
    f = make_fields(cfg, r)
    f["vlos"] = (float(rng.choice([0.05, 0.25, 1.0])) * f["vlos"]).astype(np.float32)
    return cfg, f, algo


def allowance(cfg, f, ref):
    """(plain, full): the rounding of the value itself as every fixed-workload test allows it (3e-7 of the total), and the
    sum of the allowances of DESIGN.md section 6."""
    o_sub = ref if cfg.subtract_continuum else Oracle(cfg.with_(subtract_continuum=True)).observe(f)
    o_tot = ref if not cfg.subtract_continuum else Oracle(cfg.with_(subtract_continuum=False)).observe(f)
    plain = 3e-7 * np.abs(o_tot).max(axis=-1, keepdims=True)
    sat = saturated_source(cfg, f) if cfg.transfer_mode == 0 else None
    extra = total_allowance(o_tot, o_sub) + line_centre_allowance(cfg, o_sub, sat)
    if cfg.transfer_mode == 1:
        extra = extra + selthin_source_allowance(cfg, f).reshape(ref.shape)
    if cfg.transfer_mode == 0:
        extra = extra + cancellation_allowance(cfg, f, saturated=sat).reshape(ref.shape)
    return plain, extra


@pytest.mark.parametrize("seed", range(1, 9))
def test_random_configurations_match_the_oracle(seed):
    from paper_2607_01338_b200 import IrisSO
    worst, kernels, beyond_plain = 0.0, {}, 0
    for case in range(120):
        cfg, f, algo = draw(seed, case)
        it = IrisSO(cfg, transfer_algo=algo)
        d = [torch.from_numpy(np.ascontiguousarray(f[k])).cuda() for k in ("nH2", "Tgas", "Tdust", "vlos")]
        cube = it.observe(*d).cpu().numpy()
        what = "seed %d case %d: %d x %d x %d cells, %d channels of %.2f km/s, mode (%d, %d, %d), dust %d, algo %d, kernel %s" % (
            seed, case, cfg.nx, cfg.ny, cfg.nz, cfg.nv, cfg.dv_cms / KMS, cfg.transfer_mode, cfg.integration, cfg.subsample,
            cfg.dust_on, algo, it.transfer_kernel())
        assert np.all(np.isfinite(cube)), what
        ref = Oracle(cfg).observe(f)
        plain, full = allowance(cfg, f, ref)
        ex = float(spectrum_excess(cube, ref, extra=full).max())
        assert ex <= 1.0, "%s: worst pixel at %.3g x the tolerance" % (what, ex)
        ex_plain = float(spectrum_excess(cube, ref, extra=plain).max())
        beyond_plain += ex_plain > 1.0
        if ex_plain <= 1.0:
            worst = max(worst, ex_plain)
        kernels[it.transfer_kernel()] = kernels.get(it.transfer_kernel(), 0) + 1
        it.close()
    print("seed %d: 120 random configurations, %d need more than the plain tolerance (1e-4 peak + 1e-6 K + 3e-7 total); "
          "worst of the others at %.3g of it; kernels %s" % (seed, beyond_plain, worst, kernels))
    # the derived allowances are for rare regimes: almost every draw passes the plain tolerance of the fixed-workload tests
    assert len(kernels) >= 4 and beyond_plain <= 3


def draw_gradient(seed, case):
    rng = np.random.default_rng(7000000 + 100000 * seed + case)
    nx, ny = int(rng.integers(1, 9)), int(rng.integers(1, 7))
    nz = int(rng.choice([1, 2, 3, 9, 17, 40]))
    nv = int(rng.choice([1, 3, 16, 45, 96, 200, 400]))
    integ, sub = [(0, 0), (0, 0), (0, 0), (1, 0), (1, 1), (0, 1), (1, 3)][int(rng.integers(7))]
    cfg, r = make_workload("batch", n=4, nx=nx, ny=ny, nz=nz, nv=nv, n_levels=int(rng.integers(2, 11)),
                           seed=int(rng.integers(1 << 30)), dust=bool(rng.integers(2)), dv_kms=float(rng.choice([0.25, 0.5, 1.0])))
    cfg = cfg.with_(integration=integ, subsample=sub, beam_fwhm_px=float(rng.choice([0.0, 2.0])), out_unit=int(rng.integers(2)),
                    subtract_continuum=bool(rng.integers(2)), abundance=float(10 ** rng.uniform(-7, -4.5)))
    f = make_fields(cfg, r)
    f["vlos"] = (0.2 * f["vlos"]).astype(np.float32)
    wrt = "nH2" if rng.integers(3) else "abundance"
    return cfg, f, wrt


@pytest.mark.parametrize("seed", range(1, 5))
def test_random_gradients_match_the_oracle(seed):
    """iris_so_observe_adjoint / _abundance on random shapes, molecules, abundances and thick modes (hot path: windowed
    closed-form adjoint; smooth integrator / fine grid: stored-state reverse sweep), every cell against the oracle's float64
    reverse-mode adjoint.  Bound per cell: 1e-3 |g| + 1e-5 max|g| (a cell's gradient is a sum over channels of terms of both
    signs: zero crossings sit at ~5e-6 of the largest gradient in float32) + 1e-7 of what the forward peak times the largest
    weight would give (saturated lines: the gradient is a small difference of emission and absorption terms of that size).
    Lines weaker than 0.05 K are skipped: the 1e-8 K window threshold is not small against their gradients."""
    from iris_inputs import weight_cube
    from paper_2607_01338_b200 import IrisSO
    from parity import krj
    ran, worst = 0, 0.0
    for case in range(80):
        cfg, f, wrt = draw_gradient(seed, case)
        o = Oracle(cfg)
        fwd = Oracle(cfg.with_(out_unit=1, subtract_continuum=True, beam_fwhm_px=0.0)).observe(f, beam=False, noise=False)
        peak = float(np.abs(fwd).max())
        if peak < 0.05:
            continue
        w = weight_cube(cfg)
        it = IrisSO(cfg)
        d = [torch.from_numpy(np.ascontiguousarray(f[k])).cuda() for k in ("nH2", "Tgas", "Tdust", "vlos")]
        g = it.observe_adjoint(*d, torch.from_numpy(w).cuda(), wrt=wrt).cpu().numpy().astype(np.float64)
        what = o.beam(w.astype(np.float64)) if cfg.beam_fwhm_px > 0 else w.astype(np.float64)
        ref = o.grad_adjoint(f, what, wrt=wrt).reshape(g.shape)
        unit = 1.0 if cfg.out_unit == 1 else 1.0 / krj(cfg.nu0_Hz)
        absolute = 1e-7 * peak * np.abs(what).max() * unit
        if wrt == "nH2":
            absolute = absolute / np.maximum(f["nH2"].astype(np.float64), 1e-30)
        ex = float(np.max(np.abs(g - ref) / (1e-3 * np.abs(ref) + 1e-5 * np.abs(ref).max() + absolute)))
        assert np.all(np.isfinite(g)) and ex <= 1.0, "seed %d case %d (%d x %d x %d, %d channels, integration %d, subsample %d, %s): %.3g" % (
            seed, case, cfg.nx, cfg.ny, cfg.nz, cfg.nv, cfg.integration, cfg.subsample, wrt, ex)
        worst = max(worst, ex)
        ran += 1
        it.close()
    print("seed %d: %d random gradients, worst cell at %.3g of the bound" % (seed, ran, worst))
    assert ran >= 40


@pytest.mark.parametrize("seed", range(1, 4))
def test_random_molecules_match_the_oracle_populations(seed):
    """K1 on random molecules: 2 - 10 levels, random rate-matrix bandwidths (banded and dense elimination), analytic power-law
    rates with random exponents and a random radiation temperature or random tables (1 - 13 temperatures, 1 - 4 partners),
    densities 1e-2 .. 1e9 cm^-3 and temperatures 5 .. 3000 K drawn log-uniformly per cell; component-wise relative error of
    every level fraction <= 1e-5 (north_star)."""
    from paper_2607_01338_b200 import IrisSO
    from parity import pop_errors
    worst = 0.0
    for case in range(100):
        rng = np.random.default_rng(9000000 + 100000 * seed + case)
        N = int(rng.integers(2, 11))
        max_dj = int(rng.integers(1, N)) if N > 2 else 1
        cfg, _ = make_workload("small", nx=int(rng.integers(1, 50)), ny=int(rng.integers(1, 20)), nz=int(rng.integers(1, 9)), nv=8,
                               n_levels=N, seed=int(rng.integers(1 << 30)))
        if rng.integers(2):
            grid = np.unique(np.round(np.sort(10 ** rng.uniform(0.7, 3.3, int(rng.integers(1, 14)))), 3))
            nP = int(rng.integers(1, 5))
            tab = np.zeros((nP, grid.size, N, N))
            for p in range(nP):
                for u in range(1, N):
                    for l in range(max(0, u - max_dj), u):
                        tab[p, :, u, l] = rng.uniform(0.3, 3.0) * 1e-11 * (grid / 100.0) ** rng.uniform(-0.5, 1.0) / (u - l)
            cfg = cfg.with_(coll_T_grid=grid, coll_table=tab, coll_partner_frac=rng.uniform(0.05, 1.0, nP))
        else:
            Kd = np.array(cfg.coll_down_ref, dtype=np.float64, copy=True)
            for u in range(1, N):
                for l in range(u):
                    Kd[u, l] = (10 ** rng.uniform(-12, -10)) / (u - l) if u - l <= max_dj else 0.0
            cfg = cfg.with_(coll_down_ref=Kd, coll_T_exp=float(rng.uniform(-0.5, 1.5)), T_bar=float(rng.choice([0.0, 2.725, 20.0])))
        n = (10 ** rng.uniform(-2, 9, (cfg.nz, cfg.ny, cfg.nx))).astype(np.float32)
        T = (10 ** rng.uniform(np.log10(5), np.log10(3000), n.shape)).astype(np.float32)
        it = IrisSO(cfg)
        pop = it.levelpop(torch.from_numpy(n).cuda(), torch.from_numpy(T).cuda()).cpu().numpy().reshape(N, -1)
        rel, absmax = pop_errors(pop, np.asarray(Oracle(cfg).levelpop(n, T)).reshape(N, -1))
        assert rel <= 1e-5 and absmax <= 1e-35, "seed %d case %d (%d levels, dJ <= %d, tables %s): rel %.3g" % (
            seed, case, N, max_dj, cfg.coll_table is not None, rel)
        worst = max(worst, rel)
        it.close()
    print("seed %d: 100 random molecules, worst level fraction at %.3g relative" % (seed, worst))
