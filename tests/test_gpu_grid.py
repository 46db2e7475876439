"""GPU parity of the coefficient grid (section 4.2 / 4.3: grid precomputation, runtime lookup by linear
interpolation, linear continuation outside the grid; reading S31) against the oracle's grid functions on the same seeded
inputs, plus the (reported, not asserted against a tolerance of the method) gap between the lookup and the per-cell solve."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from iris_inputs import make_fields, make_workload
from oracle import Oracle
from parity import assert_spectra, krj

pytestmark = pytest.mark.gpu


def dev_fields(f):
    return [torch.from_numpy(np.ascontiguousarray(f[k])).cuda() for k in ("nH2", "Tgas", "Tdust", "vlos")]


def iris(cfg, algo=0):
    from paper_2607_01338_b200 import IrisSO
    return IrisSO(cfg, transfer_algo=algo)


GRIDS = {"paper_128x64": dict(), "coarse_17x9": dict(grid_n_density=17, grid_n_temp=9),
         "two_nodes": dict(grid_n_density=2, grid_n_temp=2, grid_nH2_lo=10.0, grid_nH2_hi=1.0e5, grid_T_lo=20.0, grid_T_hi=200.0),
         "fields_outside_the_grid": dict(grid_n_density=33, grid_n_temp=17, grid_nH2_lo=1.0e2, grid_nH2_hi=2.0e4, grid_T_lo=40.0,
                                         grid_T_hi=100.0)}


@pytest.mark.parametrize("grid", GRIDS)
@pytest.mark.parametrize("name", ["tiny", "small"])
def test_grid_cube_matches_the_oracle_grid(name, grid):
    cfg, r = make_workload(name, n=24, nv=96)
    cfg = cfg.with_(coef_grid=1, **GRIDS[grid])
    f = make_fields(cfg, r)
    f["vlos"] = (0.25 * f["vlos"]).astype(np.float32)
    if grid == "fields_outside_the_grid":
        # a third of the cells are extrapolated, on every side.  (The node differences are float32 on the device: a point
        # u cells beyond the grid carries u times their rounding, so parity with the float64 oracle is asked up to
        # ~30 cells outside, not arbitrarily far.)
        inside = (f["nH2"] >= 1e2) & (f["nH2"] <= 2e4) & (f["Tgas"] >= 40) & (f["Tgas"] <= 100)
        assert 0.3 < inside.mean() < 0.8 and (f["nH2"] > 2e4).any() and (f["nH2"] < 1e2).any()
    cube = iris(cfg).observe(*dev_fields(f)).cpu().numpy()
    ref = Oracle(cfg).observe(f)
    worst = assert_spectra(cube, ref, what="%s, grid %s" % (name, grid))
    print("%s grid %s: worst pixel at %.3g of tolerance, peak %.3g K" % (name, grid, worst, np.abs(ref).max()))


def test_grid_transfer_intensities_T_inf_and_other_kernels():
    """iris_so_transfer with the lookup (cgs intensities), the T_inf mask after the lookup, and the lookup feeding the
    dense kernel and a mode kernel as well (the grid replaces K1 only)."""
    cfg, r = make_workload("small", n=20, nv=80)
    cfg = cfg.with_(coef_grid=1, T_inf=90.0)
    f = make_fields(cfg, r)
    f["vlos"] = (0.2 * f["vlos"]).astype(np.float32)
    assert (f["Tgas"] > 90.0).any()
    o = Oracle(cfg)
    It, Ic = iris(cfg).transfer(*dev_fields(f))
    rt, rc = o.march(o.coefficients(f["nH2"], f["Tgas"], f["Tdust"]), f["vlos"])
    It, Ic = It.cpu().numpy().reshape(-1, cfg.nv).astype(np.float64), Ic.cpu().numpy().ravel().astype(np.float64)
    assert np.allclose(Ic, rc, rtol=3e-6, atol=0.0)
    line = np.abs(rt - rc[:, None]).max(axis=1)
    assert np.all(np.abs(It - rt).max(axis=1) <= 1e-4 * line + 1e-6 / krj(cfg.nu0_Hz) + 3e-7 * np.abs(rt).max(axis=1))
    ref = o.observe(f)
    assert_spectra(iris(cfg, 1).observe(*dev_fields(f)).cpu().numpy(), ref, what="dense kernel on grid coefficients")
    c2 = cfg.with_(integration=1, subsample=1)
    assert_spectra(iris(c2).observe(*dev_fields(f)).cpu().numpy(), Oracle(c2).observe(f), what="production mode on grid coefficients")


def test_grid_gap_to_the_exact_solve_is_second_order():
    """Reported: how far the interpolated cube is from the cube of the per-cell level solve (both on the GPU).  The gap is
    the error of the paper's METHOD (linear interpolation on a coarse grid), not of the kernel; it must fall by ~4 per
    doubling of the nodes."""
    cfg, r = make_workload("small", n=32, nv=96)
    f = make_fields(cfg, r)
    f["vlos"] = (0.3 * f["vlos"]).astype(np.float32)
    d = dev_fields(f)
    exact = iris(cfg).observe(*d, beam=False, noise=False)
    peak = exact.abs().amax(dim=-1, keepdim=True)
    gaps = []
    for nn, nT in ((33, 17), (65, 33), (129, 65)):
        c = cfg.with_(coef_grid=1, grid_n_density=nn, grid_n_temp=nT, grid_nH2_lo=1.0, grid_nH2_hi=1.0e7, grid_T_lo=10.0, grid_T_hi=300.0)
        cube = iris(c).observe(*d, beam=False, noise=False)
        gaps.append(((cube - exact).abs() / (peak + 1e-3)).max().item())
    print("grid vs exact solve, max |dT| / peak for 33x17, 65x33, 129x65 nodes: %.2e %.2e %.2e" % tuple(gaps))
    assert gaps[2] < gaps[1] < gaps[0] and gaps[0] / gaps[2] > 8.0


def test_grid_refuses_the_adjoint_and_bad_grids():
    from paper_2607_01338_b200 import IrisSOError
    cfg, r = make_workload("batch", n=8, nv=16)
    f = make_fields(cfg, r)
    it = iris(cfg.with_(coef_grid=1))
    with pytest.raises(IrisSOError) as e:
        it.observe_adjoint(*dev_fields(f), torch.ones((cfg.ny, cfg.nx, cfg.nv), dtype=torch.float32, device="cuda"))
    assert e.value.status == 2
    for bad in (dict(grid_n_density=1), dict(grid_nH2_lo=0.0), dict(grid_T_hi=1.0), dict(coef_grid=2), dict(grid_n_temp=5000)):
        with pytest.raises(IrisSOError) as e:
            iris(cfg.with_(coef_grid=1).with_(**bad))
        assert e.value.status == 1
