"""Pins for the oracle's coefficient grid (section 4.2: grid precomputation with grid gradients;
section 4.3: runtime lookup by linear interpolation, linear behaviour outside the grid bounds).  Reading S31 of
DESIGN.md: two axes (n_H2, T_gas), geometric node spacing, multilinear in the variables themselves.

None of these retypes the lookup: they check it against what interpolation must satisfy (nodes reproduced, multilinear
functions reproduced exactly inside AND outside the grid, slope outside = edge finite difference, continuity across
cell faces, second-order convergence to the exact per-cell solve)."""
import numpy as np
import pytest

from iris_inputs import make_fields, make_workload
from oracle import Oracle


def grid_cfg(nn=24, nT=12, **kw):
    cfg, r = make_workload("tiny", n=4, nv=32)
    cfg = cfg.with_(coef_grid=1, grid_n_density=nn, grid_n_temp=nT, grid_nH2_lo=1.0, grid_nH2_hi=1.0e6, grid_T_lo=10.0,
                    grid_T_hi=300.0, **kw)
    return cfg, r


def test_nodes_are_geometric_and_hit_the_end_points():
    cfg, _ = grid_cfg()
    n, T = Oracle(cfg).grid_nodes()
    assert n[0] == pytest.approx(1.0, rel=1e-14, abs=0.0) and n[-1] == pytest.approx(1.0e6, rel=1e-13, abs=0.0)
    assert T[0] == pytest.approx(10.0, rel=1e-14, abs=0.0) and T[-1] == pytest.approx(300.0, rel=1e-13, abs=0.0)
    assert np.allclose(n[1:] / n[:-1], (1e6) ** (1 / 23), rtol=1e-12, atol=0.0)
    assert np.allclose(T[1:] / T[:-1], 30.0 ** (1 / 11), rtol=1e-12, atol=0.0)


def test_grid_holds_the_per_abundance_coefficients_of_the_exact_solve():
    """Eq. 4.2.1: j = chi j~, alpha = chi alpha~ with the level balance of Eq. 3.6.1 solved at the node."""
    cfg, _ = grid_cfg()
    o = Oracle(cfg)
    g = o.grid_build()
    n, T = o.grid_nodes()
    ex = Oracle(cfg.with_(coef_grid=0))
    for i, j in ((0, 0), (7, 3), (23, 11), (12, 0), (0, 11)):
        c = ex.coefficients(np.float64([n[i]]).astype(np.float32), np.float64([T[j]]).astype(np.float32), np.float32([20.0]))
        # (the exact solve sees float32 inputs; the node values are doubles: compare at the float32 node)
        nf, Tf = float(np.float32(n[i])), float(np.float32(T[j]))
        x = ex.levelpop_cell(nf, Tf)
        assert c[0, 0] > 0 and c[1, 0] > 0
        xg = ex.levelpop_cell(n[i], T[j])
        # j~ = (h nu / 4 pi) n x_u A: ratio of grid value to the exact coefficient = (n x_u)_node / (n x_u)_float32 / X
        ratio = (n[i] * xg[cfg.line_upper]) / (nf * x[cfg.line_upper]) / cfg.abundance
        assert g[0, j, i] / c[0, 0] == pytest.approx(ratio, rel=1e-12, abs=0.0)


def test_lookup_reproduces_nodes_and_multilinear_functions_everywhere():
    cfg, _ = grid_cfg()
    o = Oracle(cfg)
    n, T = o.grid_nodes()
    a, b, c, d = 3.0, -2.0e-6, 0.04, 7.0e-9
    f = lambda nn, TT: a + b * nn + c * TT + d * nn * TT                 # multilinear in (n, T)
    plane = f(n[None, :], T[:, None])
    rng = np.random.default_rng(5)
    # nodes
    for i, j in ((0, 0), (5, 2), (23, 11), (22, 11), (23, 0)):
        assert o.grid_lookup_plane(plane, n[i], T[j]) == pytest.approx(plane[j, i], rel=1e-12, abs=0.0)
    # inside, and OUTSIDE the bounds on every side (linear extrapolation of a multilinear function is the function)
    for nn, TT in list(zip(10 ** rng.uniform(0, 6, 40), 10 ** rng.uniform(1, np.log10(300), 40))) + \
            [(0.2, 50.0), (5e6, 50.0), (3e3, 4.0), (3e3, 900.0), (0.3, 3.0), (4e7, 2000.0), (0.0, 20.0)]:
        assert o.grid_lookup_plane(plane, nn, TT) == pytest.approx(f(nn, TT), rel=1e-10, abs=0.0)


def test_extrapolation_continues_the_edge_cell_and_interpolation_is_continuous():
    cfg, _ = grid_cfg()
    o = Oracle(cfg)
    n, T = o.grid_nodes()
    rng = np.random.default_rng(9)
    plane = rng.uniform(1.0, 2.0, (T.size, n.size))                     # no structure at all
    Tm = T[4]                                                           # on a node row: a function of n alone
    # below the first node the slope is the finite difference of the first cell, above the last node that of the last
    lo = (o.grid_lookup_plane(plane, 0.5 * n[0], Tm) - o.grid_lookup_plane(plane, 0.25 * n[0], Tm)) / (0.25 * n[0])
    assert lo == pytest.approx((plane[4, 1] - plane[4, 0]) / (n[1] - n[0]), rel=1e-9, abs=0.0)
    hi = (o.grid_lookup_plane(plane, 3.0 * n[-1], Tm) - o.grid_lookup_plane(plane, 2.0 * n[-1], Tm)) / n[-1]
    assert hi == pytest.approx((plane[4, -1] - plane[4, -2]) / (n[-1] - n[-2]), rel=1e-9, abs=0.0)
    nm = n[9]
    up = (o.grid_lookup_plane(plane, nm, 2.0 * T[-1]) - o.grid_lookup_plane(plane, nm, 1.5 * T[-1])) / (0.5 * T[-1])
    assert up == pytest.approx((plane[-1, 9] - plane[-2, 9]) / (T[-1] - T[-2]), rel=1e-9, abs=0.0)
    # continuity across cell faces (a node-nearest or a one-sided Taylor scheme would jump here)
    for i in (1, 7, 22):
        eps = 1e-9 * n[i]
        Tq = 0.37 * T[5] + 0.63 * T[6]
        left, right = o.grid_lookup_plane(plane, n[i] - eps, Tq), o.grid_lookup_plane(plane, n[i] + eps, Tq)
        assert abs(left - right) < 1e-7
    # inside a cell the value is the bilinear blend of its four corners (midpoint = their mean)
    mid = o.grid_lookup_plane(plane, 0.5 * (n[3] + n[4]), 0.5 * (T[6] + T[7]))
    assert mid == pytest.approx(plane[6:8, 3:5].mean(), rel=1e-12, abs=0.0)


def test_grid_coefficients_converge_to_the_exact_solve_at_second_order():
    errs = []
    cfg0, r = grid_cfg()
    f = make_fields(cfg0, r)
    for nn, nT in ((16, 8), (32, 16), (64, 32), (128, 64)):
        cfg = cfg0.with_(grid_n_density=nn + 1, grid_n_temp=nT + 1)
        cg = Oracle(cfg).coefficients(f["nH2"], f["Tgas"], f["Tdust"])
        ce = Oracle(cfg.with_(coef_grid=0)).coefficients(f["nH2"], f["Tgas"], f["Tdust"])
        assert np.array_equal(cg[2:], ce[2:])                          # Doppler width and dust are not gridded
        errs.append(max(np.abs(cg[0] / ce[0] - 1).max(), np.abs(cg[1] / ce[1] - 1).max()))
    ratios = np.array(errs[:-1]) / np.array(errs[1:])
    assert errs[-1] < 2e-3 and np.all(ratios > 3.0) and np.all(ratios < 5.0)


def test_abundance_is_applied_after_the_lookup_and_T_inf_masks():
    cfg, r = grid_cfg()
    f = make_fields(cfg, r)
    c1 = Oracle(cfg).coefficients(f["nH2"], f["Tgas"], f["Tdust"])
    c2 = Oracle(cfg.with_(abundance=3.0 * cfg.abundance)).coefficients(f["nH2"], f["Tgas"], f["Tdust"])
    assert np.allclose(c2[:2], 3.0 * c1[:2], rtol=1e-13, atol=0.0) and np.array_equal(c2[2:], c1[2:])
    c3 = Oracle(cfg.with_(T_inf=80.0)).coefficients(f["nH2"], f["Tgas"], f["Tdust"])
    hot = f["Tgas"].ravel() > 80.0
    assert hot.any() and (~hot).any()
    assert np.all(c3[:2, hot] == 0.0) and np.array_equal(c3[:2, ~hot], c1[:2, ~hot])
