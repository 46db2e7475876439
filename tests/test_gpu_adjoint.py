"""GPU parity of the gradient path (K8 + K9, BASELINE config 5): iris_so_observe_adjoint against the oracle's
float64 finite differences of L = sum(w * cube) (noise-free, beam applied), and against the oracle's analytic
float64 adjoint (itself pinned to finite differences in tests/test_oracle_pins.py) on every cell.

Tolerance (north_star): relative error <= 1e-3.  A cell's gradient is a sum over channels of terms of both
signs, so "relative" is taken per cell against |g| plus a floor of 1e-4 of the largest |g| in the cube
(DESIGN.md section 6)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from iris_inputs import make_fields, make_workload, weight_cube
from oracle import Oracle

pytestmark = pytest.mark.gpu

REL, FLOOR = 1.0e-3, 1.0e-4


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def gpu_grad(cfg, f, w):
    from paper_2607_01338_b200 import IrisSO
    g = IrisSO(cfg).observe_adjoint(*[dev(f[k]) for k in ("nH2", "Tgas", "Tdust", "vlos")], dev(w.astype(np.float32)))
    return g.cpu().numpy().astype(np.float64)


def excess(g, ref, scale):
    """max over cells of |g - ref| / (REL * |ref| + REL * FLOOR * scale); <= 1 passes."""
    return float(np.max(np.abs(g - ref) / (REL * np.abs(ref) + REL * FLOOR * scale)))


def check(cfg, f, w, n_fd=48, seed=5, label="", fd_random=True, eps=1e-5):
    o = Oracle(cfg)
    what = o.beam(w.astype(np.float64)) if cfg.beam_fwhm_px > 0 else w.astype(np.float64)
    ref = o.grad_adjoint(f, what)
    g = gpu_grad(cfg, f, w).reshape(ref.shape)
    assert np.all(np.isfinite(g))
    scale = np.abs(ref).max()
    assert scale > 0
    worst = excess(g, ref, scale)
    # finite differences on a seeded sample of cells, biased to cells that matter
    rng = np.random.default_rng(seed)
    order = np.argsort(-np.abs(ref).ravel())
    rand = rng.choice(cfg.n_cells, size=n_fd // 2, replace=False) if fd_random else order[n_fd // 2: n_fd]
    cells = np.unique(np.concatenate([order[: n_fd // 2], rand]))
    gfd = o.grad_fd(f, what, cells, eps=eps)
    worst_fd = excess(g.ravel()[cells], gfd, scale)
    print("adjoint %s: worst vs analytic %.3g, vs finite differences %.3g of tolerance (max|g| %.3g)" %
          (label, worst, worst_fd, scale))
    assert worst <= 1.0 and worst_fd <= 1.0
    return g


def test_adjoint_tiny_no_dust():
    cfg, r = make_workload("tiny", n=16, nv=64)
    f = make_fields(cfg, r)
    f["vlos"] = (0.15 * f["vlos"]).astype(np.float32)
    check(cfg, f, weight_cube(cfg), label="tiny")


@pytest.mark.parametrize("case", ["dust_beam", "thick", "intensity_out", "no_subtraction", "heavy_dust", "opaque_cells", "five_levels",
                                  "dense_collisions"])
def test_adjoint_regimes(case):
    kw = dict(n=20, nv=96)
    if case == "five_levels":
        kw["n_levels"] = 5
    cfg, r = make_workload("batch", **kw)
    f = make_fields(cfg, r)
    f["vlos"] = (0.2 * f["vlos"]).astype(np.float32)
    if case == "thick":
        cfg = cfg.with_(abundance=2e-5)
    elif case == "intensity_out":
        cfg = cfg.with_(out_unit=0)
    elif case == "no_subtraction":
        cfg = cfg.with_(subtract_continuum=False)
    elif case == "heavy_dust":
        cfg = cfg.with_(kappa_gas_cm2_g=5.0)
    elif case == "opaque_cells":          # single cells with tau_d ~ 100 (exp(tau_d) alone leaves the fp32 range)
        cfg = cfg.with_(kappa_gas_cm2_g=3.0)
        f["nH2"][: cfg.nz // 2] *= 1e-3
        f["nH2"][cfg.nz // 2:] *= 30.0
    elif case == "dense_collisions":      # every dJ collides: the dense (not the banded) state elimination
        Kd = np.array(cfg.coll_down_ref, dtype=np.float64, copy=True)
        for u in range(1, cfg.n_levels):
            for l in range(u):
                Kd[u, l] = 1e-11 / (u - l)
        cfg = cfg.with_(coll_down_ref=Kd)
    # opaque_cells: the relative step of the finite difference is below the double rounding of the objective in the
    # cells whose density was divided by 1000, so only the cells that carry the gradient are differenced there
    check(cfg, f, weight_cube(cfg), label=case, fd_random=case != "opaque_cells")


def test_adjoint_ragged_and_degenerate_shapes():
    cfg, r = make_workload("batch", n=8, nx=5, ny=3, nz=37, nv=45)
    f = make_fields(cfg, r)
    f["vlos"] = (0.1 * f["vlos"]).astype(np.float32)
    check(cfg, f, weight_cube(cfg), n_fd=20, label="ragged")
    cfg1, r1 = make_workload("batch", n=1, nx=1, ny=1, nz=1, nv=1)
    cfg1 = cfg1.with_(dv_cms=4.0e5, v0_cms=0.0, beam_fwhm_px=0.0)
    f1 = make_fields(cfg1, r1)
    f1["vlos"] = np.zeros_like(f1["vlos"])
    check(cfg1, f1, np.ones((1, 1, 1), np.float32), n_fd=2, label="1x1x1")


def test_adjoint_is_linear_in_w_and_zero_without_weights():
    cfg, r = make_workload("batch", n=12, nv=64)
    f = make_fields(cfg, r)
    f["vlos"] = (0.15 * f["vlos"]).astype(np.float32)
    w1 = weight_cube(cfg, seed=2000); w2 = weight_cube(cfg, seed=2001)
    g1, g2, g12 = gpu_grad(cfg, f, w1), gpu_grad(cfg, f, w2), gpu_grad(cfg, f, w1 + 2 * w2)
    s = np.abs(g12).max()
    assert np.max(np.abs(g12 - (g1 + 2 * g2))) <= 2e-5 * s
    assert np.all(gpu_grad(cfg, f, np.zeros_like(w1)) == 0.0)


def test_batch_workload_cubes_and_gradient():
    """BASELINE config 5 at reduced size: independent seeded cubes, each rendered with dust, beam and noise,
    plus the gradient for the seeded weight cube."""
    from paper_2607_01338_b200 import IrisSO
    from parity import assert_spectra
    for i in range(3):
        cfg, r = make_workload("batch", n=24, nv=128, seed=1000 + i)
        f = make_fields(cfg, r)
        d = [dev(f[k]) for k in ("nH2", "Tgas", "Tdust", "vlos")]
        cube = IrisSO(cfg).observe(*d).cpu().numpy()
        ref = Oracle(cfg).observe(f)
        clean = Oracle(cfg).observe(f, noise=False)
        assert_spectra(cube, ref, extra=8e-6 * cfg.noise_sigma, peak_of=clean, what="batch cube %d" % i)
        check(cfg, f, weight_cube(cfg), n_fd=24, label="batch cube %d (v_edge %.0f, sigma_t %.1f km/s)" %
              (i, f["meta"]["v_edge_kms"], f["meta"]["sigma_t_kms"]))


@pytest.mark.parametrize("case", ["dust_beam", "thick", "no_dust"])
def test_abundance_gradient(case):
    """iris_so_observe_adjoint_abundance: dL / d ln X per cell against the oracle's analytic adjoint (every cell) and its
    finite differences (sampled cells)."""
    from paper_2607_01338_b200 import IrisSO
    if case == "no_dust":
        cfg, r = make_workload("tiny", n=16, nv=64)
    else:
        cfg, r = make_workload("batch", n=20, nv=96)
    f = make_fields(cfg, r)
    f["vlos"] = (0.2 * f["vlos"]).astype(np.float32)
    if case == "thick":
        cfg = cfg.with_(abundance=2e-5)
    w = weight_cube(cfg)
    o = Oracle(cfg)
    what = o.beam(w.astype(np.float64)) if cfg.beam_fwhm_px > 0 else w.astype(np.float64)
    ref = o.grad_adjoint(f, what, wrt="abundance")
    g = IrisSO(cfg).observe_adjoint(*[dev(f[k]) for k in ("nH2", "Tgas", "Tdust", "vlos")], dev(w.astype(np.float32)),
                                    wrt="abundance").cpu().numpy().astype(np.float64).reshape(ref.shape)
    # d / d ln X is (emission term) - (absorption term), both carried in fp32: where a line is saturated they cancel, so
    # the floor is 3e-7 of the largest gradient instead of the 1e-7 of the density gradient (tolerances)
    scale = 3.0 * np.abs(ref).max()
    assert scale > 0 and np.all(np.isfinite(g))
    worst = excess(g, ref, scale)
    cells = np.argsort(-np.abs(ref).ravel())[:24]
    worst_fd = excess(g.ravel()[cells], o.grad_fd(f, what, cells, eps=1e-5, wrt="abundance"), scale)
    print("abundance gradient %s: worst vs analytic %.3g, vs finite differences %.3g of tolerance" % (case, worst, worst_fd))
    assert worst <= 1.0 and worst_fd <= 1.0


def test_adjoint_with_tabulated_rates():
    """The density derivative of the level balance with tabulated multi-partner rates (K9 TABLE variant)."""
    rng = np.random.default_rng(2)
    cfg, r = make_workload("batch", n=16, nv=64)
    grid = np.array([10.0, 30.0, 60.0, 100.0, 200.0, 500.0])
    N = cfg.n_levels
    tab = np.zeros((2, grid.size, N, N))
    for p in range(2):
        for u in range(1, N):
            for l in range(max(0, u - 2), u):
                tab[p, :, u, l] = rng.uniform(0.5, 2.0) * 1e-11 * (grid / 100.0) ** rng.uniform(0.0, 0.5) / (u - l)
    cfg = cfg.with_(coll_T_grid=grid, coll_table=tab, coll_partner_frac=np.array([0.8, 0.2]))
    f = make_fields(cfg, r)
    f["vlos"] = (0.2 * f["vlos"]).astype(np.float32)
    check(cfg, f, weight_cube(cfg), n_fd=32, label="tabulated rates")


def test_batch_workload_full_size_sampled():
    """BASELINE config 5 at full size (one of the 64 cubes: 128^3 cells, 256 channels, dust, beam 3 px, noise 0.25 K), in
    the launch configuration bench.py times: seeded pixel columns of the raw cube against the oracle, the beam on a patch,
    and the reverse-scan gradient against the oracle's finite differences on sampled cells (relative error <= 1e-3)."""
    from paper_2607_01338_b200 import IrisSO
    from parity import assert_spectra
    cfg, r = make_workload("batch", seed=1003)
    f = make_fields(cfg, r)
    d = [dev(f[k]) for k in ("nH2", "Tgas", "Tdust", "vlos")]
    it = IrisSO(cfg)
    raw = it.observe(*d, beam=False, noise=False)
    plane, n_cols = cfg.nx * cfg.ny, 32
    rng = np.random.default_rng(77)
    pix = np.sort(rng.choice(plane, size=n_cols, replace=False))
    got = raw.reshape(plane, cfg.nv)[torch.from_numpy(pix).cuda()].cpu().numpy()
    sub = {k: np.ascontiguousarray(f[k].reshape(cfg.nz, plane)[:, pix]).reshape(cfg.nz, 1, n_cols)
           for k in ("nH2", "Tgas", "Tdust", "vlos")}
    cfg_s = cfg.with_(nx=n_cols, ny=1, beam_fwhm_px=0.0, noise_sigma=0.0)
    ref = Oracle(cfg_s).observe(sub, beam=False, noise=False).reshape(n_cols, cfg.nv)
    assert_spectra(got, ref, what="batch cube, sampled columns")
    o = Oracle(cfg)
    smooth = it.observe(*d, beam=True, noise=False)
    y0, x0, wd = 60, 21, 16
    patch = raw[y0 - 6:y0 + wd + 6, x0 - 6:x0 + wd + 6].cpu().numpy()
    assert np.abs(smooth[y0:y0 + wd, x0:x0 + wd].cpu().numpy() - o.beam(patch)[6:-6, 6:-6]).max() <= 1e-5 * np.abs(patch).max() + 1e-6
    full = it.observe(*d)
    dz = (full - smooth).flatten()[::53].cpu().numpy()
    assert abs(dz.std() - cfg.noise_sigma) < 2e-3 and abs(dz.mean()) < 2e-3
    # gradient of L = sum(w * cube): finite differences of the oracle on sampled cells (biased to the cells that matter)
    w = weight_cube(cfg)
    g = it.observe_adjoint(*d, dev(w)).cpu().numpy().astype(np.float64).ravel()
    what = o.beam(w.astype(np.float64))
    order = np.argsort(-np.abs(g))
    cells = np.unique(np.concatenate([order[:16], rng.choice(cfg.n_cells, size=16, replace=False)]))
    gfd = o.grad_fd(f, what, cells, eps=1e-5)
    worst = excess(g[cells], gfd, np.abs(g).max())
    print("batch cube at full size: gradient vs finite differences at %.3g of tolerance (max|g| %.3g)" % (worst, np.abs(g).max()))
    assert np.all(np.isfinite(g)) and worst <= 1.0


# ------------------------------------------------------------------------------------------------
# Gradient outside the hot-path mode (adjoint_modes_kernel): optically thick transfer with the smooth integrator (TR + BDF2 +
# ReLU) and / or the fine velocity grid with Simpson's rule -- thick + smooth + f = 1 is the paper's production mode
# (PAPER.md:563).  Same bar as above: every cell against the oracle's float64 reverse-mode adjoint of that mode, sampled
# cells against the oracle's finite differences through that mode's forward march.
MODE_ADJ = {"thick_smooth": (1, 0), "thick_smooth_sub1": (1, 1), "thick_smooth_sub3": (1, 3), "thick_formal_sub1": (0, 1),
            "thick_formal_sub3": (0, 3)}


@pytest.mark.parametrize("case", ["dust_beam", "thick", "intensity_out", "no_subtraction", "heavy_dust", "no_dust", "relu_active"])
@pytest.mark.parametrize("mode", MODE_ADJ)
def test_adjoint_of_the_thick_modes(mode, case):
    integ, sub = MODE_ADJ[mode]
    cfg, r = make_workload("batch", n=16, nv=64)
    cfg = cfg.with_(integration=integ, subsample=sub)
    f = make_fields(cfg, r)
    f["vlos"] = (0.2 * f["vlos"]).astype(np.float32)
    eps = 1e-5
    if case == "thick":
        cfg = cfg.with_(abundance=2e-5)
    elif case == "intensity_out":
        cfg = cfg.with_(out_unit=0)
    elif case == "no_subtraction":
        cfg = cfg.with_(subtract_continuum=False)
    elif case == "heavy_dust":
        cfg = cfg.with_(kappa_gas_cm2_g=5.0)
    elif case == "no_dust":
        cfg = cfg.with_(dust_on=False)
    elif case == "relu_active":
        if integ == 0:
            pytest.skip("the formal thick step has no ReLU")
        # bright background behind cold dust that turns opaque abruptly: continuum and line points are clamped at zero for
        # a few cells (tests/test_oracle_modes.py checks that they are).  The objective is ~1e7 times a cell's share of
        # it there, so the finite differences take a wider bracket.
        cfg = cfg.with_(T_cmb=60.0, kappa_gas_cm2_g=3.0)
        f["Tdust"] = np.full_like(f["Tdust"], 3.0)
        f["nH2"][: cfg.nz // 2] *= 1e-3
        f["nH2"][cfg.nz // 2:] *= 30.0
        eps = 1e-3
    check(cfg, f, weight_cube(cfg), n_fd=32, label="%s %s" % (mode, case), fd_random=case != "relu_active", eps=eps)


@pytest.mark.parametrize("mode", ["thick_smooth_sub1", "thick_formal_sub3", "thick_smooth"])
def test_adjoint_of_the_thick_modes_ragged_and_degenerate(mode):
    integ, sub = MODE_ADJ[mode]
    cfg, r = make_workload("batch", n=8, nx=5, ny=3, nz=37, nv=45)
    cfg = cfg.with_(integration=integ, subsample=sub)
    f = make_fields(cfg, r)
    f["vlos"] = (0.1 * f["vlos"]).astype(np.float32)
    check(cfg, f, weight_cube(cfg), n_fd=20, label=mode + " ragged")
    # more points than one block of 256 per pixel, a last block of every size class
    cfg2, r2 = make_workload("batch", n=6, nx=3, ny=2, nz=12, nv=200)
    cfg2 = cfg2.with_(integration=integ, subsample=sub, dv_cms=0.3 * cfg2.dv_cms, v0_cms=0.3 * cfg2.v0_cms)
    f2 = make_fields(cfg2, r2)
    f2["vlos"] = (0.3 * f2["vlos"]).astype(np.float32)
    check(cfg2, f2, weight_cube(cfg2), n_fd=20, label=mode + " several blocks")
    for nz in (1, 2, 3):
        cfg1, r1 = make_workload("batch", n=1, nx=1, ny=1, nz=nz, nv=3)
        cfg1 = cfg1.with_(integration=integ, subsample=sub, dv_cms=1.0e5, v0_cms=-1.0e5, beam_fwhm_px=0.0)
        f1 = make_fields(cfg1, r1)
        f1["vlos"] = np.zeros_like(f1["vlos"])
        o = Oracle(cfg1)
        ref = o.grad_adjoint(f1, np.ones((1, 1, 3)))
        g = gpu_grad(cfg1, f1, np.ones((1, 1, 3), np.float32)).reshape(ref.shape)
        assert excess(g, ref, max(np.abs(ref).max(), 1e-300)) <= 1.0, (mode, nz, g, ref)


def test_adjoint_of_the_thick_modes_abundance_and_linearity():
    cfg, r = make_workload("batch", n=12, nv=64)
    cfg = cfg.with_(integration=1, subsample=1)
    f = make_fields(cfg, r)
    f["vlos"] = (0.15 * f["vlos"]).astype(np.float32)
    from paper_2607_01338_b200 import IrisSO
    d = [dev(f[k]) for k in ("nH2", "Tgas", "Tdust", "vlos")]
    w1 = weight_cube(cfg, seed=2000); w2 = weight_cube(cfg, seed=2001)
    g1, g2, g12 = gpu_grad(cfg, f, w1), gpu_grad(cfg, f, w2), gpu_grad(cfg, f, w1 + 2 * w2)
    assert np.max(np.abs(g12 - (g1 + 2 * g2))) <= 2e-5 * np.abs(g12).max()
    assert np.all(gpu_grad(cfg, f, np.zeros_like(w1)) == 0.0)
    o = Oracle(cfg)
    what = o.beam(w1.astype(np.float64))
    ref = o.grad_adjoint(f, what, wrt="abundance")
    g = IrisSO(cfg).observe_adjoint(*d, dev(w1.astype(np.float32)), wrt="abundance").cpu().numpy().astype(np.float64).reshape(ref.shape)
    scale = np.abs(ref).max()
    assert np.max(np.abs(g - ref) / (REL * np.abs(ref) + 3e-7 * scale)) <= 1.0


def test_production_mode_gradient_at_full_size_sampled():
    """One cube of BASELINE config 5 (128^3 cells, 256 channels, dust, beam 3 px) in the paper's production mode (thick,
    smooth, f = 1: 513 fine points per spectrum): the gradient against the oracle's finite differences on sampled cells."""
    from paper_2607_01338_b200 import IrisSO
    cfg, r = make_workload("batch", seed=1003)
    cfg = cfg.with_(integration=1, subsample=1)
    f = make_fields(cfg, r)
    d = [dev(f[k]) for k in ("nH2", "Tgas", "Tdust", "vlos")]
    it = IrisSO(cfg)
    w = weight_cube(cfg)
    wd = dev(w)
    g = it.observe_adjoint(*d, wd)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(3):
        it.observe_adjoint(*d, wd)
    e1.record()
    torch.cuda.synchronize()
    g = g.cpu().numpy().astype(np.float64).ravel()
    o = Oracle(cfg)
    what = o.beam(w.astype(np.float64))
    rng = np.random.default_rng(78)
    order = np.argsort(-np.abs(g))
    cells = np.unique(np.concatenate([order[:16], rng.choice(cfg.n_cells, size=16, replace=False)]))
    gfd = o.grad_fd(f, what, cells, eps=1e-5)
    worst = excess(g[cells], gfd, np.abs(g).max())
    print("production mode, 128^3 x 256 ch: gradient vs finite differences at %.3g of tolerance (max|g| %.3g), %.2f ms per call" %
          (worst, np.abs(g).max(), e0.elapsed_time(e1) / 3))
    assert np.all(np.isfinite(g)) and worst <= 1.0


def test_production_mode_gradient_of_the_medium_cube_sampled():
    """BASELINE config "medium" (256 x 256 x 288 cells, 512 channels; no dust, no beam) in the production mode: 1025 fine
    points per spectrum, several blocks of points per pixel, 288-cell columns.  Sampled cells against the oracle's finite
    differences through that mode's forward march."""
    from paper_2607_01338_b200 import IrisSO
    cfg, r = make_workload("medium")
    cfg = cfg.with_(integration=1, subsample=1)
    f = make_fields(cfg, r)
    d = [dev(f[k]) for k in ("nH2", "Tgas", "Tdust", "vlos")]
    it = IrisSO(cfg)
    w = weight_cube(cfg)
    wd = dev(w)
    g = it.observe_adjoint(*d, wd)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    it.observe_adjoint(*d, wd)
    e1.record()
    torch.cuda.synchronize()
    g = g.cpu().numpy().astype(np.float64).ravel()
    o = Oracle(cfg)
    what = o.beam(w.astype(np.float64)) if cfg.beam_fwhm_px > 0 else w.astype(np.float64)
    rng = np.random.default_rng(79)
    order = np.argsort(-np.abs(g))
    cells = np.unique(np.concatenate([order[:12], rng.choice(cfg.n_cells, size=12, replace=False)]))
    gfd = o.grad_fd(f, what, cells, eps=1e-5)
    worst = excess(g[cells], gfd, np.abs(g).max())
    print("production mode, medium cube: gradient vs finite differences at %.3g of tolerance (max|g| %.3g), %.1f ms per call" %
          (worst, np.abs(g).max(), e0.elapsed_time(e1)))
    assert np.all(np.isfinite(g)) and worst <= 1.0
