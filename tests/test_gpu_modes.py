"""GPU parity of the paper's other transfer / integration modes (transfer_modes_kernel, through the C ABI) against
the float64 oracle on the same seeded inputs: optically thin / selectively thin / thick, formal / smooth, and the
fine velocity grid with Simpson's rule.  Tolerances: tests/parity.py."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from iris_inputs import make_fields, make_workload
from iris_inputs.fields import KMS
from oracle import Oracle
from parity import assert_spectra, selthin_source_allowance, krj

pytestmark = pytest.mark.gpu

# (transfer_mode, integration, subsample).  The formal modes (thin and selectively thin with the channel-integrated
# profile, thick on the fine grid) run through the line-window series kernel by default and the thick and selectively
# thin smooth modes through the line-window smooth kernel; the "_dense" entries force transfer_modes_kernel (transfer_algo = 1).
MODES = {"thin_formal": (2, 0, 0), "thin_smooth": (2, 1, 0), "selthin_formal": (1, 0, 0), "selthin_smooth": (1, 1, 0),
         "thick_smooth": (0, 1, 0), "thick_formal_sub1": (0, 0, 1), "thick_formal_sub3": (0, 0, 3),
         "thick_smooth_sub1": (0, 1, 1), "thick_smooth_sub7": (0, 1, 7),
         "thin_formal_dense": (2, 0, 0), "selthin_formal_dense": (1, 0, 0),
         "thick_formal_sub1_dense": (0, 0, 1), "thick_formal_sub3_dense": (0, 0, 3),
         "thick_smooth_dense": (0, 1, 0), "thick_smooth_sub1_dense": (0, 1, 1), "thin_smooth_dense": (2, 1, 0),
         "selthin_smooth_dense": (1, 1, 0)}


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def dev_fields(f):
    return [dev(f[k]) for k in ("nH2", "Tgas", "Tdust", "vlos")]


def with_mode(cfg, name):
    m, i, s = MODES[name]
    cfg = cfg.with_(transfer_mode=m, integration=i, subsample=s, name=name)
    return cfg


def expected_kernel(cfg, dense):
    """What iris_so_transfer_kernel should name for a configuration."""
    m, i, s = cfg.transfer_mode, cfg.integration, cfg.subsample
    narrow = cfg.microturb_cms > 0 and cfg.dv_cms <= 0.55 * cfg.microturb_cms
    if not dense:
        if i == 0 and ((s == 0 and m in (1, 2) and narrow) or (m == 0 and s > 0)):
            return "transfer_series_kernel"
        if i == 1 and m == 2 and narrow:                       # Simpson's rule along the ray: a weighted thin sum
            return "transfer_series_kernel"
        if i == 1 and m in (0, 1) and cfg.nz >= 2 and (s > 0 or narrow):
            return "transfer_smooth_window_kernel"
    return "transfer_modes_kernel"


def gpu_cube(cfg, f, expect_kernel=True, **kw):
    from paper_2607_01338_b200 import IrisSO
    dense = cfg.name.endswith("_dense")
    it = IrisSO(cfg, transfer_algo=1 if dense else 0)
    if expect_kernel:
        assert it.transfer_kernel() == expected_kernel(cfg, dense), cfg.name
    return it.observe(*dev_fields(f), **kw).cpu().numpy()


@pytest.mark.parametrize("mode", MODES)
def test_modes_small_dust(mode):
    cfg, r = make_workload("small", n=32, nv=96)
    cfg = with_mode(cfg, mode)
    f = make_fields(cfg, r)
    f["vlos"] = (0.3 * f["vlos"]).astype(np.float32)
    cube = gpu_cube(cfg, f)
    ref = Oracle(cfg).observe(f)
    worst = assert_spectra(cube, ref, what=mode)
    assert np.abs(ref).max() > 0.05
    print("%s: worst pixel at %.3g of tolerance, peak %.3g K" % (mode, worst, np.abs(ref).max()))


@pytest.mark.parametrize("mode", MODES)
def test_modes_tiny_no_dust_ragged(mode):
    """Dust off (tau_d = 0 everywhere), sizes that fill neither the 32-pixel nor the 8-channel tile, odd and even nz."""
    for nz in (19, 20):
        cfg, r = make_workload("tiny", nx=37, ny=3, nz=nz, nv=45)
        cfg = with_mode(cfg, mode).with_(v0_cms=-11.0 * KMS)
        f = make_fields(cfg, r)
        f["vlos"] = (0.1 * f["vlos"]).astype(np.float32)
        assert_spectra(gpu_cube(cfg, f), Oracle(cfg).observe(f), what="%s nz=%d" % (mode, nz))


@pytest.mark.parametrize("mode", MODES)
@pytest.mark.parametrize("shape", [dict(nx=1, ny=1, nz=1, nv=1), dict(nx=2, ny=1, nz=2, nv=3), dict(nx=3, ny=2, nz=3, nv=9)])
def test_modes_degenerate_shapes(mode, shape):
    cfg, r = make_workload("small", **shape)
    cfg = with_mode(cfg, mode).with_(v0_cms=-0.5 * (shape["nv"] - 1) * cfg.dv_cms)
    f = make_fields(cfg, r)
    f["vlos"] = (0.01 * f["vlos"]).astype(np.float32)
    assert_spectra(gpu_cube(cfg, f), Oracle(cfg).observe(f), what=mode)


@pytest.mark.parametrize("mode", ["selthin_formal", "selthin_formal_dense", "thin_formal", "selthin_smooth", "thick_smooth",
                                  "thick_smooth_sub1", "thick_formal_sub1", "thick_formal_sub3_dense", "thick_smooth_dense",
                                  "thick_smooth_sub1_dense"])
@pytest.mark.parametrize("case", ["thick_line", "opaque_dust_clamp", "absorption"])
def test_modes_regimes(mode, case):
    """Large optical depths (A-stability of BDF2), the ReLU clamp, and lines in absorption."""
    cfg, r = make_workload("small", n=20, nv=96)
    cfg = with_mode(cfg, mode)
    f = make_fields(cfg, r)
    f["vlos"] = (0.25 * f["vlos"]).astype(np.float32)
    if case == "thick_line":
        cfg = cfg.with_(abundance=2e-4)
    elif case == "opaque_dust_clamp":
        # bright background, cold dust that turns opaque abruptly: the smooth continuum overshoots below zero and is clamped
        cfg = cfg.with_(T_cmb=60.0, kappa_gas_cm2_g=3.0)
        f["Tdust"] = np.full_like(f["Tdust"], 3.0)
        f["nH2"][: cfg.nz // 2] *= 1e-3
        f["nH2"][cfg.nz // 2:] *= 30.0
    else:
        cfg = cfg.with_(kappa_gas_cm2_g=1.0)
        f["Tdust"] = np.full_like(f["Tdust"], 150.0)
    o = Oracle(cfg)
    cfg_tot = cfg.with_(subtract_continuum=False)
    cube = gpu_cube(cfg, f)
    ref = o.observe(f)
    # a clamped spectrum is compared on the total intensity scale as well (the subtracted cube can be ~ -continuum)
    tot = gpu_cube(cfg_tot, f)
    ref_tot = Oracle(cfg_tot).observe(f)
    assert_spectra(tot, ref_tot, extra=3e-7 * np.abs(ref_tot).max(axis=-1, keepdims=True), what=mode + " total")
    assert_spectra(cube, ref, extra=3e-7 * np.abs(ref_tot).max(axis=-1, keepdims=True), what=mode + " subtracted")


@pytest.mark.parametrize("mode", ["thin_formal", "selthin_formal", "selthin_smooth", "thick_smooth_sub1", "thick_formal_sub1"])
def test_modes_transfer_intensities_and_output_units(mode):
    from paper_2607_01338_b200 import IrisSO
    cfg, r = make_workload("small", n=16, nv=64)
    cfg = with_mode(cfg, mode)
    f = make_fields(cfg, r)
    f["vlos"] = (0.2 * f["vlos"]).astype(np.float32)
    o = Oracle(cfg)
    It, Ic = IrisSO(cfg).transfer(*dev_fields(f))
    coef = o.coefficients(f["nH2"], f["Tgas"], f["Tdust"])
    rt, rc = o.march(coef, f["vlos"])
    K = krj(cfg.nu0_Hz)
    It, Ic = It.cpu().numpy().reshape(-1, cfg.nv).astype(np.float64), Ic.cpu().numpy().ravel().astype(np.float64)
    assert np.allclose(Ic, rc, rtol=3e-6)
    line = np.abs(rt - rc[:, None]).max(axis=1)
    err = np.abs(It - rt).max(axis=1)
    assert np.all(err <= 1e-4 * line + 1e-6 / K + 3e-7 * np.abs(rt).max(axis=1))
    # Planck-space subtraction through the same kernel
    cfg_p = cfg.with_(out_unit=2, subtract_space=1)
    assert_spectra(gpu_cube(cfg_p, f), Oracle(cfg_p).observe(f), rel=2.6e-4, floor=2.6e-6, what=mode + " planck")


def test_modes_kernel_selection_and_fallbacks():
    """Which kernel runs a mode (iris_so_transfer_kernel), and parity where the series kernel hands over to the dense
    modes kernel: channels wider than 0.55 xi (thin modes), fine grids that do not fit shared memory."""
    from paper_2607_01338_b200 import IrisSO
    cfg, r = make_workload("small", nx=6, ny=2, nz=12, nv=64)
    names = {}
    for mode in ("thin_formal", "selthin_formal", "thick_formal_sub1", "thick_formal_sub3", "thick_smooth", "thin_smooth",
                 "selthin_smooth"):
        names[mode] = IrisSO(with_mode(cfg, mode)).transfer_kernel()
    assert names == {"thin_formal": "transfer_series_kernel", "selthin_formal": "transfer_series_kernel",
                     "thick_formal_sub1": "transfer_series_kernel", "thick_formal_sub3": "transfer_series_kernel",
                     "thick_smooth": "transfer_smooth_window_kernel", "thin_smooth": "transfer_series_kernel",
                     "selthin_smooth": "transfer_smooth_window_kernel"}
    # wide channels: 1 km/s against xi = 1 km/s
    wide = cfg.with_(dv_cms=1.0 * KMS, v0_cms=-31.5 * KMS)
    f = make_fields(wide, r)
    f["vlos"] = (0.2 * f["vlos"]).astype(np.float32)
    for mode in ("thin_formal", "selthin_formal", "thin_smooth"):
        c = with_mode(wide, mode)
        assert IrisSO(c).transfer_kernel() == "transfer_modes_kernel"
        assert_spectra(gpu_cube(c, f), Oracle(c).observe(f), what=mode + " wide channels")
    c = with_mode(wide, "thick_formal_sub1")                      # the point profile has no such limit
    assert IrisSO(c).transfer_kernel() == "transfer_series_kernel"
    assert_spectra(gpu_cube(c, f), Oracle(c).observe(f), what="thick_formal_sub1 wide channels")
    # 4000 channels x 4 intervals = 16001 points per spectrum: beyond shared memory
    big = cfg.with_(nv=4000, dv_cms=0.05 * KMS, v0_cms=-0.5 * 3999 * 0.05 * KMS)
    fb = make_fields(big, r)
    fb["vlos"] = (0.2 * fb["vlos"]).astype(np.float32)
    c = with_mode(big, "thick_formal_sub3")
    assert IrisSO(c).transfer_kernel() == "transfer_modes_kernel"
    assert IrisSO(with_mode(big, "thick_formal_sub1")).transfer_kernel() == "transfer_series_kernel"
    for mode in ("thick_formal_sub3", "thick_formal_sub1"):
        c = with_mode(big, mode)
        assert_spectra(gpu_cube(c, fb, expect_kernel=False), Oracle(c).observe(fb), what=mode + " 4000 channels")


@pytest.mark.parametrize("mode", ["thick_smooth_sub1", "thick_smooth", "thick_formal_sub1", "thin_smooth", "selthin_smooth"])
def test_window_kernels_agree_with_the_dense_kernel_on_every_pixel_of_medium(mode):
    """The sampled-column tests above compare 24 columns of the medium cube with the oracle; here EVERY pixel of the cube
    from the line-window kernel of a mode is compared with the dense modes kernel (itself checked against the oracle),
    at half the parity tolerance."""
    from paper_2607_01338_b200 import IrisSO
    cfg, r = make_workload("medium")
    cfg = with_mode(cfg, mode)
    f = make_fields(cfg, r)
    d = dev_fields(f)
    it = IrisSO(cfg)
    assert it.transfer_kernel() != "transfer_modes_kernel"
    win = it.observe(*d, beam=False, noise=False)
    # the window march of the smooth integrator hands a pixel over where a few very dense cells in a row make the dust
    # opaque per cell (n_H2 is lognormal with sigma_ln = 2): a handful of the 65536 pixels
    assert it.smooth_fallback() <= (cfg.nx * cfg.ny) // 200
    dense = IrisSO(cfg, transfer_algo=1).observe(*d, beam=False, noise=False)
    peak = dense.abs().amax(dim=-1, keepdim=True)
    per_pixel = ((win - dense).abs() / (0.5e-4 * peak + 0.5e-6)).amax(dim=-1).reshape(-1)
    excess = per_pixel.max().item()
    print("%s: window against dense kernel on all %d pixels: worst at %.3g of half the tolerance" % (mode, cfg.nx * cfg.ny, excess))
    if mode != "selthin_smooth":
        assert excess <= 1.0
        return
    # selectively thin + smooth: two float32 evaluations of an unsaturated source differ by the rounding allowance of
    # parity.selthin_source_allowance, which only the oracle can bound: the 32 pixels where the two kernels disagree
    # most are marched by the oracle and BOTH kernels are held to it; elsewhere the two stay within 8 half-tolerances
    assert excess <= 8.0
    plane = cfg.nx * cfg.ny
    pix = np.sort(torch.topk(per_pixel, 32).indices.cpu().numpy())
    sub = {k: np.ascontiguousarray(f[k].reshape(cfg.nz, plane)[:, pix]).reshape(cfg.nz, 1, pix.size)
           for k in ("nH2", "Tgas", "Tdust", "vlos")}
    cfg_s = cfg.with_(nx=pix.size, ny=1, beam_fwhm_px=0.0, noise_sigma=0.0)
    ref = Oracle(cfg_s).observe(sub, beam=False, noise=False).reshape(pix.size, cfg.nv)
    extra = selthin_source_allowance(cfg_s, sub)
    sel = torch.from_numpy(pix).cuda()
    for what, cube in (("window kernel", win), ("dense kernel", dense)):
        worst = assert_spectra(cube.reshape(plane, cfg.nv)[sel].cpu().numpy(), ref, extra=extra,
                               what="selthin_smooth medium, %s on the 32 pixels of largest disagreement" % what)
        print("selthin_smooth %s against the oracle on those pixels: worst at %.3g of tolerance" % (what, worst))


def test_smooth_window_hands_over_when_a_relu_fires_outside_the_windows():
    """opaque_dust_clamp makes the smooth continuum overshoot below zero (the ReLU clamps every spectral point, also
    those no line window covers): the window kernel must notice, and the dense kernel, gated on its flag, must
    deliver the cube.  On the unmodified workload the flag stays down."""
    from paper_2607_01338_b200 import IrisSO
    cfg, r = make_workload("small", n=20, nv=96)
    for mode in ("thick_smooth", "thick_smooth_sub1"):
        c = with_mode(cfg, mode)
        f = make_fields(c, r)
        f["vlos"] = (0.25 * f["vlos"]).astype(np.float32)
        it = IrisSO(c)
        assert it.transfer_kernel() == "transfer_smooth_window_kernel"
        cube = it.observe(*dev_fields(f)).cpu().numpy()
        assert not it.smooth_fallback()
        assert_spectra(cube, Oracle(c).observe(f), what=mode)
        c2 = c.with_(T_cmb=60.0, kappa_gas_cm2_g=3.0)
        f["Tdust"] = np.full_like(f["Tdust"], 3.0)
        f["nH2"][: c.nz // 2] *= 1e-3
        f["nH2"][c.nz // 2:] *= 30.0
        it2 = IrisSO(c2)
        cube2 = it2.observe(*dev_fields(f)).cpu().numpy()
        assert it2.smooth_fallback() > 0
        ref2 = Oracle(c2).observe(f)
        ref_tot = Oracle(c2.with_(subtract_continuum=False)).observe(f)
        assert_spectra(cube2, ref2, extra=3e-7 * np.abs(ref_tot).max(axis=-1, keepdims=True), what=mode + " clamped")
        # every other mode reports 0
        assert not IrisSO(with_mode(cfg, "thin_smooth")).smooth_fallback()


@pytest.mark.parametrize("mode", ["thick_smooth", "thick_smooth_sub1", "thick_smooth_dense", "thick_smooth_sub1_dense"])
@pytest.mark.parametrize("tau_d", [0.05, 0.2, 0.3, 0.4, 0.45, 0.6])
def test_smooth_window_behind_sustained_moderate_dust(mode, tau_d):
    """A line 17 or more cells from the observer behind uniform dust of tau_d per cell (Eq. 4.8.10: the
    homogeneous BDF2 step has roots [2 +- sqrt(1 - 2 tau_d)] / (3 + 2 tau_d); the recessive solution dies as 3^-n only for
    tau_d << 1, and beyond tau_d = 0.5 the roots are complex).  The window kernel freezes a point 12 cells after the
    last line has touched it, which is exact only while the product of the root ratios over those cells is small: at
    tau_d >= 0.2 it must hand over to the dense kernel (flag up), at 0.05 it must not, and the cube must match the
    oracle either way.  The "_dense" twins are the control."""
    from paper_2607_01338_b200 import IrisSO
    n_far, n_near = 8, 16
    cfg, r = make_workload("small", nx=24, ny=6, nz=n_far + n_near, nv=96)
    cfg = with_mode(cfg, mode)
    f = make_fields(cfg, r)
    f["vlos"] = (0.25 * f["vlos"]).astype(np.float32)
    n_slab = 1.0e4
    cfg = cfg.with_(kappa_gas_cm2_g=tau_d / (cfg.mass_per_H2_g * n_slab * cfg.cell_cm))
    # the near slab: uniform density, no line inside the band (its velocity is far outside), dust of tau_d per cell
    f["nH2"][n_far:] = n_slab
    f["vlos"][n_far:] = 4.0e7
    f["Tdust"][n_far:] = 25.0
    dense = mode.endswith("_dense")
    it = IrisSO(cfg, transfer_algo=1 if dense else 0)
    assert it.transfer_kernel() == expected_kernel(cfg, dense)
    cube = it.observe(*dev_fields(f)).cpu().numpy()
    if not dense:
        # every pixel sees the slab: all of them are handed over from tau_d = 0.2 on, none at 0.05
        assert it.smooth_fallback() == (cfg.nx * cfg.ny if tau_d >= 0.2 else 0), "pixels handed over at tau_d = %g" % tau_d
    ref = Oracle(cfg).observe(f)
    assert np.abs(ref).max() > 30e-6                      # the attenuated line is still far above the 1e-6 K floor
    worst = assert_spectra(cube, ref, what="%s tau_d=%g" % (mode, tau_d))
    print("%s behind %d cells of tau_d = %g: worst pixel at %.3g of tolerance, peak %.3g K" % (mode, n_near, tau_d, worst, np.abs(ref).max()))


def test_modes_adjoint_is_refused_and_bad_modes_are_rejected():
    from paper_2607_01338_b200 import IrisSO, IrisSOError
    cfg, r = make_workload("batch", n=8, nv=16)
    f = make_fields(cfg, r)
    it = IrisSO(cfg.with_(transfer_mode=2))
    with pytest.raises(IrisSOError):
        it.observe_adjoint(*dev_fields(f), dev(np.ones((cfg.ny, cfg.nx, cfg.nv), np.float32)))
    for bad in (dict(transfer_mode=3), dict(integration=2), dict(subsample=2), dict(subsample=1, transfer_mode=1)):
        with pytest.raises(IrisSOError):
            IrisSO(cfg.with_(**bad))


@pytest.mark.parametrize("mode", ["thick_smooth_sub1", "thick_smooth_sub1_dense", "thick_smooth", "thick_formal_sub1",
                                  "selthin_formal", "thin_formal", "thin_smooth", "selthin_smooth", "selthin_smooth_dense"])
def test_modes_full_size_medium_sampled(mode):
    """BASELINE config "medium" at full size (256 x 256 x 288 cells, 512 channels), in the launch configuration
    bench.py times: seeded pixel columns against the oracle (columns are independent before the beam)."""
    from paper_2607_01338_b200 import IrisSO
    cfg, r = make_workload("medium")
    cfg = with_mode(cfg, mode)
    f = make_fields(cfg, r)
    it = IrisSO(cfg, transfer_algo=1 if mode.endswith("_dense") else 0)
    assert it.transfer_kernel() == expected_kernel(cfg, mode.endswith("_dense"))
    cube = it.observe(*dev_fields(f), beam=False, noise=False)
    assert it.smooth_fallback() <= (cfg.nx * cfg.ny) // 200      # pixels handed over to the dense kernel: a handful
    n_cols = 24
    plane = cfg.nx * cfg.ny
    pix = np.sort(np.random.default_rng(21).choice(plane, size=n_cols, replace=False))
    got = cube.reshape(plane, cfg.nv)[torch.from_numpy(pix).cuda()].cpu().numpy()
    sub = {k: np.ascontiguousarray(f[k].reshape(cfg.nz, plane)[:, pix]).reshape(cfg.nz, 1, n_cols)
           for k in ("nH2", "Tgas", "Tdust", "vlos")}
    cfg_s = cfg.with_(nx=n_cols, ny=1, beam_fwhm_px=0.0, noise_sigma=0.0)
    ref = Oracle(cfg_s).observe(sub, beam=False, noise=False).reshape(n_cols, cfg.nv)
    # (selectively thin + smooth: the unsaturated line source is rounded in float32, see selthin_source_allowance)
    extra = selthin_source_allowance(cfg_s, sub) if mode.startswith("selthin_smooth") else 0.0
    worst = assert_spectra(got, ref, extra=extra, what=mode + " medium, sampled columns")
    assert bool(torch.isfinite(cube).all())
    print("%s medium full size: worst sampled pixel at %.3g of tolerance" % (mode, worst))


# ------------------------------------------------------------------------------------------------
# diagnostics of section 5: density tracing and the TSRE / TAM metrics
@pytest.mark.parametrize("shape", [dict(n=24, nv=96), dict(nx=37, ny=5, nz=19, nv=45), dict(nx=1, ny=1, nz=1, nv=1)])
def test_density_trace_matches_oracle(shape):
    from paper_2607_01338_b200 import IrisSO
    cfg, r = make_workload("small", **shape)
    f = make_fields(cfg, r)
    f["vlos"] = (0.5 * f["vlos"]).astype(np.float32)
    got = IrisSO(cfg).density_trace(dev(f["nH2"]), dev(f["vlos"])).cpu().numpy().astype(np.float64)
    ref = Oracle(cfg).density_trace(f)
    # the channel of every cell is decided identically (both in double); the sums differ by fp32 accumulation only
    assert np.array_equal(got > 0, ref > 0)
    assert np.allclose(got, ref, rtol=2e-5, atol=0)


def test_metrics_match_oracle():
    from paper_2607_01338_b200 import IrisSO
    cfg, r = make_workload("small", n=24, nv=80)
    f = make_fields(cfg, r)
    f["vlos"] = (0.3 * f["vlos"]).astype(np.float32)
    it = IrisSO(cfg)
    d = dev_fields(f)
    T1 = it.observe(*d)
    T2 = IrisSO(cfg.with_(transfer_mode=1)).observe(*d)            # selectively thin against thick
    got = it.metrics(T1, T2)
    ref = Oracle(cfg).metrics(T1.cpu().numpy(), T2.cpu().numpy())
    assert ref["active1"] > 100 and ref["tsre_lbv"] > 0
    for k in ref:
        assert got[k] == pytest.approx(ref[k], rel=1e-9, abs=1e-12), k
    same = it.metrics(T1, T1)
    assert same["tsre_lbv"] == 0.0 and same["tsre_lv"] == 0.0 and same["tam1"] == same["tam2"]
