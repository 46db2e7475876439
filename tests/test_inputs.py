"""The seeded input recipe (SURVEY.md section 8(d) / BASELINE.json configs): shapes, statistics, determinism."""
import math

import numpy as np
import pytest

from iris_inputs import WORKLOADS, gaussian_random_field, make_fields, make_workload, weight_cube
from iris_inputs.fields import KMS, PC_CM


def test_grf_statistics_and_spectrum():
    g = gaussian_random_field((32, 32, 32), seed=4, stream=1)
    assert g.dtype == np.float32 and g.shape == (32, 32, 32) and g.flags.c_contiguous
    assert abs(float(g.mean())) < 1e-5 and float(g.std()) == pytest.approx(1.0, abs=1e-4)
    # power spectrum slope ~ -11/3: compare shell-averaged power at |k| ~ 2 and ~ 8 (x 4 in k)
    p = np.abs(np.fft.fftn(g.astype(np.float64))) ** 2
    k = np.sqrt(sum(np.meshgrid(*[np.fft.fftfreq(32) ** 2] * 3, indexing="ij"))) * 32
    p2 = p[(k > 1.5) & (k < 2.5)].mean()
    p8 = p[(k > 7.0) & (k < 9.0)].mean()
    assert math.log(p2 / p8) / math.log(4.0) == pytest.approx(11.0 / 3.0, abs=0.5)
    assert np.array_equal(g, gaussian_random_field((32, 32, 32), seed=4, stream=1))
    assert not np.array_equal(g, gaussian_random_field((32, 32, 32), seed=4, stream=2))


def test_tiny_workload_recipe():
    cfg, r = make_workload("tiny")
    assert (cfg.nx, cfg.ny, cfg.nz, cfg.nv, cfg.n_levels) == (32, 32, 32, 64, 5)
    assert cfg.cell_cm == pytest.approx(3 * PC_CM) and cfg.dv_cms == 0.5 * KMS and not cfg.dust_on
    assert cfg.nu0_Hz == pytest.approx(220.404e9, rel=1e-9) and (cfg.line_upper, cfg.line_lower) == (2, 1)
    assert cfg.abundance == 2e-6 and cfg.T_cmb == 2.725 and cfg.microturb_cms == 1e5
    f = make_fields(cfg, r)
    for k in ("nH2", "Tgas", "Tdust", "vlos"):
        assert f[k].dtype == np.float32 and f[k].shape == (32, 32, 32) and f[k].flags.c_contiguous
    assert 30.0 <= f["Tgas"].min() and f["Tgas"].max() < 120.0 and np.array_equal(f["Tgas"], f["Tdust"])
    ln = np.log(f["nH2"].astype(np.float64))
    assert ln.std() == pytest.approx(1.5, rel=1e-3)
    assert ln.mean() == pytest.approx(math.log(1e3) - 1.5 ** 2 / 2, abs=1e-3)
    # rotation: mean v_los per x column is the solid-body ramp, +-100 km/s at the box edge
    vx = f["vlos"].astype(np.float64).mean(axis=(0, 1)) / KMS
    slope = np.polyfit(np.arange(32) + 0.5 - 16, vx, 1)[0]
    assert slope == pytest.approx(100.0 / 16.0, rel=0.1)
    f2 = make_fields(cfg, r)
    assert all(np.array_equal(f[k], f2[k]) for k in ("nH2", "Tgas", "vlos"))


def test_medium_layers_and_other_workloads():
    cfg, r = make_workload("medium", n=16)
    assert cfg.nz == 16 + 32 and cfg.beam_fwhm_px == 3.0 and cfg.noise_sigma == 0.25 and cfg.dust_on
    f = make_fields(cfg, r)
    for sl in (slice(0, 16), slice(-16, None)):
        assert np.all(f["nH2"][sl] == 100.0) and np.all(f["Tgas"][sl] == 20.0) and np.all(f["vlos"][sl] == 0.0)
    assert f["nH2"][16:-16].std() > 0
    assert set(WORKLOADS) == {"tiny", "small", "medium", "large", "batch"}
    cl, _ = make_workload("large")
    assert (cl.nx, cl.nz, cl.nv, cl.dv_cms) == (512, 512, 1024, 0.25 * KMS) and cl.cell_cm == pytest.approx(0.5 * PC_CM)
    assert cl.v0_cms - cl.dv_cms / 2 == pytest.approx(-128 * KMS)
    cb, rb = make_workload("batch", n=8)
    m0 = make_fields(cb, rb, seed=1000)["meta"]
    m1 = make_fields(cb, rb, seed=1001)["meta"]
    assert m0 != m1 and 5 <= m0["sigma_t_kms"] <= 20 and 50 <= m0["v_edge_kms"] <= 150
    w = weight_cube(cb)
    assert w.shape == (8, 8, 256) and w.dtype == np.float32 and 0 <= w.min() and w.max() < 1
