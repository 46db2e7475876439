"""Sanitizer coverage.

* compute-sanitizer memcheck / racecheck over tests/sanitizer_target.py (small calls of every kernel; the line-window
  kernels keep spectra and march records in shared memory behind __syncwarp only).  The B200 profiling recipe allows ONE
  compute-sanitizer tool per GPU call, so each tool runs only when IRIS_SO_SANITIZER names it:
      IRIS_SO_SANITIZER=memcheck  python -m pytest tests/test_sanitizers.py -m gpu -q
      IRIS_SO_SANITIZER=racecheck python -m pytest tests/test_sanitizers.py -m gpu -q
  (summaries of the runs: profiles/r02_sanitizers.md).
* AddressSanitizer + UndefinedBehaviorSanitizer build of the oracle, exercised in a subprocess (CPU)."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.gpu
@pytest.mark.parametrize("tool", ["memcheck", "racecheck"])
def test_compute_sanitizer(tool):
    if os.environ.get("IRIS_SO_SANITIZER") != tool:
        pytest.skip("set IRIS_SO_SANITIZER=%s (one compute-sanitizer tool per GPU call)" % tool)
    cmd = ["compute-sanitizer", "--tool", tool, "--error-exitcode", "1", sys.executable, os.path.join(ROOT, "tests", "sanitizer_target.py")]
    p = subprocess.run(cmd, capture_output=True, text=True, timeout=1500)
    text = p.stdout + p.stderr
    out = os.path.join(ROOT, "gpurun_out")
    if os.path.isdir(out):
        with open(os.path.join(out, "sanitizer_%s.log" % tool), "w") as fh:
            fh.write(text)
    print(text[-3000:])
    if "closed on this pool" in text:
        pytest.skip("compute-sanitizer is closed on this GPU pool: " + text.strip().splitlines()[-1][:200])
    assert p.returncode == 0, text[-3000:]
    assert "host path" in text and ("ERROR SUMMARY: 0 errors" in text or "RACECHECK SUMMARY: 0 hazards" in text)


@pytest.mark.gpu
def test_bounds_checked_build_runs_every_kernel():
    """The library built with -DIRIS_SO_CHECKED (every shared-memory access of the line-window kernels tested against the
    region of its warp, __trap outside it) runs the same small calls of every kernel."""
    sys.path.insert(0, ROOT)
    from paper_2607_01338_b200 import build as cuda_build
    lib = cuda_build.build(checked=True)
    env = dict(os.environ, IRIS_SO_LIB=lib)
    p = subprocess.run([sys.executable, os.path.join(ROOT, "tests", "sanitizer_target.py")], capture_output=True, text=True,
                       env=env, timeout=1500)
    text = p.stdout + p.stderr
    assert p.returncode == 0 and "host path" in text and "IRIS_SO_CHECKED" not in text, text[-3000:]


ORACLE_DRIVER = r"""
import numpy as np
from iris_inputs import make_fields, make_workload, weight_cube
from oracle import Oracle
for name, kw in (("tiny", dict()), ("small", dict(integration=1, subsample=1)), ("small", dict(transfer_mode=1)),
                 ("small", dict(transfer_mode=2, integration=1)), ("small", dict(coef_grid=1, grid_n_density=9, grid_n_temp=5)),
                 ("small", dict(dust_per_channel=1))):
    cfg, r = make_workload(name, nx=5, ny=3, nz=7, nv=19)
    cfg = cfg.with_(beam_fwhm_px=3.0, noise_sigma=0.25, **kw)
    f = make_fields(cfg, r)
    o = Oracle(cfg, threads=2)
    cube = o.observe(f)
    assert np.isfinite(cube).all()
cfg, r = make_workload("batch", nx=4, ny=3, nz=6, nv=17)
f = make_fields(cfg, r)
o = Oracle(cfg, threads=2)
w = weight_cube(cfg)
g = o.grad_adjoint(f, w)
o.grad_fd(f, w, np.arange(5))
o.density_trace(f); o.metrics(w, w); o.levelpop(f["nH2"], f["Tgas"])
print("oracle under ASan + UBSan: ok")
"""


def test_oracle_under_address_and_undefined_behaviour_sanitizers(tmp_path):
    libasan = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip()
    libubsan = subprocess.run(["gcc", "-print-file-name=libubsan.so"], capture_output=True, text=True).stdout.strip()
    if not (os.path.isabs(libasan) and os.path.exists(libasan)):
        pytest.skip("libasan not installed")
    lib = str(tmp_path / "liboracle_san.so")
    subprocess.run(["g++", "-O1", "-g", "-std=c++17", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
                    "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer",
                    "-o", lib, os.path.join(ROOT, "oracle", "iris_oracle.cpp")], check=True)
    env = dict(os.environ, IRIS_ORACLE_LIB=lib, LD_PRELOAD=libasan + (":" + libubsan if os.path.exists(libubsan) else ""),
               ASAN_OPTIONS="detect_leaks=0:abort_on_error=0:exitcode=23", UBSAN_OPTIONS="print_stacktrace=1:halt_on_error=1",
               PYTHONPATH=ROOT, OMP_NUM_THREADS="2")
    p = subprocess.run([sys.executable, "-c", ORACLE_DRIVER], capture_output=True, text=True, env=env, cwd=ROOT, timeout=900)
    text = p.stdout + p.stderr
    assert p.returncode == 0 and "oracle under ASan + UBSan: ok" in text, text[-4000:]
    assert "ERROR: AddressSanitizer" not in text and "runtime error:" not in text, text[-4000:]
