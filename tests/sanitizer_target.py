"""Small calls of every kernel of the library, meant to be run under compute-sanitizer (tests/test_sanitizers.py):
every LOS transfer kernel (series modes 0 - 3, window, dense, dense per-channel, modes, smooth window + hand-over list),
the level / coefficient / grid kernels, beam, noise, diagnostics and the adjoints (hot path and the other thick modes).  Prints one line per call."""
import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from iris_inputs import make_fields, make_workload, weight_cube  # noqa: E402
from paper_2607_01338_b200 import IrisSO  # noqa: E402


def main():
    dev = torch.device("cuda", 0)
    cfg0, r = make_workload("small", nx=13, ny=5, nz=21, nv=45)
    cfg0 = cfg0.with_(v0_cms=-0.5 * 44 * cfg0.dv_cms, beam_fwhm_px=3.0, noise_sigma=0.25, seed=5)
    f = make_fields(cfg0, r)
    f["vlos"] = (0.1 * f["vlos"]).astype(np.float32)
    d = [torch.from_numpy(f[k]).to(dev) for k in ("nH2", "Tgas", "Tdust", "vlos")]
    variants = [("series", dict(), 0), ("series no dust", dict(dust_on=False, kappa_gas_cm2_g=0.0), 0),
                ("window edge", dict(dv_cms=1.0e5, v0_cms=-22.0e5), 0), ("dense", dict(), 1),
                ("dense per channel", dict(dust_per_channel=1), 0), ("coefficient grid", dict(coef_grid=1), 0),
                ("series selectively thin", dict(transfer_mode=1), 0), ("series thin", dict(transfer_mode=2), 0),
                ("series thin simpson", dict(transfer_mode=2, integration=1), 0), ("series fine grid", dict(subsample=1), 0),
                ("smooth window", dict(integration=1), 0), ("smooth window fine", dict(integration=1, subsample=1), 0),
                ("smooth window hand-over", dict(integration=1, kappa_gas_cm2_g=40.0 * cfg0.kappa_gas_cm2_g), 0),
                ("smooth window selectively thin", dict(transfer_mode=1, integration=1), 0),
                ("modes selectively thin smooth", dict(transfer_mode=1, integration=1), 1),
                ("modes dense thick smooth", dict(integration=1, subsample=3), 1)]
    for name, kw, algo in variants:
        it = IrisSO(cfg0.with_(**kw), transfer_algo=algo)
        cube = it.observe(*d)
        torch.cuda.synchronize()
        assert bool(torch.isfinite(cube).all()), name
        print("%-32s %-30s ok" % (name, it.transfer_kernel()))
        it.close()
    it = IrisSO(cfg0)
    pop = it.levelpop(d[0], d[1])
    It, Ic = it.transfer(*d, pop=pop)
    it.density_trace(d[0], d[3])
    it.metrics(It, It)
    w = torch.from_numpy(weight_cube(cfg0)).to(dev)
    g = it.observe_adjoint(*d, w)
    ga = it.observe_adjoint(*d, w, wrt="abundance")
    torch.cuda.synchronize()
    assert bool(torch.isfinite(g).all()) and bool(torch.isfinite(ga).all())
    print("%-32s ok" % "levelpop / transfer / diagnostics / adjoint")
    # the stored-state reverse sweep of the other thick modes (adjoint_modes_kernel): smooth / formal, coarse / fine grid
    for name, kw in (("adjoint thick smooth", dict(integration=1)), ("adjoint production mode", dict(integration=1, subsample=1)),
                     ("adjoint formal fine grid", dict(subsample=3))):
        itm = IrisSO(cfg0.with_(**kw))
        gm = itm.observe_adjoint(*d, w)
        gma = itm.observe_adjoint(*d, w, wrt="abundance")
        torch.cuda.synchronize()
        assert bool(torch.isfinite(gm).all()) and bool(torch.isfinite(gma).all()), name
        print("%-32s ok" % name)
        itm.close()
    # the entry point that allocates nothing (coefficient planes in the library's static scratch), twice in a row
    raw = torch.empty(it.shape_cube, dtype=torch.float32, device=dev)
    for _ in range(2):
        it.observe_raw_static(*d, raw)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(raw).all())
    print("%-32s ok" % "static-scratch entry point")
    h = [torch.from_numpy(f[k]).pin_memory() for k in ("nH2", "Tgas", "Tdust", "vlos")]
    hc = torch.empty(it.shape_cube, dtype=torch.float32).pin_memory()
    it.observe_host(*h, hc)
    print("%-32s ok" % "host path")
    it.close()


if __name__ == "__main__":
    main()
