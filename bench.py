#!/usr/bin/env python
"""Benchmark of the IRIS-SO hot path (BASELINE.json metric) -- one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload large] [--algo window|dense]

A "step" is one pass of the whole hot path (iris_so_observe: K1..K7) over one synthetic cube of the
workload.  `value` = whole-job (cell x channel) updates per second = N * nx*ny*nz*nv * K / t, inputs resident
in HBM.  `e2e` is the same metric through iris_so_observe_host (pinned host buffers, H2D + D2H inside the
timed region).  `roofline` describes the dominant kernel (the LOS transfer, K3) as DESIGN.md section 7
defines it; `cpu_baseline` is the float64 oracle timed on this box's host cores on a bounded column sample.
With --gpus N > 1 (torchrun) every rank renders its own independent cube ("replicas only": the path has no
exchange step).  --impl reference times the oracle instead (rank 0 only).
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from iris_inputs import make_fields, make_workload  # noqa: E402

METRIC = "los_transfer_cell_channel_updates_per_s"
UNIT = "updates/s"

# Algorithmic work of the LOS transfer kernel.  Per evaluated (cell, channel) update the
# recurrence needs 3 SFU operations (2^(-x^2) of the profile, 2^(-t) of 1 - exp(-tau_L), 1 / tau_T) -- 2 without dust --
# and 17 (13) FP32 multiply-adds; per (pixel, cell) it needs 5 SFU operations (window: log, sqrt, 1 / s; dust:
# exp(-tau_d); source function: 1 / a_c) and about 60 FP32 operations.  Peaks measured on this pool's B200
# (profiles/r01_pipe_microbench.md): MUFU 0.50 warp instructions / clk / SM = 16 lanes, FFMA 3.90 = 124.9 lanes.
SFU_PER_UPDATE = {True: 3, False: 2}            # keyed by dust_on
FP32_PER_UPDATE = {True: 17, False: 13}
SFU_PER_PIXEL_CELL = {True: 5, False: 4}
FP32_PER_PIXEL_CELL = 60
SM_COUNT, SFU_LANES_PER_SM_CLK, FP32_LANES_PER_SM_CLK = 148, 16.0, 124.9


# STORED figures, not values of this run: dram__bytes_read.sum + dram__bytes_write.sum of one launch of the dominant kernel
# from the committed `ncu --set full` capture of the named profiles/ pass, keyed by (workload, kernel).  Refreshed with
# every profiles/ pass; `roofline.traffic_source` names the pass in the JSON line.
NCU_TRAFFIC_BYTES = {
    ("large", "transfer_series_kernel"): (4412700000, "profiles/r02_final.md (3.2538 + 1.0450 GB reachable-range variant, 0.1105 + 0.0034 GB list pass)"),
    ("medium", "transfer_series_kernel"): (566200000, "profiles/r02_final.md (453.1 + 113.1 MB)"),
}


def env_rank():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return dict(hbm_gbs=float(d["hbm_gbs"]), sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


# --------------------------------------------------------------------------------------------------------
# distributed plumbing (NCCL on GPUs; the same helpers run under gloo in tests/test_bench_dist.py)
def dist_init(world, backend):
    if world <= 1:
        return None
    import torch.distributed as dist
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    os.environ.setdefault("MASTER_PORT", "29511")
    if not dist.is_initialized():
        dist.init_process_group(backend=backend)
    return dist


def dist_barrier(dist):
    if dist is not None:
        dist.barrier()


def dist_max(dist, value, device="cpu"):
    """Max over ranks of a python float."""
    if dist is None:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def dist_sum(dist, value, device="cpu"):
    if dist is None:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def aggregate_throughput(dist, units_this_rank, ms_this_rank, device="cpu"):
    """Whole-job throughput: all ranks' units / the slowest rank's time (weak scaling, replicas)."""
    ms = dist_max(dist, ms_this_rank, device)
    units = dist_sum(dist, units_this_rank, device)
    return units / (ms * 1e-3), ms


# --------------------------------------------------------------------------------------------------------
class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, uuid):
        self.proc = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", uuid, "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                                          "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            pass
        self.t0 = time.time()

    def stop(self):
        out = dict(sm_mhz=None, sm_max_mhz=None, reasons=[], samples=0)
        if self.proc is None:
            return out
        time.sleep(0.15)
        self.proc.terminate()
        try:
            text, _ = self.proc.communicate(timeout=5)
        except Exception:
            self.proc.kill()
            return out
        sm, smax, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in text.strip().splitlines():
            parts = [p.strip() for p in line.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); smax.append(float(parts[1])); power.append(float(parts[2]))
            except ValueError:
                continue
            for n, v in zip(names, parts[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        if sm:
            # median over the samples taken under load (the busiest half)
            hot = sorted(sm)[len(sm) // 2:]
            out.update(sm_mhz=statistics.median(hot), sm_max_mhz=max(smax), reasons=sorted(reasons), samples=len(sm),
                       power_w_max=max(power))
        return out


# --------------------------------------------------------------------------------------------------------
def oracle_sample(cfg, fields, n_cols, seed=123, threads=None):
    """Whole path of the oracle on n_cols seeded columns of the workload, as an independent (nz, 1, n_cols) cube
    (columns do not interact before the beam).  Returns (seconds, updates, threads)."""
    from oracle import Oracle
    rng = np.random.default_rng(seed)
    plane = cfg.nx * cfg.ny
    pix = np.sort(rng.choice(plane, size=min(n_cols, plane), replace=False))
    sub = {k: np.ascontiguousarray(fields[k].reshape(cfg.nz, plane)[:, pix]).reshape(cfg.nz, 1, pix.size)
           for k in ("nH2", "Tgas", "Tdust", "vlos")}
    cfg_s = cfg.with_(nx=int(pix.size), ny=1, beam_fwhm_px=0.0, noise_sigma=0.0, noise_mu=0.0)
    o = Oracle(cfg_s, threads=threads)
    t0 = time.perf_counter()
    o.observe(sub, beam=False, noise=False)
    dt = time.perf_counter() - t0
    return dt, int(pix.size) * cfg.nz * cfg.nv, omp_threads(threads)


def omp_threads(threads=None):
    if threads is not None:
        return int(threads)
    try:
        import ctypes
        return int(ctypes.CDLL("libgomp.so.1").omp_get_max_threads())
    except OSError:
        return os.cpu_count() or 1


def cpu_baseline(cfg, fields, budget_s=12.0):
    """Oracle, as it stands, on a bounded sample: about budget_s seconds of wall time on all host cores, then about
    budget_s / 2 seconds on ONE thread (BASELINE.md section 2 asks for both)."""
    th = omp_threads()
    n0 = max(2 * th, 16)
    dt, upd, th = oracle_sample(cfg, fields, n0)
    n = int(min(max(n0, n0 * budget_s / max(dt, 1e-3)), cfg.nx * cfg.ny, 65536))
    if n > n0:
        dt, upd, th = oracle_sample(cfg, fields, n)
    per_col_1 = dt * th / max(n, 1)                       # a column on one thread, if the scaling were perfect
    n1 = int(min(max(4, 0.5 * budget_s / max(per_col_1, 1e-4)), n))
    dt1, upd1, _ = oracle_sample(cfg, fields, n1, threads=1)
    return dict(value=upd / dt, unit=UNIT, cores=th, kind="oracle",
                sample="%d of %d seeded pixel columns of the %s workload (whole path K1-K5 per column, float64, g++ -O2, "
                       "OpenMP over columns), %.1f s" % (min(n, cfg.nx * cfg.ny), cfg.nx * cfg.ny, cfg.name, dt),
                single_thread={"value": upd1 / dt1, "unit": UNIT, "cores": 1,
                               "sample": "%d of the same columns on one thread, %.1f s" % (n1, dt1)})


# --------------------------------------------------------------------------------------------------------
def run_reference(args):
    rank, _, world = env_rank()
    if rank != 0:
        return 0
    cfg, recipe = make_workload(args.workload)
    fields = make_fields(cfg, recipe)
    th = omp_threads()
    # size the per-step sample so that warmup + steps end within a few minutes
    dt, upd, th = oracle_sample(cfg, fields, max(2 * th, 16))
    per_col = dt / max(2 * th, 16)
    total_budget = 150.0
    n_cols = int(min(max(2 * th, total_budget / (args.steps + args.warmup) / per_col), cfg.nx * cfg.ny, 16384))
    for _ in range(args.warmup):
        oracle_sample(cfg, fields, n_cols)
    t = 0.0
    updates = 0
    for s in range(args.steps):
        dt, upd, th = oracle_sample(cfg, fields, n_cols, seed=1000 + s)
        t += dt
        updates += upd
    value = updates / t
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * t / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(cfg, args, sample="%d pixel columns per step" % n_cols),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": th, "kind": "oracle",
                         "sample": "%d of %d seeded pixel columns per step, whole path per column" % (n_cols, cfg.nx * cfg.ny)},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def workload_config(cfg, args, **extra):
    c = {"workload": "%s: %dx%dx%d cells, %d channels x %.3g km/s, %d levels, dust %s, beam %.3g px, noise %.3g K"
                     % (cfg.name, cfg.nx, cfg.ny, cfg.nz, cfg.nv, cfg.dv_cms / 1e5, cfg.n_levels,
                        "on" if cfg.dust_on else "off", cfg.beam_fwhm_px, cfg.noise_sigma),
         "baseline_config_index": {"tiny": 0, "small": 1, "medium": 2, "large": 3, "batch": 4}.get(cfg.name),
         "parallelism": "replicas x%d (no sharding, no collective in the data path)" % args.gpus,
         "cache": "inputs larger than L2 (4 field planes + 6 coefficient planes per step)"}
    c.update(extra)
    return c


# --------------------------------------------------------------------------------------------------------
def timed_steps(torch, it, d, steps, cube):
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for _ in range(steps):
        it.observe(*d, cube=cube)
    b.record()
    torch.cuda.synchronize()
    return a.elapsed_time(b)


def bench_workload(torch, dist, name, algo, steps, warmup, rank, peaks, want_e2e, want_dense_probe, sampler_uuid):
    from paper_2607_01338_b200 import IrisSO, ALGO_DENSE, ALGO_WINDOW
    dev = torch.device("cuda", torch.cuda.current_device())
    cfg, recipe = make_workload(name)
    fields = make_fields(cfg, recipe, seed=recipe["seed"] + rank)
    d = [torch.from_numpy(fields[k]).to(dev) for k in ("nH2", "Tgas", "Tdust", "vlos")]
    it = IrisSO(cfg, transfer_algo=ALGO_DENSE if algo == "dense" else ALGO_WINDOW)
    cube = torch.empty(it.shape_cube, dtype=torch.float32, device=dev)
    for _ in range(max(warmup, 3)):
        it.observe(*d, cube=cube)
    torch.cuda.synchronize()
    sampler = ClockSampler(sampler_uuid) if sampler_uuid else None
    dist_barrier(dist)
    torch.cuda.synchronize()
    it.profile(True)
    l0 = it.launch_count()
    ms = timed_steps(torch, it, d, steps, cube)
    launches = it.launch_count() - l0
    prof = it.profile_read()
    it.profile(False)
    dist_barrier(dist)
    clocks = sampler.stop() if sampler else None
    updates = cfg.nx * cfg.ny * cfg.nz * cfg.nv
    value, ms_max = aggregate_throughput(dist, updates * steps, ms, dev)

    res = dict(cfg=cfg, fields=fields, value=value, ms=ms_max, ms_per_step=ms_max / steps, launches=launches, clocks=clocks,
               stages={k: {"ms_per_step": v[0] / steps, "launches_per_step": v[1] / steps} for k, v in prof.items() if v[1]})
    # roofline of the dominant kernel (LOS transfer): the slower of HBM bytes, SFU operations and FP32 operations
    # seconds per step of the transfer stage (the series kernel with reachable-range spectra is two launches: the
    # circular-buffer variant, then the whole-spectrum variant over the pixels it handed over)
    t_k3 = prof["transfer"][0] / steps * 1e-3
    ncell = cfg.nx * cfg.ny * cfg.nz
    win_updates = it.transfer_work()
    dense_kernel = it.transfer_kernel() == "transfer_dense_kernel"
    n_upd = updates if dense_kernel else win_updates
    clk = peaks["sm_max_mhz"] * 1e6
    sfu_ops = n_upd * SFU_PER_UPDATE[cfg.dust_on] + ncell * SFU_PER_PIXEL_CELL[cfg.dust_on]
    fp32_ops = n_upd * FP32_PER_UPDATE[cfg.dust_on] + ncell * FP32_PER_PIXEL_CELL
    sfu_peak = SM_COUNT * SFU_LANES_PER_SM_CLK * clk
    fp32_peak = SM_COUNT * FP32_LANES_PER_SM_CLK * clk
    alg_bytes = 24 * ncell + 4 * cfg.nx * cfg.ny * cfg.nv
    t_sfu, t_fp32, t_hbm = sfu_ops / sfu_peak, fp32_ops / fp32_peak, alg_bytes / (peaks["hbm_gbs"] * 1e9)
    res["roofline"] = {
        "bound": "alu", "pipe": "sfu (MUFU.EX2 / MUFU.RCP)", "kernel": it.transfer_kernel(), "algorithm": algo,
        "achieved": sfu_ops / t_k3 / 1e12, "peak": sfu_peak / 1e12, "unit": "Tops/s (SFU lane operations)",
        "frac": t_sfu / t_k3, "traffic": NCU_TRAFFIC_BYTES.get((cfg.name, it.transfer_kernel()), (None, None))[0],
        "traffic_source": "stored ncu figure, not measured in this run: %s"
                          % NCU_TRAFFIC_BYTES.get((cfg.name, it.transfer_kernel()), (None, "no capture for this workload / kernel"))[1],
        "peak_source": "148 SMs x 16 SFU lanes/clk (measured MUFU issue rate, profiles/r01_pipe_microbench.md) x %.0f MHz "
                       "max SM clock (MEASURED_PEAKS.json, %s)" % (peaks["sm_max_mhz"], peaks["source"]),
        "ms_per_launch": t_k3 * 1e3, "updates_evaluated": n_upd, "updates_nominal": updates,
        "sfu_per_update": SFU_PER_UPDATE[cfg.dust_on], "sfu_per_pixel_cell": SFU_PER_PIXEL_CELL[cfg.dust_on],
        "floors_ms": {"sfu": t_sfu * 1e3, "fp32": t_fp32 * 1e3, "hbm": t_hbm * 1e3},
        "nominal_updates_per_s": updates / t_k3,
        "fp32": {"ops": fp32_ops, "achieved_Tops_s": fp32_ops / t_k3 / 1e12, "peak_Tops_s": fp32_peak / 1e12,
                 "frac": t_fp32 / t_k3},
        "hbm": {"algorithmic_bytes": alg_bytes, "achieved_gbs": alg_bytes / t_k3 / 1e9, "peak_gbs": peaks["hbm_gbs"],
                "frac": t_hbm / t_k3},
    }
    if clocks and clocks.get("sm_mhz"):
        res["roofline"]["frac_at_measured_clock"] = res["roofline"]["frac"] * peaks["sm_max_mhz"] / clocks["sm_mhz"]

    if want_dense_probe and algo != "dense":
        itd = IrisSO(cfg, transfer_algo=ALGO_DENSE)
        for _ in range(2):
            itd.observe(*d, cube=cube, beam=False, noise=False)
        torch.cuda.synchronize()
        itd.profile(True)
        for _ in range(2):
            itd.observe(*d, cube=cube, beam=False, noise=False)
        pd = itd.profile_read()
        t_d = pd["transfer"][0] / pd["transfer"][1] * 1e-3
        res["dense_probe"] = {"kernel": "transfer_dense_kernel", "ms_per_launch": t_d * 1e3, "nominal_updates_per_s": updates / t_d,
                              "note": "north_star's literal kernel (register-resident channel blocks, erfc edges); it skips "
                                      "16-channel blocks beyond the erfc range, so no roofline fraction is quoted for it"}
        itd.close()

    if want_e2e:
        h = [torch.from_numpy(fields[k]).pin_memory() for k in ("nH2", "Tgas", "Tdust", "vlos")]
        hc = torch.empty(it.shape_cube, dtype=torch.float32).pin_memory()
        it.observe_host(*h, hc)                               # allocates the staging buffers (untimed)
        n_e2e = max(1, min(steps, 3))
        dist_barrier(dist)
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(n_e2e):
            it.observe_host(*h, hc)
        b.record()
        torch.cuda.synchronize()
        e_val, e_ms = aggregate_throughput(dist, updates * n_e2e, a.elapsed_time(b), dev)
        res["e2e"] = {"value": e_val, "unit": UNIT, "h2d_bytes_per_step": int(4 * ncell * 4),
                      "d2h_bytes_per_step": int(cfg.nx * cfg.ny * cfg.nv * 4), "ms_per_step": e_ms / n_e2e, "steps": n_e2e,
                      "api": "iris_so_observe_host (pinned host buffers)", "checksum": float(hc.double().abs().sum())}
        del h, hc
    it.close()
    return res


MODE_PROBES = {"thick_smooth_subsample1 (the paper's production mode)": (0, 1, 1), "thick_formal_subsample1": (0, 0, 1),
               "thick_smooth": (0, 1, 0), "selectively_thin_formal": (1, 0, 0), "selectively_thin_smooth": (1, 1, 0),
               "thin_formal": (2, 0, 0), "thin_smooth": (2, 1, 0)}


def bench_modes(torch, warmup):
    """The paper's other transfer / integration modes on the medium cube: ms per transfer stage and nominal
    spectral-point updates per second (cells x points of the spectrum), with the kernel that ran them."""
    from paper_2607_01338_b200 import IrisSO
    dev = torch.device("cuda", torch.cuda.current_device())
    cfg0, recipe = make_workload("medium")
    fields = make_fields(cfg0, recipe)
    d = [torch.from_numpy(fields[k]).to(dev) for k in ("nH2", "Tgas", "Tdust", "vlos")]
    out = {}
    for name, (m, i, sub) in MODE_PROBES.items():
        cfg = cfg0.with_(transfer_mode=m, integration=i, subsample=sub)
        it = IrisSO(cfg)
        cube = torch.empty(it.shape_cube, dtype=torch.float32, device=dev)
        for _ in range(warmup):
            it.observe(*d, cube=cube)
        torch.cuda.synchronize()
        it.profile(True)
        for _ in range(3):
            it.observe(*d, cube=cube)
        prof = it.profile_read()
        it.profile(False)
        # the smooth line-window march is followed by the gated dense kernel (two launches per call; the second returns
        # at once unless fell_back): the time is that of the transfer stage of one call
        t = prof["transfer"][0] / 3 * 1e-3
        points = cfg.nv * (3 * (sub + 1) // 2 if sub else 1)      # (f + 1) / 2 Simpson panels x 3 points per channel
        out[name] = {"kernel": it.transfer_kernel(), "ms_per_launch": t * 1e3,
                     "launches_per_call": prof["transfer"][1] / 3, "pixels_handed_over": it.smooth_fallback(),
                     "point_updates_per_s": cfg.nx * cfg.ny * cfg.nz * points / t,
                     "ms_per_cube": sum(v[0] for v in prof.values()) / 3}
        if m == 0 and it.transfer_kernel() != "transfer_modes_kernel":
            # roofline of the thick modes on their line-window kernels: SFU operations per evaluated
            # point update -- formal 3 (profile, exp(-tau_L), 1 / tau_T), smooth 2 (profile, 1 / (3 + 2 tau)) -- and 5 per
            # (pixel, cell); evaluated = points inside the windows (formal) / inside the 12-cell hulls (smooth)
            evaluated = it.transfer_work()
            per_update = 2 if i == 1 else 3
            ncell = cfg.nx * cfg.ny * cfg.nz
            sfu = per_update * evaluated + 5 * ncell
            t_floor = sfu / (SM_COUNT * SFU_LANES_PER_SM_CLK * measured_peaks()["sm_max_mhz"] * 1e6)
            out[name]["roofline"] = {"bound": "alu", "pipe": "sfu", "updates_evaluated": evaluated, "sfu_per_update": per_update,
                                     "floor_ms": t_floor * 1e3, "frac": t_floor / t,
                                     "note": "time includes the list-driven dense launch for the pixels handed over"}
        it.close()
    return out


def bench_small_configs(torch, warmup):
    """BASELINE configs 0, 1 and 4 (tiny, small, batch): whole-path time per cube, and for the batch config the
    reverse-scan adjoint d(sum w cube)/d n_H2 (K8 + K9) and the 64-cube render rate (cubes rendered back to back on
    one stream, one context, fields of all cubes resident in HBM)."""
    from paper_2607_01338_b200 import IrisSO
    from iris_inputs import weight_cube
    dev = torch.device("cuda", torch.cuda.current_device())
    out = {}

    def timed(fn, reps):
        for _ in range(warmup):
            fn()
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(reps):
            fn()
        b.record()
        torch.cuda.synchronize()
        return a.elapsed_time(b) / reps

    for name in ("tiny", "small"):
        cfg, recipe = make_workload(name)
        f = make_fields(cfg, recipe)
        d = [torch.from_numpy(f[k]).to(dev) for k in ("nH2", "Tgas", "Tdust", "vlos")]
        it = IrisSO(cfg)
        cube = torch.empty(it.shape_cube, dtype=torch.float32, device=dev)
        ms = timed(lambda: it.observe(*d, cube=cube), 50)
        out[name] = {"ms_per_cube": ms, "nominal_updates_per_s": cfg.nx * cfg.ny * cfg.nz * cfg.nv / (ms * 1e-3),
                     "what": "%dx%dx%d cells, %d channels" % (cfg.nx, cfg.ny, cfg.nz, cfg.nv)}
        it.close()
    # batch: 64 independent seeded cubes (8 distinct field sets cycled, all resident), then the adjoint of one
    cfg, recipe = make_workload("batch", seed=1000)
    sets = []
    for i in range(8):
        c_i, r_i = make_workload("batch", seed=1000 + i)
        f = make_fields(c_i, r_i)
        sets.append([torch.from_numpy(f[k]).to(dev) for k in ("nH2", "Tgas", "Tdust", "vlos")])
    it = IrisSO(cfg)
    cubes = torch.empty((64,) + tuple(it.shape_cube), dtype=torch.float32, device=dev)

    def render64():
        for i in range(64):
            it.observe(*sets[i % 8], cube=cubes[i])

    ms64 = timed(render64, 3)
    w = torch.from_numpy(weight_cube(cfg)).to(dev)
    grad = torch.empty((cfg.nz, cfg.ny, cfg.nx), dtype=torch.float32, device=dev)
    ms_adj = timed(lambda: it.observe_adjoint(*sets[0], w, grad=grad), 10)
    # the same gradient in the paper's production mode (thick, smooth TR + BDF2 + ReLU, f = 1): adjoint_modes_kernel
    it_p = IrisSO(cfg.with_(integration=1, subsample=1))
    cube_p = torch.empty(it_p.shape_cube, dtype=torch.float32, device=dev)
    ms_fwd_p = timed(lambda: it_p.observe(*sets[0], cube=cube_p), 10)
    ms_adj_p = timed(lambda: it_p.observe_adjoint(*sets[0], w, grad=grad), 10)
    it_p.close()
    out["batch"] = {"cubes": 64, "ms_per_64_cubes": ms64, "cubes_per_s": 64e3 / ms64, "adjoint_ms_per_cube": ms_adj,
                    "production_mode_ms_per_cube": ms_fwd_p, "production_mode_adjoint_ms_per_cube": ms_adj_p,
                    "nominal_updates_per_s": 64 * cfg.nx * cfg.ny * cfg.nz * cfg.nv / (ms64 * 1e-3),
                    "what": "64 x (%dx%dx%d cells, %d channels, dust, beam %.3g px, noise %.3g K)"
                            % (cfg.nx, cfg.ny, cfg.nz, cfg.nv, cfg.beam_fwhm_px, cfg.noise_sigma)}
    it.close()
    # level populations from tabulated rates of three partners on a 13-point temperature grid (medium cube, K1 + K2 only)
    cfg, recipe = make_workload("medium")
    grid = np.array([5.0, 10.0, 20.0, 30.0, 50.0, 70.0, 100.0, 150.0, 200.0, 300.0, 500.0, 1000.0, 2000.0])
    base = cfg.coll_down_ref[None] * (grid[:, None, None] / cfg.coll_T_ref) ** cfg.coll_T_exp
    frac = np.array([0.25, 0.75, 0.2])
    cfg_t = cfg.with_(coll_T_grid=grid, coll_table=np.stack([base * 0.3 / frac[0], base * 0.5 / frac[1], base * 0.2 / frac[2]]),
                      coll_partner_frac=frac)
    f = make_fields(cfg, recipe)
    d = [torch.from_numpy(f[k]).to(dev) for k in ("nH2", "Tgas", "Tdust", "vlos")]
    res = {}
    for label, c in (("power_law", cfg), ("tabulated_3_partners", cfg_t)):
        it = IrisSO(c)
        cube = torch.empty(it.shape_cube, dtype=torch.float32, device=dev)
        for _ in range(warmup):
            it.observe(*d, cube=cube)
        torch.cuda.synchronize()
        it.profile(True)
        for _ in range(5):
            it.observe(*d, cube=cube)
        prof = it.profile_read()
        it.profile(False)
        res[label] = prof["cell"][0] / prof["cell"][1]
        it.close()
    out["cell_kernel_ms_medium"] = res
    return out


def bench_grid(torch, warmup, large_fields=None):
    """The coefficient grid of PAPER.md section 4.2 / 4.3 (coef_grid = 1, the paper's 128 x 64 nodes over n_H2 = 1e-2 .. 1e9
    cm^-3 and T = 5 .. 3000 K) in place of the per-cell level solve: time of the cell stage (K1 + K2) per cube, and the
    gap of the interpolated medium cube to the cube of the exact solve (reported, not a parity claim)."""
    from paper_2607_01338_b200 import IrisSO
    dev = torch.device("cuda", torch.cuda.current_device())
    out = {}
    for name in ("medium", "large"):
        cfg, recipe = make_workload(name)
        if name == "large" and large_fields is not None:
            fields = large_fields
        else:
            fields = make_fields(cfg, recipe)
        d = [torch.from_numpy(fields[k]).to(dev) for k in ("nH2", "Tgas", "Tdust", "vlos")]
        cubes = {}
        res = {}
        for label, c in (("exact", cfg), ("grid", cfg.with_(coef_grid=1))):
            it = IrisSO(c)
            cube = torch.empty(it.shape_cube, dtype=torch.float32, device=dev)
            for _ in range(warmup):
                it.observe(*d, cube=cube, beam=False, noise=False)
            torch.cuda.synchronize()
            it.profile(True)
            for _ in range(5):
                it.observe(*d, cube=cube, beam=False, noise=False)
            prof = it.profile_read()
            it.profile(False)
            res["cell_stage_ms_" + label] = prof["cell"][0] / prof["cell"][1]
            if name == "medium":
                cubes[label] = cube.clone()
            it.close()
            del cube
        if name == "medium":
            peak = cubes["exact"].abs().amax(dim=-1, keepdim=True)
            res["max_abs_dT_over_pixel_peak"] = float(((cubes["grid"] - cubes["exact"]).abs() / (peak + 1e-3)).max())
            res["max_abs_dT_K"] = float((cubes["grid"] - cubes["exact"]).abs().max())
        ncell = cfg.nx * cfg.ny * cfg.nz
        res["hbm_floor_ms"] = 40.0 * ncell / (measured_peaks()["hbm_gbs"] * 1e9) * 1e3     # 16 B of fields in, 24 B of planes out
        out[name] = res
        del d
        torch.cuda.empty_cache()
    out["grid"] = "128 x 64 nodes, n_H2 1e-2 .. 1e9 cm^-3, T 5 .. 3000 K (ObsConfig defaults)"
    return out


def run_ours(args):
    import torch
    rank, local_rank, world = env_rank()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA path has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank % torch.cuda.device_count())
    from paper_2607_01338_b200 import build as cuda_build
    if rank == 0:
        cuda_build.build()
    dist = dist_init(world, "nccl")
    dist_barrier(dist)
    peaks = measured_peaks()
    uuid = str(torch.cuda.get_device_properties(torch.cuda.current_device()).uuid)
    uuid = uuid if uuid.startswith("GPU-") else "GPU-" + uuid

    main = bench_workload(torch, dist, args.workload, args.algo, args.steps, args.warmup, rank, peaks, want_e2e=not args.no_e2e,
                          want_dense_probe=(world == 1 and not args.no_extras), sampler_uuid=uuid if rank == 0 else None)
    cfg = main["cfg"]
    extra = {}
    if not args.no_extras and args.workload != "medium":
        med = bench_workload(torch, dist, "medium", args.algo, max(args.steps, 5), args.warmup, rank, peaks, want_e2e=False,
                             want_dense_probe=False, sampler_uuid=None)
        extra["cubes_per_s_256x256x288_512ch"] = {
            "value": world * 1e3 / med["ms_per_step"], "unit": "cubes/s", "ms_per_cube": med["ms_per_step"],
            "what": "iris_so_observe on BASELINE config 2 (medium: 256^2 x (256+32) cells, 512 channels, dust, beam 3 px, noise 0.25 K)",
            "stages": med["stages"], "transfer_roofline_frac": med["roofline"]["frac"],
            "transfer_nominal_updates_per_s": med["roofline"]["nominal_updates_per_s"]}
    if not args.no_extras and world == 1:
        extra["other_modes_256x256x288_512ch"] = bench_modes(torch, max(args.warmup, 3))
        extra["other_configs"] = bench_small_configs(torch, max(args.warmup, 3))
        extra["coefficient_grid"] = bench_grid(torch, max(args.warmup, 3), main["fields"] if cfg.name == "large" else None)
    if rank != 0:
        return 0
    cb = None
    if world == 1 and not args.no_cpu_baseline:
        cb = cpu_baseline(cfg, main["fields"])
    line = {
        "metric": METRIC, "value": main["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": main["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic", "impl": "ours",
        "config": workload_config(cfg, args, transfer_algo=args.algo),
        "roofline": main["roofline"], "cpu_baseline": cb, "e2e": main.get("e2e"), "gpu_launches": main["launches"],
        "clocks": main["clocks"], "stages": main["stages"], "extra": extra,
    }
    if "dense_probe" in main:
        line["extra"]["dense_algorithm_probe"] = main["dense_probe"]
    print(json.dumps(line))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="large", choices=["tiny", "small", "medium", "large"])
    ap.add_argument("--algo", default="window", choices=["window", "dense"])
    ap.add_argument("--no-extras", action="store_true", help="skip the medium-cube and dense-algorithm side measurements")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer leg (profiling runs: its slab pipeline launches per slab)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
