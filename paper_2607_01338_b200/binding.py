"""ctypes binding of include/iris_so.h: argument marshalling only (every step runs in the CUDA kernels)."""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# IRIS_SO_LIB: another build of the same library to load instead (the bounds-checked build of tests/test_sanitizers.py)
_LIB_PATH = os.environ.get("IRIS_SO_LIB") or os.path.join(_HERE, "libiris_so.so")
_lib = None

ALGO_AUTO, ALGO_DENSE, ALGO_WINDOW, ALGO_WINDOW_EDGE = 0, 1, 2, 3

# every entry point include/iris_so.h declares
DECLARED_SYMBOLS = (
    "iris_so_create", "iris_so_destroy", "iris_so_last_error", "iris_so_status_string", "iris_so_version",
    "iris_so_launch_count", "iris_so_scratch_bytes", "iris_so_levelpop", "iris_so_transfer", "iris_so_observe",
    "iris_so_observe_stages", "iris_so_observe_host", "iris_so_observe_adjoint", "iris_so_beam", "iris_so_noise",
    "iris_so_profile", "iris_so_profile_read", "iris_so_transfer_work", "iris_so_transfer_kernel", "iris_so_smooth_fallback",
    "iris_so_density_trace", "iris_so_metrics", "iris_so_observe_adjoint_abundance", "iris_so_observe_raw_static",
)
STATIC_MAX_CELLS = 1 << 19      # IRIS_SO_STATIC_MAX_CELLS of include/iris_so.h
STAGES = {"cell": 0, "transfer": 1, "beam": 2, "noise": 3, "adjoint": 4}


class IrisSOError(RuntimeError):
    def __init__(self, status, text):
        super().__init__("iris_so status %d: %s" % (status, text))
        self.status = status


class _Config(C.Structure):
    _fields_ = [
        ("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
        ("cell_cm", C.c_double),
        ("n_levels", C.c_int32),
        ("energy_K", C.POINTER(C.c_double)), ("weight", C.POINTER(C.c_double)),
        ("einstein_A", C.POINTER(C.c_double)), ("coll_down_ref", C.POINTER(C.c_double)),
        ("coll_T_ref", C.c_double), ("coll_T_exp", C.c_double),
        ("line_upper", C.c_int32), ("line_lower", C.c_int32),
        ("nu0_Hz", C.c_double), ("mol_mass_g", C.c_double), ("abundance", C.c_double),
        ("microturb_cms", C.c_double), ("T_bar", C.c_double), ("T_cmb", C.c_double), ("T_inf", C.c_double),
        ("dust_on", C.c_int32),
        ("kappa_gas_cm2_g", C.c_double), ("mass_per_H2_g", C.c_double),
        ("nv", C.c_int32),
        ("v0_cms", C.c_double), ("dv_cms", C.c_double),
        ("subtract_continuum", C.c_int32), ("subtract_space", C.c_int32), ("out_unit", C.c_int32),
        ("beam_fwhm_px", C.c_double), ("noise_mu", C.c_double), ("noise_sigma", C.c_double),
        ("noise_gamma_mode", C.c_int32),
        ("seed", C.c_uint64),
        ("transfer_algo", C.c_int32),
        ("transfer_mode", C.c_int32), ("integration", C.c_int32), ("subsample", C.c_int32),
        ("coll_n_partners", C.c_int32), ("coll_nT", C.c_int32),
        ("coll_T_grid", C.POINTER(C.c_double)), ("coll_table", C.POINTER(C.c_double)),
        ("coll_partner_frac", C.POINTER(C.c_double)),
        ("coef_grid", C.c_int32), ("grid_n_density", C.c_int32), ("grid_n_temp", C.c_int32),
        ("grid_nH2_lo", C.c_double), ("grid_nH2_hi", C.c_double), ("grid_T_lo", C.c_double), ("grid_T_hi", C.c_double),
        ("dust_per_channel", C.c_int32),
    ]


def lib_path():
    return _LIB_PATH


def load_library():
    """Load libiris_so.so (built in-tree by paper_2607_01338_b200.build). Raises if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise IrisSOError(-1, "CUDA library %s is missing: run `python -m paper_2607_01338_b200.build` "
                              "(there is no CPU fallback)" % _LIB_PATH)
    lib = C.CDLL(_LIB_PATH)
    vp, fp, st = C.c_void_p, C.c_void_p, C.c_int
    lib.iris_so_create.restype = st
    lib.iris_so_create.argtypes = [C.POINTER(_Config), C.POINTER(vp)]
    lib.iris_so_destroy.restype = None
    lib.iris_so_destroy.argtypes = [vp]
    lib.iris_so_last_error.restype = C.c_char_p
    lib.iris_so_last_error.argtypes = [vp]
    lib.iris_so_status_string.restype = C.c_char_p
    lib.iris_so_status_string.argtypes = [st]
    lib.iris_so_version.restype = C.c_int
    lib.iris_so_launch_count.restype = C.c_uint64
    lib.iris_so_launch_count.argtypes = [vp]
    lib.iris_so_scratch_bytes.restype = C.c_uint64
    lib.iris_so_scratch_bytes.argtypes = [vp]
    lib.iris_so_levelpop.restype = st
    lib.iris_so_levelpop.argtypes = [vp, fp, fp, fp, vp]
    lib.iris_so_transfer.restype = st
    lib.iris_so_transfer.argtypes = [vp, fp, fp, fp, fp, fp, fp, fp, vp]
    lib.iris_so_observe.restype = st
    lib.iris_so_observe.argtypes = [vp, fp, fp, fp, fp, fp, vp]
    lib.iris_so_observe_stages.restype = st
    lib.iris_so_observe_stages.argtypes = [vp, fp, fp, fp, fp, C.c_int32, fp, vp]
    lib.iris_so_observe_host.restype = st
    lib.iris_so_observe_host.argtypes = [vp, fp, fp, fp, fp, fp, vp]
    lib.iris_so_observe_raw_static.restype = st
    lib.iris_so_observe_raw_static.argtypes = [vp, fp, fp, fp, fp, fp, vp]
    lib.iris_so_observe_adjoint.restype = st
    lib.iris_so_observe_adjoint.argtypes = [vp, fp, fp, fp, fp, fp, fp, vp]
    lib.iris_so_observe_adjoint_abundance.restype = st
    lib.iris_so_observe_adjoint_abundance.argtypes = [vp, fp, fp, fp, fp, fp, fp, vp]
    lib.iris_so_beam.restype = st
    lib.iris_so_beam.argtypes = [vp, fp, fp, fp, vp]
    lib.iris_so_noise.restype = st
    lib.iris_so_noise.argtypes = [vp, fp, vp]
    lib.iris_so_profile.restype = st
    lib.iris_so_profile.argtypes = [vp, C.c_int32]
    lib.iris_so_profile_read.restype = st
    lib.iris_so_profile_read.argtypes = [vp, C.c_int32, C.POINTER(C.c_double), C.POINTER(C.c_uint64)]
    lib.iris_so_transfer_kernel.restype = C.c_char_p
    lib.iris_so_transfer_kernel.argtypes = [vp]
    lib.iris_so_transfer_work.restype = st
    lib.iris_so_transfer_work.argtypes = [vp, C.POINTER(C.c_uint64), vp]
    lib.iris_so_smooth_fallback.restype = st
    lib.iris_so_smooth_fallback.argtypes = [vp, C.POINTER(C.c_int32), vp]
    lib.iris_so_density_trace.restype = st
    lib.iris_so_density_trace.argtypes = [vp, fp, fp, fp, vp]
    lib.iris_so_metrics.restype = st
    lib.iris_so_metrics.argtypes = [vp, fp, fp, C.c_double, C.POINTER(C.c_double), vp]
    _lib = lib
    return lib


def _make_config(cfg, transfer_algo):
    keep = [np.ascontiguousarray(np.asarray(getattr(cfg, k), dtype=np.float64))
            for k in ("energy_K", "weight", "einstein_A", "coll_down_ref")]
    s = _Config()
    table = getattr(cfg, "coll_table", None)
    if table is not None:
        tab = np.ascontiguousarray(np.asarray(table, dtype=np.float64))
        grid = np.ascontiguousarray(np.asarray(cfg.coll_T_grid, dtype=np.float64))
        frac = np.ascontiguousarray(np.asarray(cfg.coll_partner_frac, dtype=np.float64))
        n = len(keep[0])
        if tab.ndim != 4 or tab.shape[1:] != (grid.size, n, n) or frac.shape != (tab.shape[0],):
            raise ValueError("coll_table must be [P, nT, n_levels, n_levels] with coll_T_grid [nT], coll_partner_frac [P]")
        keep += [tab, grid, frac]
    for name, ctype in _Config._fields_:
        if name in ("energy_K", "weight", "einstein_A", "coll_down_ref", "coll_T_grid", "coll_table", "coll_partner_frac"):
            continue
        if name == "coll_n_partners":
            s.coll_n_partners = 0 if table is None else int(tab.shape[0])
        elif name == "coll_nT":
            s.coll_nT = 0 if table is None else int(grid.size)
        elif name == "n_levels":
            s.n_levels = len(keep[0])
        elif name == "transfer_algo":
            s.transfer_algo = int(transfer_algo)
        else:
            val = getattr(cfg, name, 0)
            setattr(s, name, float(val) if ctype is C.c_double else int(val))
    ptr = lambda a: a.ctypes.data_as(C.POINTER(C.c_double))
    s.energy_K, s.weight, s.einstein_A, s.coll_down_ref = (ptr(a) for a in keep[:4])
    if table is not None:
        s.coll_table, s.coll_T_grid, s.coll_partner_frac = (ptr(a) for a in keep[4:7])
    return s, keep


class IrisSO:
    """One iris_so_ctx.  Methods mirror the C entry points; tensors are float32 CUDA torch tensors."""

    def __init__(self, cfg, transfer_algo=ALGO_AUTO):
        self.lib = load_library()
        self.cfg = cfg
        s, keep = _make_config(cfg, transfer_algo)
        h = C.c_void_p()
        st = self.lib.iris_so_create(C.byref(s), C.byref(h))
        if st != 0:
            raise IrisSOError(st, self.lib.iris_so_last_error(None).decode())
        self._h = h
        self.n_levels = int(s.n_levels)
        self.shape_fields = (int(cfg.nz), int(cfg.ny), int(cfg.nx))
        self.shape_cube = (int(cfg.ny), int(cfg.nx), int(cfg.nv))

    def close(self):
        if getattr(self, "_h", None):
            self.lib.iris_so_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- helpers ---------------------------------------------------------------------------------
    def _check(self, st):
        if st != 0:
            raise IrisSOError(st, self.lib.iris_so_last_error(self._h).decode())

    @staticmethod
    def _stream():
        import torch
        return C.c_void_p(torch.cuda.current_stream().cuda_stream)

    def _dev(self, t, numel, what):
        import torch
        if t is None:
            return None
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()):
            raise TypeError("%s must be a contiguous float32 CUDA tensor" % what)
        if t.numel() != numel:
            raise ValueError("%s has %d elements, expected %d" % (what, t.numel(), numel))
        return C.c_void_p(t.data_ptr())

    @property
    def n_cells(self):
        return self.shape_fields[0] * self.shape_fields[1] * self.shape_fields[2]

    @property
    def n_vox(self):
        return self.shape_cube[0] * self.shape_cube[1] * self.shape_cube[2]

    def launch_count(self):
        return int(self.lib.iris_so_launch_count(self._h))

    def scratch_bytes(self):
        return int(self.lib.iris_so_scratch_bytes(self._h))

    def profile(self, enable=True):
        self._check(self.lib.iris_so_profile(self._h, 1 if enable else 0))

    def profile_read(self):
        """{stage: (total_ms, launches)} since profiling was switched on (waits for the recorded events)."""
        out = {}
        for name, sid in STAGES.items():
            ms, n = C.c_double(), C.c_uint64()
            self._check(self.lib.iris_so_profile_read(self._h, sid, C.byref(ms), C.byref(n)))
            out[name] = (ms.value, int(n.value))
        return out

    def transfer_kernel(self):
        """Name of the LOS transfer kernel this context launches."""
        return self.lib.iris_so_transfer_kernel(self._h).decode()

    def transfer_work(self):
        n = C.c_uint64()
        self._check(self.lib.iris_so_transfer_work(self._h, C.byref(n), self._stream()))
        return int(n.value)

    def smooth_fallback(self):
        """Number of pixels the last smooth-integrator call of this context handed over to the dense kernel."""
        n = C.c_int32()
        self._check(self.lib.iris_so_smooth_fallback(self._h, C.byref(n), self._stream()))
        return int(n.value)

    # -- entry points ----------------------------------------------------------------------------
    def levelpop(self, nH2, Tgas, pop=None):
        import torch
        n = nH2.numel()
        if n != self.n_cells:
            raise ValueError("field has %d cells, context expects %d" % (n, self.n_cells))
        if pop is None:
            pop = torch.empty((self.n_levels,) + tuple(nH2.shape), dtype=torch.float32, device=nH2.device)
        self._check(self.lib.iris_so_levelpop(self._h, self._dev(nH2, n, "nH2"), self._dev(Tgas, n, "Tgas"),
                                              self._dev(pop, n * self.n_levels, "pop"), self._stream()))
        return pop

    def transfer(self, nH2, Tgas, Tdust, vlos, pop=None, I_total=None, I_cont=None):
        import torch
        n = self.n_cells
        dev = nH2.device
        if I_total is None:
            I_total = torch.empty(self.shape_cube, dtype=torch.float32, device=dev)
        if I_cont is None and not getattr(self.cfg, "dust_per_channel", 0):     # (then the continuum is a spectrum: not returned)
            I_cont = torch.empty(self.shape_cube[:2], dtype=torch.float32, device=dev)
        self._check(self.lib.iris_so_transfer(
            self._h, self._dev(nH2, n, "nH2"), self._dev(Tgas, n, "Tgas"), self._dev(Tdust, n, "Tdust"),
            self._dev(vlos, n, "vlos"), self._dev(pop, n * self.n_levels, "pop"),
            self._dev(I_total, self.n_vox, "I_total"), self._dev(I_cont, self.n_vox // self.shape_cube[2], "I_cont"),
            self._stream()))
        return I_total, I_cont

    def observe(self, nH2, Tgas, Tdust, vlos, cube=None, beam=True, noise=True):
        import torch
        n = self.n_cells
        if cube is None:
            cube = torch.empty(self.shape_cube, dtype=torch.float32, device=nH2.device)
        args = [self._h, self._dev(nH2, n, "nH2"), self._dev(Tgas, n, "Tgas"), self._dev(Tdust, n, "Tdust"),
                self._dev(vlos, n, "vlos")]
        if beam and noise:
            st = self.lib.iris_so_observe(*args, self._dev(cube, self.n_vox, "cube"), self._stream())
        else:
            mask = (1 if beam else 0) | (2 if noise else 0)
            st = self.lib.iris_so_observe_stages(*args, C.c_int32(mask), self._dev(cube, self.n_vox, "cube"), self._stream())
        self._check(st)
        return cube

    def observe_raw_static(self, nH2, Tgas, Tdust, vlos, cube):
        """iris_so_observe_raw_static: K1 - K5 (no beam, no noise) of the hot-path mode with the library's static scratch; the
        library call allocates nothing, so the caller passes the output cube too."""
        n = self.n_cells
        self._check(self.lib.iris_so_observe_raw_static(
            self._h, self._dev(nH2, n, "nH2"), self._dev(Tgas, n, "Tgas"), self._dev(Tdust, n, "Tdust"),
            self._dev(vlos, n, "vlos"), self._dev(cube, self.n_vox, "cube"), self._stream()))
        return cube

    def observe_host(self, nH2, Tgas, Tdust, vlos, cube):
        """Host buffers (numpy arrays or CPU torch tensors, ideally pinned); synchronises."""
        def hp(a, numel, what):
            if hasattr(a, "data_ptr"):
                if a.is_cuda or str(a.dtype) != "torch.float32" or not a.is_contiguous() or a.numel() != numel:
                    raise TypeError("%s must be a contiguous float32 host tensor of %d elements" % (what, numel))
                return C.c_void_p(a.data_ptr())
            if a.dtype != np.float32 or not a.flags.c_contiguous or a.size != numel:
                raise TypeError("%s must be a C-contiguous float32 array of %d elements" % (what, numel))
            return C.c_void_p(a.ctypes.data)
        n = self.n_cells
        self._check(self.lib.iris_so_observe_host(self._h, hp(nH2, n, "nH2"), hp(Tgas, n, "Tgas"), hp(Tdust, n, "Tdust"),
                                                  hp(vlos, n, "vlos"), hp(cube, self.n_vox, "cube"), self._stream()))
        return cube

    def observe_adjoint(self, nH2, Tgas, Tdust, vlos, w, grad=None, wrt="nH2"):
        """d(sum w * cube) / d n_H2 per cell (wrt="nH2") or / d ln X per cell (wrt="abundance")."""
        import torch
        n = self.n_cells
        if grad is None:
            grad = torch.empty(self.shape_fields, dtype=torch.float32, device=nH2.device)
        fn = self.lib.iris_so_observe_adjoint if wrt == "nH2" else self.lib.iris_so_observe_adjoint_abundance
        self._check(fn(
            self._h, self._dev(nH2, n, "nH2"), self._dev(Tgas, n, "Tgas"), self._dev(Tdust, n, "Tdust"),
            self._dev(vlos, n, "vlos"), self._dev(w, self.n_vox, "w"), self._dev(grad, n, "grad"), self._stream()))
        return grad

    def beam(self, cube_in, cube_out=None, tmp=None):
        import torch
        if cube_out is None:
            cube_out = torch.empty_like(cube_in)
        self._check(self.lib.iris_so_beam(self._h, self._dev(cube_in, self.n_vox, "cube_in"),
                                          self._dev(cube_out, self.n_vox, "cube_out"),
                                          self._dev(tmp, self.n_vox, "tmp"), self._stream()))
        return cube_out

    def noise(self, cube):
        self._check(self.lib.iris_so_noise(self._h, self._dev(cube, self.n_vox, "cube"), self._stream()))
        return cube

    def density_trace(self, nH2, vlos, cube=None):
        """Column density per unit velocity (section 5.10), float32 CUDA tensor [ny, nx, nv]."""
        import torch
        if cube is None:
            cube = torch.empty(self.shape_cube, dtype=torch.float32, device=nH2.device)
        self._check(self.lib.iris_so_density_trace(self._h, self._dev(nH2, self.n_cells, "nH2"),
                                                   self._dev(vlos, self.n_cells, "vlos"),
                                                   self._dev(cube, self.n_vox, "cube"), self._stream()))
        return cube

    def metrics(self, T1, T2, T_min=5e-2):
        """Section 5.1 metrics of two cubes [ny, nx, nv]: dict of mean-TSRE (lbv, lb, lv), TAM, maxima, active counts."""
        out = (C.c_double * 9)()
        self._check(self.lib.iris_so_metrics(self._h, self._dev(T1, self.n_vox, "T1"), self._dev(T2, self.n_vox, "T2"),
                                             C.c_double(T_min), out, self._stream()))
        keys = ("tsre_lbv", "tsre_lb", "tsre_lv", "tam1", "tam2", "max1", "max2", "active1", "active2")
        return dict(zip(keys, [float(v) for v in out]))
