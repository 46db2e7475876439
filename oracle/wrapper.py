"""ORACLE -- test infrastructure only.  ctypes marshalling for oracle/iris_oracle.cpp.

The config argument is duck-typed (any object with the attribute names of the parameter record);
nothing here imports the CUDA package.
"""
import ctypes as C
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "iris_oracle.cpp")
# IRIS_ORACLE_LIB: an already built oracle library to load instead (the sanitizer build of tests/test_sanitizers.py)
_LIB = os.environ.get("IRIS_ORACLE_LIB") or os.path.join(_HERE, "liboracle.so")
_lock = threading.Lock()


def oracle_lib_path():
    return _LIB


def build_oracle(force=False):
    """Compile the oracle with g++ -O2 (+OpenMP over cells / pixel columns). Returns the .so path."""
    with _lock:
        if os.environ.get("IRIS_ORACLE_LIB"):
            return _LIB
        if (not force and os.path.exists(_LIB)
                and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
            return _LIB
        tmp = _LIB + ".tmp%d" % os.getpid()
        cmd = ["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
               "-o", tmp, _SRC]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
        return _LIB


class _Cfg(C.Structure):
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
        ("transfer_mode", C.c_int32), ("integration", C.c_int32), ("subsample", C.c_int32),
        ("coll_n_partners", C.c_int32), ("coll_nT", C.c_int32),
        ("coll_T_grid", C.POINTER(C.c_double)), ("coll_table", C.POINTER(C.c_double)),
        ("coll_partner_frac", C.POINTER(C.c_double)),
        ("coef_grid", C.c_int32), ("grid_n_density", C.c_int32), ("grid_n_temp", C.c_int32),
        ("grid_nH2_lo", C.c_double), ("grid_nH2_hi", C.c_double), ("grid_T_lo", C.c_double), ("grid_T_hi", C.c_double),
        ("dust_per_channel", C.c_int32),
    ]


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _fp(a):
    return a.ctypes.data_as(C.POINTER(C.c_float))


def _ip(a):
    return a.ctypes.data_as(C.POINTER(C.c_int64))


def _f32(a):
    a = np.ascontiguousarray(a, dtype=np.float32)
    return a


class Oracle:
    """One parameter record bound to the oracle library."""

    def __init__(self, cfg, threads=None):
        self.lib = C.CDLL(build_oracle())
        self.cfg = cfg
        self._keep = [np.ascontiguousarray(np.asarray(getattr(cfg, k), dtype=np.float64))
                      for k in ("energy_K", "weight", "einstein_A", "coll_down_ref")]
        s = _Cfg()
        table = getattr(cfg, "coll_table", None)
        if table is not None:
            tab = np.ascontiguousarray(np.asarray(table, dtype=np.float64))
            grid = np.ascontiguousarray(np.asarray(cfg.coll_T_grid, dtype=np.float64))
            frac = np.ascontiguousarray(np.asarray(cfg.coll_partner_frac, dtype=np.float64))
            n = len(self._keep[0])
            assert tab.ndim == 4 and tab.shape[1:] == (grid.size, n, n) and frac.shape == (tab.shape[0],)
            self._keep += [tab, grid, frac]
        for name, ctype in _Cfg._fields_:
            if name in ("energy_K", "weight", "einstein_A", "coll_down_ref", "coll_T_grid", "coll_table",
                        "coll_partner_frac"):
                continue
            if name == "coll_n_partners":
                s.coll_n_partners = 0 if table is None else int(tab.shape[0])
                continue
            if name == "coll_nT":
                s.coll_nT = 0 if table is None else int(grid.size)
                continue
            if name == "n_levels":
                s.n_levels = len(self._keep[0])
                continue
            val = getattr(cfg, name)
            setattr(s, name, float(val) if ctype is C.c_double else int(val))
        s.energy_K, s.weight, s.einstein_A, s.coll_down_ref = (_dp(a) for a in self._keep[:4])
        if table is not None:
            s.coll_table, s.coll_T_grid, s.coll_partner_frac = (_dp(a) for a in self._keep[4:7])
        self.s = s
        self.N = int(s.n_levels)
        self.threads = threads
        L = self.lib
        L.orc_planck.restype = C.c_double
        L.orc_planck.argtypes = [C.c_double, C.c_double]
        L.orc_planck_TB.restype = C.c_double
        L.orc_planck_TB.argtypes = [C.c_double, C.c_double]
        L.orc_rayleigh_jeans_T.restype = C.c_double
        L.orc_rayleigh_jeans_T.argtypes = [C.c_double, C.c_double]
        L.orc_phibar.restype = C.c_double
        L.orc_phibar.argtypes = [C.c_void_p, C.c_int, C.c_double, C.c_double]
        L.orc_phi_point.restype = C.c_double
        L.orc_phi_point.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_double]
        L.orc_normal.restype = C.c_double
        L.orc_normal.argtypes = [C.c_uint64, C.c_uint64]
        L.orc_noise_gamma.restype = C.c_double
        L.orc_beam_radius.restype = C.c_int
        L.orc_beam_radius.argtypes = [C.c_double]

    # -- helpers ---------------------------------------------------------------------------------
    def _p(self):
        return C.byref(self.s)

    def _omp(self):
        if self.threads is not None:
            try:
                omp = C.CDLL("libgomp.so.1")
                omp.omp_set_num_threads(int(self.threads))
            except OSError:
                pass

    @property
    def n_cells(self):
        return int(self.s.nx) * int(self.s.ny) * int(self.s.nz)

    # -- scalar functions ------------------------------------------------------------------------
    def planck(self, nu, T):
        return self.lib.orc_planck(float(nu), float(T))

    def planck_TB(self, nu, I):
        return self.lib.orc_planck_TB(float(nu), float(I))

    def rayleigh_jeans_T(self, nu, I):
        return self.lib.orc_rayleigh_jeans_T(float(nu), float(I))

    def phibar(self, k, vlos, b):
        return self.lib.orc_phibar(self._p(), int(k), float(vlos), float(b))

    def phi_point(self, v, vlos, b):
        return self.lib.orc_phi_point(self._p(), float(v), float(vlos), float(b))

    def normal(self, seed, voxel):
        return self.lib.orc_normal(int(seed), int(voxel))

    def philox(self, seed, ctr_lo, ctr_hi=0):
        out = (C.c_uint32 * 4)()
        self.lib.orc_philox4x32_10(C.c_uint64(seed), C.c_uint64(ctr_lo), C.c_uint64(ctr_hi), out)
        return [int(v) for v in out]

    def noise_gamma(self):
        self.lib.orc_noise_gamma.argtypes = [C.c_void_p]
        return self.lib.orc_noise_gamma(self._p())

    def beam_weights(self, fwhm):
        R = self.lib.orc_beam_radius(float(fwhm))
        g = np.zeros(2 * R + 1)
        self.lib.orc_beam_weights(C.c_double(fwhm), _dp(g))
        return g

    # -- level balance ---------------------------------------------------------------------------
    def rates(self, nH2, Tgas):
        R = np.zeros((self.N, self.N))
        self.lib.orc_rates(self._p(), C.c_double(nH2), C.c_double(Tgas), _dp(R))
        return R

    def balance_matrix(self, nH2, Tgas):
        M = np.zeros((self.N, self.N))
        self.lib.orc_balance_matrix(self._p(), C.c_double(nH2), C.c_double(Tgas), _dp(M))
        return M

    def levelpop_cell(self, nH2, Tgas):
        x = np.zeros(self.N)
        self.lib.orc_levelpop_cell(self._p(), C.c_double(nH2), C.c_double(Tgas), _dp(x))
        return x

    def levelpop(self, nH2, Tgas):
        """pop[N, ncell] (float64) for flat float32 arrays of cells."""
        self._omp()
        nH2, Tgas = _f32(nH2).ravel(), _f32(Tgas).ravel()
        pop = np.zeros((self.N, nH2.size))
        self.lib.orc_levelpop(self._p(), C.c_int64(nH2.size), _fp(nH2), _fp(Tgas), _dp(pop))
        return pop

    # -- coefficients ----------------------------------------------------------------------------
    def coefficients(self, nH2, Tgas, Tdust, pop=None):
        """coef[5, ncell] = j0, kappa0, b, alpha_d, S_d."""
        self._omp()
        nH2, Tgas, Tdust = _f32(nH2).ravel(), _f32(Tgas).ravel(), _f32(Tdust).ravel()
        coef = np.zeros((5, nH2.size))
        pp = None
        if pop is not None:
            pop = np.ascontiguousarray(pop, dtype=np.float64)
            pp = _dp(pop)
        self.lib.orc_coefficients(self._p(), C.c_int64(nH2.size), _fp(nH2), _fp(Tgas), _fp(Tdust), pp, _dp(coef))
        return coef

    # -- coefficient grid (sections 4.2 - 4.3) ---------------------------------------------------
    def grid_build(self):
        """grid[2, nT, nn]: j0 / X and kappa0 / X at the nodes."""
        self._omp()
        g = np.zeros((2, int(self.s.grid_n_temp), int(self.s.grid_n_density)))
        self.lib.orc_grid_build(self._p(), _dp(g))
        return g

    def grid_nodes(self):
        f = self.lib.orc_grid_node
        f.restype = C.c_double
        f.argtypes = [C.c_double, C.c_double, C.c_int, C.c_int]
        nn, nT = int(self.s.grid_n_density), int(self.s.grid_n_temp)
        return (np.array([f(self.s.grid_nH2_lo, self.s.grid_nH2_hi, nn, i) for i in range(nn)]),
                np.array([f(self.s.grid_T_lo, self.s.grid_T_hi, nT, j) for j in range(nT)]))

    def grid_lookup_plane(self, plane, nH2, Tgas):
        """Multilinear interpolation / extrapolation of one plane [nT, nn] at (nH2, Tgas)."""
        f = self.lib.orc_grid_lookup_plane
        f.restype = C.c_double
        f.argtypes = [C.POINTER(C.c_double), C.c_int, C.c_int] + [C.c_double] * 6
        plane = np.ascontiguousarray(plane, dtype=np.float64)
        nT, nn = plane.shape
        return f(_dp(plane), nn, nT, self.s.grid_nH2_lo, self.s.grid_nH2_hi, self.s.grid_T_lo, self.s.grid_T_hi,
                 float(nH2), float(Tgas))

    # -- transfer --------------------------------------------------------------------------------
    def march(self, coef, vlos, pix=None):
        """I_tot[npix, nv], I_cont[npix] for the listed pixel columns (all if None)."""
        self._omp()
        coef = np.ascontiguousarray(coef, dtype=np.float64)
        vlos = _f32(vlos).ravel()
        assert coef.shape == (5, self.n_cells) and vlos.size == self.n_cells
        plane = int(self.s.nx) * int(self.s.ny)
        pix = np.arange(plane, dtype=np.int64) if pix is None else np.ascontiguousarray(pix, dtype=np.int64)
        It = np.zeros((pix.size, int(self.s.nv)))
        Ic = np.zeros(pix.size)
        self.lib.orc_march(self._p(), _dp(coef), _fp(vlos), C.c_int64(pix.size), _ip(pix), _dp(It), _dp(Ic))
        return It, Ic

    def march_perchannel(self, coef, vlos, Tdust, pix=None):
        """Hot-path march with the dust source / background at every channel's own frequency: I_tot[npix, nv], I_cont[npix, nv]."""
        self._omp()
        coef = np.ascontiguousarray(coef, dtype=np.float64)
        vlos, Tdust = _f32(vlos).ravel(), _f32(Tdust).ravel()
        plane = int(self.s.nx) * int(self.s.ny)
        pix = np.arange(plane, dtype=np.int64) if pix is None else np.ascontiguousarray(pix, dtype=np.int64)
        It = np.zeros((pix.size, int(self.s.nv)))
        Ic = np.zeros((pix.size, int(self.s.nv)))
        self.lib.orc_march_perchannel(self._p(), _dp(coef), _fp(vlos), _fp(Tdust), C.c_int64(pix.size), _ip(pix), _dp(It), _dp(Ic))
        return It, Ic

    def channel_frequency(self, k):
        f = self.lib.orc_channel_frequency
        f.restype = C.c_double
        f.argtypes = [C.c_void_p, C.c_int]
        return f(self._p(), int(k))

    def brute_column(self, coef, vlos, pix, nsub):
        coef = np.ascontiguousarray(coef, dtype=np.float64)
        vlos = _f32(vlos).ravel()
        out = np.zeros(int(self.s.nv))
        self.lib.orc_brute_column(self._p(), _dp(coef), _fp(vlos), C.c_int64(pix), C.c_int(nsub), _dp(out))
        return out

    def convert(self, I_tot, I_cont):
        I_tot = np.ascontiguousarray(I_tot, dtype=np.float64)
        I_cont = np.ascontiguousarray(I_cont, dtype=np.float64)
        cube = np.zeros_like(I_tot)
        self.lib.orc_convert(self._p(), C.c_int64(I_cont.size), _dp(I_tot), _dp(I_cont), _dp(cube))
        return cube

    # -- post-processing -------------------------------------------------------------------------
    def beam(self, cube, fwhm=None):
        self._omp()
        cube = np.ascontiguousarray(cube, dtype=np.float64)
        ny, nx, nv = cube.shape
        out = np.zeros_like(cube)
        fwhm = float(self.s.beam_fwhm_px if fwhm is None else fwhm)
        self.lib.orc_beam(C.c_int(ny), C.c_int(nx), C.c_int(nv), C.c_double(fwhm), _dp(cube), _dp(out))
        return out

    def noise(self, cube):
        cube = np.array(cube, dtype=np.float64, order="C", copy=True)
        self.lib.orc_noise(self._p(), C.c_int64(cube.size), _dp(cube))
        return cube

    def observe(self, fields, beam=True, noise=True):
        """Whole path; cube[ny, nx, nv] float64."""
        self._omp()
        f = [_f32(fields[k]).ravel() for k in ("nH2", "Tgas", "Tdust", "vlos")]
        assert all(a.size == self.n_cells for a in f)
        cube = np.zeros((int(self.s.ny), int(self.s.nx), int(self.s.nv)))
        mask = (1 if beam else 0) | (2 if noise else 0)
        self.lib.orc_observe(self._p(), *[_fp(a) for a in f], C.c_int(mask), _dp(cube))
        return cube

    # -- diagnostics (sections 5.1, 5.10) ---------------------------------------------------------
    def density_trace(self, fields):
        """Column density per unit velocity, cube[ny, nx, nv] float64 (cm^-2 per cm/s)."""
        n, v = _f32(fields["nH2"]).ravel(), _f32(fields["vlos"]).ravel()
        cube = np.zeros((int(self.s.ny), int(self.s.nx), int(self.s.nv)))
        self.lib.orc_density_trace(self._p(), _fp(n), _fp(v), _dp(cube))
        return cube

    def metrics(self, T1, T2, T_min=5e-2):
        """dict of mean-TSRE (lbv, lb, lv), TAM, maxima and active counts of two cubes [ny, nx, nv]."""
        a = np.ascontiguousarray(T1, dtype=np.float64)
        b = np.ascontiguousarray(T2, dtype=np.float64)
        assert a.shape == b.shape and a.ndim == 3
        out = np.zeros(9)
        self.lib.orc_metrics(C.c_int(a.shape[0]), C.c_int(a.shape[1]), C.c_int(a.shape[2]), _dp(a), _dp(b),
                             C.c_double(T_min), _dp(out))
        keys = ("tsre_lbv", "tsre_lb", "tsre_lv", "tam1", "tam2", "max1", "max2", "active1", "active2")
        return dict(zip(keys, out.tolist()))

    # -- gradient --------------------------------------------------------------------------------
    def grad_fd(self, fields, what, cells, eps=1e-4, wrt="nH2"):
        """Central finite differences of L = sum(what * raw cube) w.r.t. n_H2 of the listed cells (wrt="nH2") or
        w.r.t. the logarithm of a per-cell factor on the tracer abundance (wrt="abundance")."""
        self._omp()
        f = [_f32(fields[k]).ravel() for k in ("nH2", "Tgas", "Tdust", "vlos")]
        what = np.ascontiguousarray(what, dtype=np.float64)
        cells = np.ascontiguousarray(cells, dtype=np.int64)
        g = np.zeros(cells.size)
        fn = self.lib.orc_grad_fd if wrt == "nH2" else self.lib.orc_grad_fd_abundance
        fn(self._p(), *[_fp(a) for a in f], _dp(what), C.c_int64(cells.size), _ip(cells), C.c_double(eps), _dp(g))
        return g

    def grad_adjoint(self, fields, what, wrt="nH2"):
        self._omp()
        f = [_f32(fields[k]).ravel() for k in ("nH2", "Tgas", "Tdust", "vlos")]
        what = np.ascontiguousarray(what, dtype=np.float64)
        g = np.zeros(self.n_cells)
        fn = self.lib.orc_grad_adjoint if wrt == "nH2" else self.lib.orc_grad_adjoint_abundance
        fn(self._p(), *[_fp(a) for a in f], _dp(what), _dp(g))
        return g.reshape(int(self.s.nz), int(self.s.ny), int(self.s.nx))
