"""ctypes front end of the CPU oracle (oracle/rmhd_oracle.cpp).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It imports nothing from the CUDA package.

All arrays are float64, variable-major SoA: batches ``a[var, cell]``, grids ``a[var, k, j, i]``
(x fastest), interior cells only.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

RESISTIVE, TWO_FLUID = 0, 1
BC_OUTFLOW, BC_PERIODIC = 0, 1
NCONS = {0: 14, 1: 18}
NPRIM = {0: 11, 1: 16}


class OracleParams(C.Structure):
    _fields_ = [
        ("model", C.c_int), ("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int), ("ng", C.c_int),
        ("xmin", C.c_double), ("xmax", C.c_double), ("ymin", C.c_double), ("ymax", C.c_double),
        ("zmin", C.c_double), ("zmax", C.c_double),
        ("bc", C.c_int * 3),
        ("gamma", C.c_double), ("sigma", C.c_double), ("eta", C.c_double), ("mu_e", C.c_double),
        ("mu_p", C.c_double), ("kappa", C.c_double), ("cfl", C.c_double), ("tol_c2p", C.c_double),
        ("tol_stage", C.c_double),
        ("max_iter_c2p", C.c_int), ("max_iter_stage", C.c_int), ("integrator", C.c_int),
    ]


def make_params(model=0, nx=1, ny=1, nz=1, ng=4, xlim=(0.0, 1.0), ylim=(0.0, 1.0), zlim=(0.0, 1.0),
                bc=(0, 0, 0), gamma=4.0 / 3.0, sigma=0.0, eta=0.0, mu_e=-1.0, mu_p=1.0, kappa=1.0, cfl=0.4,
                tol_c2p=1e-13, tol_stage=1e-12, max_iter_c2p=100, max_iter_stage=50, integrator=0, **_ignored):
    p = OracleParams()
    p.model, p.nx, p.ny, p.nz, p.ng = model, nx, ny, nz, ng
    p.xmin, p.xmax = xlim
    p.ymin, p.ymax = ylim
    p.zmin, p.zmax = zlim
    p.bc = (C.c_int * 3)(*bc)
    p.gamma, p.sigma, p.eta, p.mu_e, p.mu_p, p.kappa, p.cfl = gamma, sigma, eta, mu_e, mu_p, kappa, cfl
    p.tol_c2p, p.tol_stage = tol_c2p, tol_stage
    p.max_iter_c2p, p.max_iter_stage = max_iter_c2p, max_iter_stage
    p.integrator = {"ssp2": 0, "ssp3": 1}.get(integrator, integrator)   # 2 = SSP2(222) via the general stepper (tests)
    return p


_lib = None
_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int)
_lp = C.POINTER(C.c_longlong)


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        L.oracle_create.restype = C.c_void_p
        L.oracle_create.argtypes = [C.POINTER(OracleParams)]
        L.oracle_destroy.argtypes = [C.c_void_p]
        L.oracle_dt.restype = C.c_double
        L.oracle_dt.argtypes = [C.c_void_p]
        L.oracle_time.restype = C.c_double
        L.oracle_time.argtypes = [C.c_void_p]
        L.oracle_set_initial.argtypes = [C.c_void_p, _dp, _dp]
        L.oracle_set_cons.argtypes = [C.c_void_p, _dp, _dp]
        L.oracle_step.argtypes = [C.c_void_p, C.c_int]
        L.oracle_get_state.argtypes = [C.c_void_p, _dp, _dp]
        L.oracle_eval_L.argtypes = [C.c_void_p, _dp]
        L.oracle_get_stats.argtypes = [C.c_void_p, _lp, _lp, C.c_int, _lp, _lp]
        L.oracle_set_threads.argtypes = [C.c_int]
        L.oracle_set_c2p_switch.argtypes = [C.c_int]
        L.oracle_prim2cons_batch.argtypes = [C.POINTER(OracleParams), C.c_longlong, _dp, _dp, _dp]
        L.oracle_con2prim_batch.argtypes = [C.POINTER(OracleParams), C.c_longlong, _dp, _dp, _dp, _ip, _ip]
        L.oracle_flux_vector_batch.argtypes = [C.POINTER(OracleParams), C.c_longlong, C.c_int, _dp, _dp, _dp, _dp]
        L.oracle_source_batch.argtypes = [C.POINTER(OracleParams), C.c_longlong, _dp, _dp, _dp, _dp]
        L.oracle_species_split.argtypes = [C.c_double, C.c_double, C.c_longlong, _dp, _dp, _dp, _dp]
        L.oracle_weno3.argtypes = [C.c_longlong, _dp, _dp, _dp, _dp]
        L.oracle_stage_guess_batch.argtypes = [C.POINTER(OracleParams), C.c_longlong, _dp, _dp, _dp, C.c_double, _dp]
        L.oracle_stage_batch.argtypes = [C.POINTER(OracleParams), C.c_longlong, _dp, _dp, _dp, C.c_double, _dp, _dp,
                                         _ip, _ip]
        L.oracle_stage_residual_batch.argtypes = [C.POINTER(OracleParams), C.c_longlong, _dp, _dp, _dp, C.c_double,
                                                  _dp, _ip]
        _lib = L
    return _lib


def _d(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _c(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def set_threads(n=0):
    """n > 0 sets the OpenMP thread count; returns the count in force."""
    return lib().oracle_set_threads(int(n))


def set_c2p_switch(n=20):
    """Iterations of the first con2prim residual before the second (quartic in W) takes over; 0 = second only.  Returns the previous value."""
    return lib().oracle_set_c2p_switch(int(n))


# ---- batched per-cell operations -------------------------------------------------------
def prim2cons(params, prims, rho_charge=None):
    prims = _c(prims); rho_charge = _c(rho_charge)
    n = prims.shape[1]
    cons = np.empty((NCONS[params.model], n))
    lib().oracle_prim2cons_batch(C.byref(params), n, _d(prims), _d(rho_charge), _d(cons))
    return cons


def con2prim(params, cons, prim_guess=None):
    cons = _c(cons); prim_guess = _c(prim_guess)
    n = cons.shape[1]
    prims = np.empty((NPRIM[params.model], n))
    iters = np.zeros(n, dtype=np.int32); fail = np.zeros(n, dtype=np.int32)
    lib().oracle_con2prim_batch(C.byref(params), n, _d(cons), _d(prim_guess), _d(prims),
                                iters.ctypes.data_as(_ip), fail.ctypes.data_as(_ip))
    return prims, iters, fail


def flux_vector(params, direction, cons, prims, sigma_cell=None):
    cons = _c(cons); prims = _c(prims); sigma_cell = _c(sigma_cell)
    n = cons.shape[1]
    f = np.empty_like(cons)
    lib().oracle_flux_vector_batch(C.byref(params), n, int(direction), _d(cons), _d(prims), _d(sigma_cell), _d(f))
    return f


def source(params, cons, prims, sigma_cell=None):
    cons = _c(cons); prims = _c(prims); sigma_cell = _c(sigma_cell)
    n = cons.shape[1]
    s = np.empty_like(cons)
    lib().oracle_source_batch(C.byref(params), n, _d(cons), _d(prims), _d(sigma_cell), _d(s))
    return s


def species_split(mu_e, mu_p, x, xbar):
    x = _c(x); xbar = _c(xbar)
    xe = np.empty_like(x); xp = np.empty_like(x)
    rc = lib().oracle_species_split(mu_e, mu_p, x.size, _d(x), _d(xbar), _d(xe), _d(xp))
    if rc:
        raise ValueError("mu_e == mu_p")
    return xe, xp


def weno3(a, b, c):
    a = _c(a); b = _c(b); c = _c(c)
    out = np.empty_like(a)
    lib().oracle_weno3(a.size, _d(a), _d(b), _d(c), _d(out))
    return out


def stage_guess(params, q_ex, prim_guess, a_dt, sigma_cell=None):
    q_ex = _c(q_ex); prim_guess = _c(prim_guess); sigma_cell = _c(sigma_cell)
    n = q_ex.shape[1]
    Eg = np.empty((3, n))
    lib().oracle_stage_guess_batch(C.byref(params), n, _d(q_ex), _d(prim_guess), _d(sigma_cell), a_dt, _d(Eg))
    return Eg


def stage_batch(params, q_ex, prim_guess, a_dt, sigma_cell=None):
    """One implicit stage  q* - q_ex - a_dt Psi(q*) = 0  on independent cells."""
    q_ex = _c(q_ex); prim_guess = _c(prim_guess); sigma_cell = _c(sigma_cell)
    n = q_ex.shape[1]
    q = np.empty_like(q_ex); w = np.empty((NPRIM[params.model], n))
    iters = np.zeros(n, dtype=np.int32); fail = np.zeros(n, dtype=np.int32)
    lib().oracle_stage_batch(C.byref(params), n, _d(q_ex), _d(prim_guess), _d(sigma_cell), a_dt, _d(q), _d(w),
                             iters.ctypes.data_as(_ip), fail.ctypes.data_as(_ip))
    return q, w, iters, fail


def stage_residual(params, q, q_ex, a_dt, sigma_cell=None):
    q = _c(q); q_ex = _c(q_ex); sigma_cell = _c(sigma_cell)
    n = q.shape[1]
    R = np.empty_like(q); fail = np.zeros(n, dtype=np.int32)
    lib().oracle_stage_residual_batch(C.byref(params), n, _d(q), _d(q_ex), _d(sigma_cell), a_dt, _d(R),
                                      fail.ctypes.data_as(_ip))
    return R, fail


# ---- grid simulation -----------------------------------------------------------------------
class OracleSim:
    """One grid, one model: set_initial / step / get_state (mirrors the rmhd_* C-ABI)."""

    def __init__(self, params):
        self.params = params
        self._h = lib().oracle_create(C.byref(params))
        if not self._h:
            raise ValueError("oracle_create: bad parameters")
        self.shape = (params.nz, params.ny, params.nx)
        self.nc, self.np_ = NCONS[params.model], NPRIM[params.model]

    def close(self):
        if self._h:
            lib().oracle_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def dt(self):
        return lib().oracle_dt(self._h)

    @property
    def time(self):
        return lib().oracle_time(self._h)

    def set_initial(self, prims, rho_charge=None):
        prims = _c(prims).reshape((self.np_,) + self.shape)
        rho_charge = _c(rho_charge)
        return lib().oracle_set_initial(self._h, _d(prims), _d(rho_charge))

    def set_cons(self, cons, prim_guess=None):
        cons = _c(cons).reshape((self.nc,) + self.shape)
        prim_guess = _c(prim_guess)
        return lib().oracle_set_cons(self._h, _d(cons), _d(prim_guess))

    def step(self, n=1):
        return lib().oracle_step(self._h, int(n))

    def get_state(self):
        cons = np.empty((self.nc,) + self.shape); prims = np.empty((self.np_,) + self.shape)
        lib().oracle_get_state(self._h, _d(cons), _d(prims))
        return cons, prims

    def eval_L(self):
        L = np.empty((self.nc,) + self.shape)
        lib().oracle_eval_L(self._h, _d(L))
        return L

    def get_stats(self, nbins=64):
        hs = np.zeros(nbins, dtype=np.int64); hc = np.zeros(nbins, dtype=np.int64)
        nf = C.c_longlong(0); ff = C.c_longlong(-1)
        lib().oracle_get_stats(self._h, hs.ctypes.data_as(_lp), hc.ctypes.data_as(_lp), nbins, C.byref(nf), C.byref(ff))
        return {"hist_stage": hs, "hist_c2p": hc, "n_failed": nf.value, "first_failed_cell": ff.value}
