"""Thin ctypes binding of librmhd.so (include/rmhd.h): argument marshalling only.

Every step of the path runs in the library's CUDA kernels.  PyTorch is used for device
memory (``tensor.data_ptr()``) and for the stream the kernels are launched on.  There is no
CPU fallback: if the library cannot be loaded, or there is no CUDA device, calls raise.

Buffers may be ``torch`` CUDA tensors (``on_device=1``), or host ``numpy`` arrays / CPU
tensors (``on_device=0``: the library copies host<->device inside the call).  All float64,
C-contiguous, variable-major SoA (see include/rmhd.h).
"""
import ctypes as C
import os

import numpy as np

RMHD_RESISTIVE, RMHD_TWO_FLUID = 0, 1
RMHD_BC_OUTFLOW, RMHD_BC_PERIODIC = 0, 1
RMHD_OK, RMHD_ERR_BAD_PARAM, RMHD_ERR_CUDA, RMHD_ERR_NONCONVERGED, RMHD_ERR_UNPHYSICAL_INPUT = 0, -1, -2, -3, -4
NCONS = {0: 14, 1: 18}
NPRIM = {0: 11, 1: 16}
NHYD = {0: 5, 1: 10}     # hydro primitive rows (rho, v, p per species); B, E follow
KERNEL_CLASSES = ("stage1", "stage2", "flux", "combine_c2p", "other")

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("RMHD_LIB") or os.path.join(_HERE, "librmhd.so")   # RMHD_LIB: an alternative build of the same library

EXPORTS = (
    "rmhd_create", "rmhd_set_initial", "rmhd_set_cons", "rmhd_step", "rmhd_get_state", "rmhd_flux_divergence",
    "rmhd_get_stats", "rmhd_set_profiling", "rmhd_get_kernel_times", "rmhd_dt", "rmhd_time", "rmhd_last_error",
    "rmhd_destroy", "rmhd_stage_batch", "rmhd_prim2cons_batch", "rmhd_con2prim_batch", "rmhd_probe_fp64",
    "rmhd_probe_hbm", "rmhd_flux_divergence_static", "rmhd_release_staging",
)
RMHD_STATIC_MAX_CELLS = 262144   # include/rmhd.h: capacity of the library's fixed scratch array (rmhd_flux_divergence_static)


class RmhdError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"rmhd error {code}: {msg}")
        self.code = code


class rmhd_params(C.Structure):
    _fields_ = [
        ("model", C.c_int), ("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int), ("ng", C.c_int),
        ("xmin", C.c_double), ("xmax", C.c_double), ("ymin", C.c_double), ("ymax", C.c_double),
        ("zmin", C.c_double), ("zmax", C.c_double),
        ("bc", C.c_int * 3),
        ("gamma", C.c_double), ("sigma", C.c_double), ("eta", C.c_double), ("mu_e", C.c_double), ("mu_p", C.c_double),
        ("kappa", C.c_double), ("cfl", C.c_double), ("tol_c2p", C.c_double), ("tol_stage", C.c_double),
        ("max_iter_c2p", C.c_int), ("max_iter_stage", C.c_int),
        ("device", C.c_int), ("stream", C.c_void_p), ("integrator", C.c_int),
    ]


def make_params(model=0, nx=1, ny=1, nz=1, ng=4, xlim=(0.0, 1.0), ylim=(0.0, 1.0), zlim=(0.0, 1.0), bc=(0, 0, 0),
                gamma=4.0 / 3.0, sigma=0.0, eta=0.0, mu_e=-1.0, mu_p=1.0, kappa=1.0, cfl=0.4, tol_c2p=1e-13,
                tol_stage=1e-12, max_iter_c2p=100, max_iter_stage=50, device=0, stream=None, integrator=0, **_ignored):
    p = rmhd_params()
    p.model, p.nx, p.ny, p.nz, p.ng = model, nx, ny, nz, ng
    p.xmin, p.xmax = xlim
    p.ymin, p.ymax = ylim
    p.zmin, p.zmax = zlim
    p.bc = (C.c_int * 3)(*bc)
    p.gamma, p.sigma, p.eta, p.mu_e, p.mu_p, p.kappa, p.cfl = gamma, sigma, eta, mu_e, mu_p, kappa, cfl
    p.tol_c2p, p.tol_stage, p.max_iter_c2p, p.max_iter_stage = tol_c2p, tol_stage, max_iter_c2p, max_iter_stage
    p.device = device
    p.stream = _current_stream(device) if stream is None else stream
    p.integrator = {"ssp2": 0, "ssp3": 1}.get(integrator, integrator)
    return p


def _current_stream(device):
    """The torch current CUDA stream handle (0 = default stream if torch has no CUDA)."""
    try:
        import torch
        if torch.cuda.is_available():
            return torch.cuda.current_stream(device).cuda_stream
    except Exception:
        pass
    return 0


_lib = None
_dp, _ip, _lp = C.POINTER(C.c_double), C.POINTER(C.c_int), C.POINTER(C.c_longlong)


def lib():
    """Load librmhd.so; raises if it is missing (no fallback)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RmhdError(RMHD_ERR_CUDA, f"{LIB_PATH} is not built: run `python -m paper_1808_09721_b200.build` "
                                       "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    pp = C.POINTER(rmhd_params)
    vp = C.c_void_p
    L.rmhd_create.argtypes = [pp, C.POINTER(vp)]
    L.rmhd_set_initial.argtypes = [vp, vp, vp, C.c_int]
    L.rmhd_set_cons.argtypes = [vp, vp, vp, C.c_int]
    L.rmhd_step.argtypes = [vp, C.c_int]
    L.rmhd_get_state.argtypes = [vp, vp, vp, C.c_int]
    L.rmhd_flux_divergence.argtypes = [vp, vp, C.c_int]
    L.rmhd_get_stats.argtypes = [vp, _lp, _lp, C.c_int, _lp, _lp]
    L.rmhd_set_profiling.argtypes = [vp, C.c_int]
    L.rmhd_get_kernel_times.argtypes = [vp, _dp, _lp, C.c_int]
    L.rmhd_dt.argtypes = [vp]
    L.rmhd_dt.restype = C.c_double
    L.rmhd_time.argtypes = [vp]
    L.rmhd_time.restype = C.c_double
    L.rmhd_last_error.argtypes = [vp]
    L.rmhd_last_error.restype = C.c_char_p
    L.rmhd_destroy.argtypes = [vp]
    L.rmhd_destroy.restype = None
    L.rmhd_stage_batch.argtypes = [pp, C.c_longlong, vp, vp, vp, C.c_double, vp, vp, vp, vp, C.c_int]
    L.rmhd_prim2cons_batch.argtypes = [pp, C.c_longlong, vp, vp, vp, C.c_int]
    L.rmhd_con2prim_batch.argtypes = [pp, C.c_longlong, vp, vp, vp, vp, vp, C.c_int]
    L.rmhd_probe_fp64.argtypes = [C.c_int, vp, _dp]
    L.rmhd_probe_hbm.argtypes = [C.c_int, vp, C.c_longlong, _dp]
    L.rmhd_flux_divergence_static.argtypes = [pp, vp, vp, _lp]
    L.rmhd_release_staging.argtypes = [C.c_int]
    _lib = L
    return L


def _is_torch(x):
    return type(x).__module__.startswith("torch")


def _ptr(x, dtype=np.float64):
    """(pointer, on_device) of a torch tensor / numpy array (None -> (None, None))."""
    if x is None:
        return None, None
    if _is_torch(x):
        import torch
        want = {np.float64: torch.float64, np.int32: torch.int32}[dtype]
        if x.dtype != want or not x.is_contiguous():
            raise ValueError("tensor must be contiguous and of dtype %s" % want)
        return x.data_ptr(), 1 if x.is_cuda else 0
    if not isinstance(x, np.ndarray) or x.dtype != dtype or not x.flags["C_CONTIGUOUS"]:
        raise ValueError("array must be a C-contiguous numpy array of dtype %s" % np.dtype(dtype))
    return x.ctypes.data, 0


def _numel(x):
    return int(x.numel()) if _is_torch(x) else int(x.size)


def _expect(x, rows, n, what, device=None):
    """Marshalling check: buffer `x` (None allowed) must hold rows * n elements, and, if it is a CUDA tensor and `device` is given, live
    on that device.  A wrong size would be an out-of-bounds device access inside the library, not an RMHD_ERR_BAD_PARAM."""
    if x is None:
        return
    if _numel(x) != rows * n:
        raise ValueError("%s: expected %d x %d elements, got %d" % (what, rows, n, _numel(x)))
    if device is not None and _is_torch(x) and x.is_cuda and x.device.index != device:
        raise ValueError("%s lives on cuda:%d, the context on cuda:%d" % (what, x.device.index, device))


def _same_side(*flags):
    f = {v for v in flags if v is not None}
    if len(f) > 1:
        raise ValueError("all buffers of one call must be on the same side (all device or all host)")
    return f.pop() if f else 1


def _check(code, ctx=None):
    if code != RMHD_OK:
        msg = lib().rmhd_last_error(ctx)
        raise RmhdError(code, msg.decode() if msg else "")


# ---- the C-ABI calls, same names -------------------------------------------------------------
def rmhd_create(params):
    h = C.c_void_p()
    _check(lib().rmhd_create(C.byref(params), C.byref(h)))
    return h


def rmhd_destroy(ctx):
    lib().rmhd_destroy(ctx)


def rmhd_set_initial(ctx, prims, rho_charge=None):
    p, d1 = _ptr(prims); r, d2 = _ptr(rho_charge)
    _check(lib().rmhd_set_initial(ctx, p, r, _same_side(d1, d2)), ctx)


def rmhd_set_cons(ctx, cons, prim_guess=None):
    p, d1 = _ptr(cons); g, d2 = _ptr(prim_guess)
    return lib().rmhd_set_cons(ctx, p, g, _same_side(d1, d2))


def rmhd_step(ctx, nsteps=1, check=True):
    rc = lib().rmhd_step(ctx, int(nsteps))
    if check:
        _check(rc, ctx)
    return rc


def rmhd_get_state(ctx, cons=None, prims=None):
    p, d1 = _ptr(cons); w, d2 = _ptr(prims)
    _check(lib().rmhd_get_state(ctx, p, w, _same_side(d1, d2)), ctx)


def rmhd_flux_divergence(ctx, Lout):
    p, d = _ptr(Lout)
    _check(lib().rmhd_flux_divergence(ctx, p, d), ctx)


def rmhd_get_stats(ctx, nbins=64):
    hs = np.zeros(nbins, dtype=np.int64); hc = np.zeros(nbins, dtype=np.int64)
    nf = C.c_longlong(0); ff = C.c_longlong(-1)
    _check(lib().rmhd_get_stats(ctx, hs.ctypes.data_as(_lp), hc.ctypes.data_as(_lp), nbins, C.byref(nf), C.byref(ff)), ctx)
    return {"hist_stage": hs, "hist_c2p": hc, "n_failed": nf.value, "first_failed_cell": ff.value}


def rmhd_set_profiling(ctx, enabled):
    _check(lib().rmhd_set_profiling(ctx, int(bool(enabled))), ctx)


def rmhd_get_kernel_times(ctx):
    n = len(KERNEL_CLASSES)
    ms = np.zeros(n); ln = np.zeros(n, dtype=np.int64)
    _check(lib().rmhd_get_kernel_times(ctx, ms.ctypes.data_as(_dp), ln.ctypes.data_as(_lp), n), ctx)
    return {k: {"ms": float(ms[i]), "launches": int(ln[i])} for i, k in enumerate(KERNEL_CLASSES)}


def rmhd_dt(ctx):
    return lib().rmhd_dt(ctx)


def rmhd_time(ctx):
    return lib().rmhd_time(ctx)


def rmhd_stage_batch(params, q_ex, prim_guess, a_dt, q_out, prims_out, sigma_cell=None, iters=None, fail=None):
    n = q_ex.shape[-1]
    nc, npr, dev = NCONS[params.model], NPRIM[params.model], params.device
    _expect(q_ex, nc, n, "q_ex", dev); _expect(q_out, nc, n, "q_out", dev)
    _expect(prim_guess, npr, n, "prim_guess", dev); _expect(prims_out, npr, n, "prims_out", dev)
    for x, what in ((sigma_cell, "sigma_cell"), (iters, "iters"), (fail, "fail")):
        _expect(x, 1, n, what, dev)
    a, d1 = _ptr(q_ex); b, d2 = _ptr(prim_guess); s, d3 = _ptr(sigma_cell)
    qo, d4 = _ptr(q_out); po, d5 = _ptr(prims_out); it, d6 = _ptr(iters, np.int32); fl, d7 = _ptr(fail, np.int32)
    _check(lib().rmhd_stage_batch(C.byref(params), n, a, b, s, float(a_dt), qo, po, it, fl,
                                  _same_side(d1, d2, d3, d4, d5, d6, d7)))


def rmhd_prim2cons_batch(params, prims, cons, rho_charge=None):
    n = prims.shape[-1]
    _expect(prims, NPRIM[params.model], n, "prims", params.device); _expect(cons, NCONS[params.model], n, "cons", params.device)
    _expect(rho_charge, 1, n, "rho_charge", params.device)
    a, d1 = _ptr(prims); r, d2 = _ptr(rho_charge); c, d3 = _ptr(cons)
    _check(lib().rmhd_prim2cons_batch(C.byref(params), n, a, r, c, _same_side(d1, d2, d3)))


def rmhd_con2prim_batch(params, cons, prims, prim_guess=None, iters=None, fail=None):
    n = cons.shape[-1]
    _expect(cons, NCONS[params.model], n, "cons", params.device); _expect(prims, NPRIM[params.model], n, "prims", params.device)
    _expect(prim_guess, NPRIM[params.model], n, "prim_guess", params.device)
    _expect(iters, 1, n, "iters", params.device); _expect(fail, 1, n, "fail", params.device)
    a, d1 = _ptr(cons); g, d2 = _ptr(prim_guess); w, d3 = _ptr(prims)
    it, d4 = _ptr(iters, np.int32); fl, d5 = _ptr(fail, np.int32)
    _check(lib().rmhd_con2prim_batch(C.byref(params), n, a, g, w, it, fl, _same_side(d1, d2, d3, d4, d5)))


def rmhd_flux_divergence_static(params, cons, Lout, check=True):
    """L(q) of a conserved state held by the caller, for callers that cannot let the library allocate device memory (their
    own pool owns the card, or their loop cannot take the device-wide stall of cudaMalloc / cudaFree).  `cons` and `Lout`
    are CUDA tensors [14|18][nz][ny][nx] on params.device; the grid may have at most RMHD_STATIC_MAX_CELLS cells, because
    the scratch is one fixed array inside the library, shared by all calls on that GPU: do not overlap two calls.
    Returns (code, n_failed); with check=True a non-zero code raises instead."""
    n = params.nx * params.ny * params.nz
    nc = NCONS[params.model]
    _expect(cons, nc, n, "cons", params.device); _expect(Lout, nc, n, "Lout", params.device)
    a, d1 = _ptr(cons); b, d2 = _ptr(Lout)
    if d1 != 1 or d2 != 1:
        raise ValueError("rmhd_flux_divergence_static takes device buffers only (CUDA tensors)")
    nf = C.c_longlong(0)
    rc = lib().rmhd_flux_divergence_static(C.byref(params), a, b, C.byref(nf))
    if check:
        _check(rc)
    return rc, nf.value


def rmhd_release_staging(device=-1):
    """Free the staging area the host-buffer batch calls keep on `device` (-1: on every GPU)."""
    _check(lib().rmhd_release_staging(int(device)))


def rmhd_debug_hm_cycles(device=0, reset=False):
    """Cycle account of k_flux_hm ([role H | M][phase 0..6, warp-planes], csrc/flux_hm.cuh), or None: only a measurement build
    of the library (-DRMHD_HM_CYCLES) exports it."""
    L = lib()
    if not hasattr(L, "rmhd_debug_hm_cycles"):
        return None
    out = np.zeros((2, 8), dtype=np.uint64)
    L.rmhd_debug_hm_cycles.argtypes = [C.c_int, C.c_void_p, C.c_int]
    _check(L.rmhd_debug_hm_cycles(device, out.ctypes.data, int(bool(reset))))
    return out


def rmhd_probe_fp64(device=0, stream=None):
    v = C.c_double(0.0)
    _check(lib().rmhd_probe_fp64(device, _current_stream(device) if stream is None else stream, C.byref(v)))
    return v.value


def rmhd_probe_hbm(nbytes=1 << 30, device=0, stream=None):
    v = C.c_double(0.0)
    _check(lib().rmhd_probe_hbm(device, _current_stream(device) if stream is None else stream, int(nbytes), C.byref(v)))
    return v.value


# ---- a small convenience wrapper (still marshalling only) --------------------------------------
class Rmhd:
    """One grid on one GPU: set_initial / step / get_state, mirroring the C-ABI."""

    def __init__(self, **kw):
        self.params = make_params(**kw)
        self.model = self.params.model
        self.shape = (self.params.nz, self.params.ny, self.params.nx)
        self.ctx = rmhd_create(self.params)

    def close(self):
        if getattr(self, "ctx", None):
            rmhd_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    dt = property(lambda self: rmhd_dt(self.ctx))
    time = property(lambda self: rmhd_time(self.ctx))

    @property
    def ncells(self):
        return self.shape[0] * self.shape[1] * self.shape[2]

    def set_initial(self, prims, rho_charge=None):
        _expect(prims, NPRIM[self.model], self.ncells, "prims", self.params.device)
        _expect(rho_charge, 1, self.ncells, "rho_charge", self.params.device)
        rmhd_set_initial(self.ctx, prims, rho_charge)

    def set_cons(self, cons, prim_guess=None):
        _expect(cons, NCONS[self.model], self.ncells, "cons", self.params.device)
        if prim_guess is not None and _numel(prim_guess) not in (NHYD[self.model] * self.ncells, NPRIM[self.model] * self.ncells):
            raise ValueError("prim_guess: expected the %d hydro rows (or all %d primitive rows) per cell" % (NHYD[self.model], NPRIM[self.model]))
        return rmhd_set_cons(self.ctx, cons, prim_guess)

    def step(self, n=1, check=True):
        return rmhd_step(self.ctx, n, check)

    def get_state(self, device=False):
        """Returns (cons, prims): numpy arrays, or torch CUDA tensors if device=True."""
        if device:
            import torch
            dev = torch.device("cuda", self.params.device)
            cons = torch.empty((NCONS[self.model],) + self.shape, dtype=torch.float64, device=dev)
            prims = torch.empty((NPRIM[self.model],) + self.shape, dtype=torch.float64, device=dev)
        else:
            cons = np.empty((NCONS[self.model],) + self.shape)
            prims = np.empty((NPRIM[self.model],) + self.shape)
        rmhd_get_state(self.ctx, cons, prims)
        return cons, prims

    def flux_divergence(self):
        L = np.empty((NCONS[self.model],) + self.shape)
        rmhd_flux_divergence(self.ctx, L)
        return L

    def stats(self, nbins=64):
        return rmhd_get_stats(self.ctx, nbins)
