"""rmhd_flux_divergence_static (include/rmhd.h): L(q) of a state the caller holds, for programs that cannot let this
library allocate device memory -- the host application's own pool owns the card (a cudaMalloc behind its back can fail
while the pool has room), or the time loop cannot take the device-wide stall that cudaFree causes and cudaMalloc may.
Its scratch (recovered primitives, failure counters) is one fixed array inside the library, shared by every call on the
GPU and never cleared between calls by anyone but the call itself.

The check: the same numbers as the allocating path (rmhd_create + rmhd_set_cons + rmhd_flux_divergence) within the
bound the flux parity tests use (1e-12 of max |L| per variable), on calls made one after the other: a large grid, then a
smaller grid of the other model with one unrecoverable cell (the counter must say so), then a clean grid (the counter
must be back at zero, and stale primitives of the larger grids must not leak into the result).

This file is named to be collected last: `pytest -x` stops at the first failure, and one here must not hide the parity
tests.  It passes alone in a fresh process (its first call does the per-device set-up) and after all the other tests.
"""
import ctypes as C

import numpy as np
import pytest

G43 = 4.0 / 3.0


@pytest.fixture(scope="module")
def B():
    from paper_1808_09721_b200 import build, binding
    build.build()
    binding.lib()
    return binding


def _random_prims(model, shape, seed):
    rng = np.random.default_rng(seed)
    w = np.zeros((11 if model == 0 else 16,) + shape)
    for s in range(1 if model == 0 else 2):
        w[5 * s] = 10 ** rng.uniform(-0.5, 0.5, shape)
        w[5 * s + 4] = 10 ** rng.uniform(-1, 0.5, shape)
        w[5 * s + 1:5 * s + 4] = rng.uniform(-0.5, 0.5, (3,) + shape)
    w[-6:] = 0.3 * rng.standard_normal((6,) + shape)
    return w


def _case(B, model, shape, bc, seed, poison=None):
    """Conserved state of random primitives (through the library's own prim2cons), optionally with one cell made unrecoverable."""
    nz, ny, nx = shape
    kw = dict(model=model, nx=nx, ny=ny, nz=nz, bc=bc, xlim=(0.0, 1.0), ylim=(-1.0, 0.5), zlim=(0.0, 0.7), gamma=G43,
              sigma=25.0, eta=1e-3, mu_e=-20.0, mu_p=10.0)
    w = _random_prims(model, shape, seed)
    n = nx * ny * nz
    q = np.empty((B.NCONS[model], n))
    B.rmhd_prim2cons_batch(B.make_params(**kw), np.ascontiguousarray(w.reshape(w.shape[0], n)), q)
    q = q.reshape((B.NCONS[model],) + shape)
    if poison is not None:
        q[(4,) + poison] = -50.0      # tau far below what any admissible state allows: no root
    return kw, q


def _allocating_path(B, kw, q):
    sim = B.Rmhd(**kw)
    rc = sim.set_cons(q)
    L = sim.flux_divergence()
    nf = sim.stats()["n_failed"]
    sim.close()
    return rc, nf, L


@pytest.mark.gpu
def test_static_scratch_flux_divergence_matches_the_allocating_path_call_after_call(B):
    import torch
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device (there is no CPU fallback)")
    calls = [
        (0, (20, 19, 70), (1, 0, 1), 11, None),           # 3-D resistive, partial tiles, several z segments
        (1, (1, 12, 37), (0, 1, 0), 12, (0, 5, 17)),      # 2-D two-fluid with one unrecoverable cell
        (0, (7, 10, 34), (0, 1, 0), 13, None),            # clean again, smaller than the first: nothing may be left over
        (0, (1, 1, 130), (1, 1, 1), 14, None),            # 1-D (the per-axis kernel)
    ]
    for model, shape, bc, seed, poison in calls:
        kw, q = _case(B, model, shape, bc, seed, poison)
        rc_ref, nf_ref, L_ref = _allocating_path(B, kw, q)
        qd = torch.from_numpy(q).cuda()
        Ld = torch.full_like(qd, float("nan"))
        rc, nf = B.rmhd_flux_divergence_static(B.make_params(**kw), qd, Ld, check=False)
        L = Ld.cpu().numpy()
        assert nf == nf_ref and rc == rc_ref, (shape, rc, rc_ref, nf, nf_ref)
        if poison is None:
            assert rc == B.RMHD_OK and nf == 0
        else:
            assert rc == B.RMHD_ERR_NONCONVERGED and nf >= 1
            assert b"recovery failed" in B.lib().rmhd_last_error(None)
        fin = np.isfinite(L_ref)
        assert np.array_equal(fin, np.isfinite(L)), shape
        assert fin.mean() > 0.9
        scale = np.abs(np.where(fin, L_ref, 0.0)).max(axis=(1, 2, 3), keepdims=True) + 1e-30
        err = np.where(fin, np.abs(np.where(fin, L, 0.0) - np.where(fin, L_ref, 0.0)), 0.0) / scale
        assert err.max() < 1e-12, (shape, float(err.max()))
        assert torch.equal(qd.cpu(), torch.from_numpy(q))          # the input is only read


def test_static_scratch_limit_is_enforced_before_anything_runs(B):
    """A grid beyond RMHD_STATIC_MAX_CELLS is refused with a message that names the limit; checked before the device
    is touched, so this runs without a GPU (the pointers are never dereferenced)."""
    nf = C.c_longlong(-7)
    for kw in (dict(nx=513, ny=512), dict(nx=64, ny=64, nz=65), dict(model=1, nx=B.RMHD_STATIC_MAX_CELLS + 1, mu_e=-1.0, mu_p=1.0)):
        p = B.make_params(**{**dict(sigma=1.0), **kw})
        rc = B.lib().rmhd_flux_divergence_static(C.byref(p), C.c_void_p(256), C.c_void_p(512), C.byref(nf))
        assert rc == B.RMHD_ERR_BAD_PARAM
        msg = B.lib().rmhd_last_error(None).decode()
        assert "RMHD_STATIC_MAX_CELLS = 262144" in msg and "rmhd_create" in msg
    p = B.make_params(nx=8, sigma=1.0)
    assert B.lib().rmhd_flux_divergence_static(C.byref(p), None, C.c_void_p(512), None) == B.RMHD_ERR_BAD_PARAM
    with pytest.raises(ValueError):      # host arrays are not accepted: this call stages nothing
        B.rmhd_flux_divergence_static(p, np.zeros((14, 8)), np.zeros((14, 8)))
