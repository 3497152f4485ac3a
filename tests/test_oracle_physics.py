"""Grid-level pins of the CPU oracle: invariants, exact solutions, symmetry, convergence.

No GPU.  Each check is against physics/mathematics, not against the oracle itself
(SURVEY.md 8(c) "What pins each part"; north_star's list of oracle checks).
"""
import math
import os

import numpy as np
import pytest
from scipy.special import erf

G43 = 4.0 / 3.0
PER, OUT = 1, 0


def _sim(O, **kw):
    return O.OracleSim(O.make_params(**kw))


def _stage_R(z):
    """SSP2(222) stability function from Table 2; see tests/golden/ssp222_table2.txt."""
    g = 1 - 1 / math.sqrt(2)
    k1 = 1 / (1 - g * z)
    k2 = (1 + (1 - 2 * g) * z * k1) / (1 - g * z)
    return 1 + 0.5 * z * (k1 + k2)


def _smooth_resistive(nx, ny, nz, seed, amp=0.2):
    """Smooth periodic random primitive field (few Fourier modes) for invariance tests."""
    rng = np.random.default_rng(seed)
    x = (np.arange(nx) + 0.5) / nx; y = (np.arange(ny) + 0.5) / ny; z = (np.arange(nz) + 0.5) / nz
    Z, Y, X = np.meshgrid(z, y, x, indexing="ij")

    def fld():
        f = np.zeros_like(X)
        for _ in range(3):
            k = rng.integers(0, 2, 3) * np.array([nx > 1, ny > 1, nz > 1])
            f += rng.uniform(-1, 1) * np.sin(2 * np.pi * (k[0] * X + k[1] * Y + k[2] * Z) + rng.uniform(0, 6.28))
        return f

    w = np.zeros((11, nz, ny, nx))
    w[0] = 1.0 + amp * fld(); w[4] = 1.0 + amp * fld()
    for c in range(3):
        w[1 + c] = amp * fld(); w[5 + c] = amp * fld(); w[8 + c] = amp * fld()
    return w


# ------------------------------------------------------------------------------------------
# L(q): uniform state, telescoping conservation
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("model", [0, 1])
def test_uniform_state_has_zero_flux_divergence_bitwise(O, model):
    np_ = 11 if model == 0 else 16
    rng = np.random.default_rng(2)
    vals = rng.uniform(0.1, 0.5, np_)
    w = np.ones((np_, 6, 7, 8)) * vals[:, None, None, None]
    S = _sim(O, model=model, nx=8, ny=7, nz=6, bc=(PER, OUT, PER), sigma=50.0, eta=1e-3, mu_e=-10.0, mu_p=10.0)
    S.set_initial(w, None if model else np.full((6, 7, 8), 0.3))
    L = S.eval_L()
    assert np.all(L == 0.0)


@pytest.mark.parametrize("model", [0, 1])
def test_periodic_conservation_of_source_free_rows(O, synth, model):
    """Rows with zero source (eq 1 P:L57 / A2 P:L445) are conserved to round-off on periodic grids."""
    nx, ny, nz = 12, 10, 6
    if model == 0:
        w = _smooth_resistive(nx, ny, nz, seed=1)
        rows = [0, 1, 2, 3, 4, 5, 6, 7, 11]
    else:
        w0 = _smooth_resistive(nx, ny, nz, seed=1)
        w = np.zeros((16, nz, ny, nx))
        w[0:5] = w0[0:5]; w[5:10] = w0[0:5]; w[6:9] *= -0.5; w[5] *= 0.7
        w[10:13] = 0.05 * w0[5:8]; w[13:16] = 0.05 * w0[8:11]
        rows = [0, 1, 2, 3, 4, 5, 10, 11, 12]
    S = _sim(O, model=model, nx=nx, ny=ny, nz=nz, bc=(PER, PER, PER), sigma=20.0, eta=1e-3, mu_e=-5.0, mu_p=5.0,
             cfl=0.3)
    S.set_initial(w)
    q0, _ = S.get_state()
    L = S.eval_L()
    assert S.step(3) == 0
    q1, _ = S.get_state()
    ncell = nx * ny * nz
    for r in range(q0.shape[0]):
        # telescoping: the flux divergence sums to zero for every row
        assert abs(L[r].sum()) < 1e-10 * max(1.0, np.abs(L[r]).sum())
    for r in rows:
        assert abs(q1[r].sum() - q0[r].sum()) < 2e-13 * max(np.abs(q0[r]).sum(), ncell * 1e-3), r
    # something did happen
    assert np.abs(q1 - q0).max() > 1e-4


# ------------------------------------------------------------------------------------------
# full step against closed forms
# ------------------------------------------------------------------------------------------
def test_full_step_decay_matches_ssp222_stability_function(O):
    """Uniform fluid at rest, B = 0, rhoc = 0: E' = -sigma E exactly (v stays 0, Joule heat
    only changes p), so one step multiplies E by R(-sigma dt).  phi' = -kappa phi likewise;
    psi' = rhoc - kappa psi is affine, so (psi - rhoc/kappa) is multiplied by R(-kappa dt)."""
    nx = 8
    S = _sim(O, model=0, nx=nx, bc=(PER, PER, PER), xlim=(0.0, 1.0), cfl=0.4, sigma=20.0, kappa=3.0, gamma=G43)
    dt = S.dt
    assert abs(dt - 0.05) < 1e-15
    w = np.zeros((11, 1, 1, nx)); w[0] = 1.0; w[4] = 1.0
    w[8], w[9], w[10] = 0.01, -0.02, 0.005
    S.set_initial(w, np.zeros((1, 1, nx)))
    q0, _ = S.get_state()
    q0[11] = 0.7        # uniform charge density, fluid at rest: J = sigma E only
    q0[12] = 0.4; q0[13] = -0.3
    assert S.set_cons(q0) == 0
    S.step(1)
    q1, w1 = S.get_state()
    Rz = _stage_R(-20.0 * dt)
    assert abs(Rz - 0.350440262760) < 1e-11
    for c in range(3):
        assert np.allclose(q1[8 + c], Rz * q0[8 + c], rtol=1e-11, atol=1e-16)
    Rk = _stage_R(-3.0 * dt)
    assert np.allclose(q1[13], Rk * q0[13], rtol=1e-12)
    assert np.allclose(q1[12] - 0.7 / 3.0, Rk * (q0[12] - 0.7 / 3.0), rtol=1e-12)
    assert np.allclose(q1[11], 0.7, rtol=1e-14)
    assert np.abs(w1[1:4]).max() < 1e-14
    # energy conservation: tau unchanged, so the pressure rose by the lost field energy
    assert np.allclose(q1[4], q0[4], rtol=1e-14)
    assert np.all(w1[4] > 1.0)


def test_steady_uniform_flow_is_left_unchanged(O):
    """Uniform flow with E = -v x B, rhoc = 0 => J = 0 => nothing changes (to round-off)."""
    nx, ny = 8, 6
    v = np.array([0.3, -0.2, 0.4]); B = np.array([0.5, 0.1, -0.3]); E = -np.cross(v, B)
    w = np.zeros((11, 1, ny, nx)); w[0] = 1.3; w[4] = 0.8
    for c in range(3):
        w[1 + c] = v[c]; w[5 + c] = B[c]; w[8 + c] = E[c]
    S = _sim(O, model=0, nx=nx, ny=ny, bc=(PER, OUT, OUT), sigma=1e4)
    S.set_initial(w)
    q0, _ = S.get_state()
    assert np.abs(q0[11]).max() == 0.0                      # Gauss's law of a uniform E
    S.step(5)
    q1, w1 = S.get_state()
    assert np.abs(q1 - q0).max() < 1e-12
    assert np.abs(w1 - w).max() < 1e-12


def test_two_fluid_steady_state(O):
    """Equal species co-moving with E = -v x B: rhoc = 0, J = rho0 u = 0 => Psi = 0."""
    nx = 8
    v = np.array([0.2, 0.1, -0.3]); B = np.array([0.2, -0.1, 0.3]); E = -np.cross(v, B)
    w = np.zeros((16, 1, 1, nx))
    for s in range(2):
        w[5 * s] = 0.5; w[5 * s + 4] = 0.5
        for c in range(3):
            w[5 * s + 1 + c] = v[c]
    for c in range(3):
        w[10 + c] = B[c]; w[13 + c] = E[c]
    S = _sim(O, model=1, nx=nx, bc=(PER, PER, PER), eta=1e-3, mu_e=-100.0, mu_p=100.0)
    S.set_initial(w)
    q0, _ = S.get_state()
    assert S.step(4) == 0
    q1, w1 = S.get_state()
    assert np.abs(q1 - q0).max() < 1e-10 and np.abs(w1 - w).max() < 1e-11


# ------------------------------------------------------------------------------------------
# Maxwell flux signs: vacuum plane wave along each axis (SURVEY 8(c) "flux/Maxwell signs")
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_vacuum_plane_wave_travels_right_and_converges(O, axis):
    """sigma = 0, rhoc = 0, fluid at rest: E_b = B_c = A sin 2 pi (s - t) with (a,b,c) cyclic,
    a = propagation axis, is an exact solution.  Error after one period must fall at ~2nd
    order; a sign slip in the B/E flux rows sends the wave backwards (error O(A))."""
    A = 1e-3
    errs = []
    b, c = (axis + 1) % 3, (axis + 2) % 3
    for n in (16, 32, 64):
        dims = [1, 1, 1]; dims[axis] = n
        S = _sim(O, model=0, nx=dims[0], ny=dims[1], nz=dims[2], bc=(PER, PER, PER), sigma=0.0, cfl=0.4, gamma=G43)
        nsteps = int(round(1.0 / S.dt))
        assert abs(nsteps * S.dt - 1.0) < 1e-12
        s = (np.arange(n) + 0.5) / n
        shape = [1, 1, 1]; shape[2 - axis] = n
        prof = (A * np.sin(2 * np.pi * s)).reshape(shape)
        w = np.zeros((11, dims[2], dims[1], dims[0])); w[0] = 1.0; w[4] = 1.0
        # wave along a: E_c? Faraday: dB_c/dt = -(curl E)_c = -dE_b/da  with B_c = E_b = f(a - t)
        w[8 + b] = prof; w[5 + c] = prof
        S.set_initial(w, np.zeros((dims[2], dims[1], dims[0])))
        # a quarter period first: the wave must have moved by +1/4 (direction check)
        S.step(nsteps // 4)
        q, _ = S.get_state()
        moved = (A * np.sin(2 * np.pi * (s - 0.25))).reshape(shape)
        assert np.abs(q[8 + b] - moved).max() < 0.15 * A
        S.step(nsteps - nsteps // 4)
        q, wf = S.get_state()
        err = np.abs(q[8 + b] - prof).mean() + np.abs(q[5 + c] - prof).mean()
        errs.append(err / A)
        assert np.abs(wf[1:4]).max() < 1e-6          # fluid stays at rest (O(A^2) at most)
    o1, o2 = math.log2(errs[0] / errs[1]), math.log2(errs[1] / errs[2])
    assert errs[2] < 0.02
    assert o1 > 1.6 and o2 > 1.6, (errs, o1, o2)


# ------------------------------------------------------------------------------------------
# bitwise mirror symmetry (north_star)
# ------------------------------------------------------------------------------------------
def _mirror_x_resistive(a, kind):
    """Mirror image under x -> -x of a [var,k,j,i] array; kind 'prims' (11) or 'cons' (14).
    Polar vectors (v, S, E) flip the x component; axial B flips y and z; phi is a pseudoscalar."""
    m = a[..., ::-1].copy()
    if kind == "prims":
        odd = [1, 6, 7, 8]
    else:
        odd = [1, 6, 7, 8, 13]
    m[odd] = -m[odd]
    return m


def test_bitwise_mirror_symmetry_2d_resistive(O):
    nx, ny = 16, 12
    w = _smooth_resistive(nx, ny, 1, seed=7, amp=0.15)
    kw = dict(model=0, nx=nx, ny=ny, bc=(OUT, PER, OUT), xlim=(-0.5, 0.5), ylim=(0.0, 1.0), sigma=300.0, cfl=0.4)
    S = _sim(O, **kw); S.set_initial(w); S.step(4); qa, wa = S.get_state()
    S2 = _sim(O, **kw); S2.set_initial(_mirror_x_resistive(w, "prims")); S2.step(4); qb, wb = S2.get_state()
    assert np.array_equal(_mirror_x_resistive(qb, "cons"), qa)
    assert np.array_equal(_mirror_x_resistive(wb, "prims"), wa)
    assert np.abs(qa[12:]).max() > 0     # cleaning fields were exercised


def test_bitwise_mirror_symmetry_3d_blast(O, synth):
    """cfg5 is x-mirror symmetric as it stands (B_x even under x -> -x): the solution must
    stay its own mirror image bit for bit."""
    c = synth.config5(n=12, nsteps=3)
    P = dict(c["params"])
    S = _sim(O, **P); S.set_initial(c["prims"]); assert S.step(3) == 0
    q, w = S.get_state()
    assert np.array_equal(_mirror_x_resistive(q, "cons"), q)
    assert np.abs(q[1]).max() > 1e-3
    # y-mirror needs the extra charge conjugation: (E,B,rhoc,psi,phi) -> -(...)
    m = q[:, :, ::-1, :].copy()
    for r in (2,):            # S_y polar
        m[r] = -m[r]
    for r in (5, 7):          # B_x, B_z axial tangential flip, then conjugation flips all B
        m[r] = -m[r]
    m[5:8] = -m[5:8]
    m[9] = -m[9]              # E_y polar normal flips
    m[8:11] = -m[8:11]
    m[11] = -m[11]; m[12] = -m[12]   # rhoc, psi scalars: conjugation only; phi pseudoscalar: both
    assert np.array_equal(m, q)


# ------------------------------------------------------------------------------------------
# resistive physics: self-similar current sheet (G12)
# ------------------------------------------------------------------------------------------
def _current_sheet(O, n, gold):
    t0, t1, sig = gold["t_start"], gold["t_end"], gold["sigma"]
    dx = 3.0 / n
    nsteps = int(math.ceil((t1 - t0) / (0.4 * dx)))
    cfl = (t1 - t0) / nsteps / dx
    S = _sim(O, model=0, nx=n, bc=(OUT, OUT, OUT), xlim=(-1.5, 1.5), sigma=sig, cfl=cfl, gamma=2.0)
    x = -1.5 + (np.arange(n) + 0.5) * dx
    w = np.zeros((11, 1, 1, n)); w[0] = gold["rho"]; w[4] = gold["p"]
    w[6, 0, 0] = gold["B0"] * erf(x / (2 * math.sqrt(t0 / sig)))
    S.set_initial(w)
    assert S.step(nsteps) == 0
    q, _ = S.get_state()
    return x, q[6, 0, 0]


def test_current_sheet_second_order_and_near_analytic(O):
    gold = {}
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "current_sheet.txt")):
        if not line.startswith("#") and line.strip():
            k, v = line.split(); gold[k] = float(v)
    sol = {}
    for n in (50, 100, 200):
        sol[n] = _current_sheet(O, n, gold)
    coarsen = lambda a: 0.5 * (a[0::2] + a[1::2])
    e1 = np.abs(coarsen(sol[100][1]) - sol[50][1]).mean()
    e2 = np.abs(coarsen(sol[200][1]) - sol[100][1]).mean()
    order = math.log2(e1 / e2)
    assert order > 1.7, (e1, e2, order)
    x = sol[200][0]
    exact = gold["B0"] * erf(x / (2 * math.sqrt(gold["t_end"] / gold["sigma"])))
    # eq (15) neglects the displacement current and the back-reaction: close, not identical
    assert np.abs(sol[200][1] - exact).max() < 2e-2
    x = sol[50][0]
    exact = gold["B0"] * erf(x / (2 * math.sqrt(gold["t_end"] / gold["sigma"])))
    assert np.abs(sol[50][1] - exact).max() < 3e-2        # "indistinguishable" at N = 50


def test_ideal_limit_of_riemann_tube(O, synth):
    """Fig 1 / P:L287: as sigma grows the solution tends to a limit: successive differences shrink."""
    c = synth.config1(nx=64)
    By = {}
    for sig in (1e1, 1e2, 1e3, 1e4, 1e5):
        P = dict(c["params"]); P["sigma"] = sig
        S = _sim(O, **P); S.set_initial(c["prims"]); assert S.step(c["nsteps"]) == 0
        By[sig] = S.get_state()[0][6, 0, 0]
    d = [np.abs(By[s] - By[10 * s]).mean() for s in (1e1, 1e2, 1e3, 1e4)]
    assert d[0] > d[1] > d[2] > d[3]
    assert d[3] < 0.1 * d[0]


# ------------------------------------------------------------------------------------------
# two-fluid source: Langmuir oscillation (SURVEY 8(c) "two-fluid source")
# ------------------------------------------------------------------------------------------
def _langmuir(O, steps_per_period, eta, periods=1):
    mu = 100.0
    omega = math.sqrt(2 * mu * mu * 0.5 / 5.0)      # omega^2 = sum mu_s^2 rho_s / h_s, h_s = 5
    T = 2 * math.pi / omega
    dt = T / steps_per_period
    nx = 4
    S = _sim(O, model=1, nx=nx, bc=(PER, PER, PER), xlim=(0.0, nx * dt / 0.4), cfl=0.4, eta=eta, mu_e=-mu, mu_p=mu,
             gamma=G43)
    assert abs(S.dt - dt) < 1e-15
    w = np.zeros((16, 1, 1, nx)); w[0] = w[5] = 0.5; w[4] = w[9] = 0.5
    w[13] = 1e-6
    S.set_initial(w)
    Ex = [1e-6]
    for _ in range(steps_per_period * periods):
        S.step(1)
        Ex.append(S.get_state()[0][13, 0, 0, 0])
    return np.array(Ex) / 1e-6, omega, dt


def test_two_fluid_langmuir_frequency_and_damping(O):
    Ex, omega, dt = _langmuir(O, 64, 0.0)
    t = np.arange(Ex.size) * dt
    e64 = np.abs(Ex - np.cos(omega * t)).max()
    Ex2, _, dt2 = _langmuir(O, 128, 0.0)
    t2 = np.arange(Ex2.size) * dt2
    e128 = np.abs(Ex2 - np.cos(omega * t2)).max()
    assert e128 < 0.01
    assert math.log2(e64 / e128) > 1.7            # second order in dt
    # friction damps: J'' + (eta wp^2/h) J' + (wp^2/h) J = 0  ->  amplitude ~ exp(-eta omega^2 t / 2)
    eta = 1e-3
    Ex3, _, dt3 = _langmuir(O, 128, eta)
    T = 128 * dt3
    ratio = Ex3[-1] / Ex2[-1]
    assert abs(ratio - math.exp(-0.5 * eta * omega ** 2 * T)) < 0.02
