"""Pins of the oracle's general IMEX stepper and of SSP3(332) (Table 3).

Nothing here compares the oracle with itself through the same route: the expected values are closed
forms built in this file from the Butcher tables (tests/golden/ssp3_332_table3.txt), a textbook
re-arrangement of the explicit part (Shu-Osher convex-combination form) driven through eval_L, or the
already pinned SSP2(222) path.
"""
import math
import os

import numpy as np

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
PER = 1
G43 = 4.0 / 3.0
g = 1 - 1 / math.sqrt(2)

# Table 3 (reading G13) written out here independently of oracle/
AT3 = np.array([[0, 0, 0], [1, 0, 0], [0.25, 0.25, 0]], float)
WT3 = np.array([1 / 6, 1 / 6, 2 / 3])
A3 = np.array([[g, 0, 0], [1 - 2 * g, g, 0], [0.5 - g, 0, g]])
W3 = np.array([1 / 6, 1 / 6, 2 / 3])
# Table 2
AT2 = np.array([[0, 0], [1, 0]], float)
WT2 = np.array([0.5, 0.5])
A2 = np.array([[g, 0], [1 - 2 * g, g]])
W2 = np.array([0.5, 0.5])


def _sim(O, **kw):
    return O.OracleSim(O.make_params(**kw))


def imex_linear_map(Le, Li, dt, at, wt, a, w):
    """One step of eq (10)-(11) for the linear system y' = Le y + Li y (Le explicit, Li implicit)."""
    n = Le.shape[0]
    I = np.eye(n, dtype=complex)
    Y = []
    for i in range(len(w)):
        rhs = I.copy()
        for j in range(i):
            rhs = rhs + dt * (at[i, j] * Le + a[i, j] * Li) @ Y[j]
        Y.append(np.linalg.solve(I - a[i, i] * dt * Li, rhs))
    G = I.copy()
    for j in range(len(w)):
        G = G + dt * (wt[j] * Le + w[j] * Li) @ Y[j]
    return G


def test_table3_satisfies_the_order_conditions():
    """Explicit part third order, implicit part second order, stage times consistent (Pareschi & Russo):
    fixes the reading G13 of the garbled row."""
    ct, c = AT3.sum(1), A3.sum(1)
    assert np.allclose(ct, [0, 1, 0.5]) and np.allclose(c, [g, 1 - g, 0.5])
    assert abs(WT3.sum() - 1) < 1e-15 and abs(W3.sum() - 1) < 1e-15
    assert abs(WT3 @ ct - 0.5) < 1e-15 and abs(WT3 @ ct ** 2 - 1 / 3) < 1e-15 and abs(WT3 @ (AT3 @ ct) - 1 / 6) < 1e-15
    assert abs(W3 @ c - 0.5) < 1e-15 and abs(WT3 @ c - 0.5) < 1e-15 and abs(W3 @ ct - 0.5) < 1e-15
    gold = [l for l in open(os.path.join(GOLD, "ssp3_332_table3.txt")) if l.startswith("R(-1)")]
    R = imex_linear_map(np.zeros((1, 1)), np.array([[-1.0]]), 1.0, AT3, WT3, A3, W3)[0, 0].real
    assert abs(R - float(gold[0].split()[1])) < 1e-11


def test_ssp3_decay_matches_the_implicit_stability_function(O):
    """Uniform fluid at rest, B = 0: E' = -sigma E, phi' = -kappa phi exactly, L == 0, so one step multiplies by the
    stability function of the implicit tableau (a wrong a_31, a_21 or w changes it: a_31 = 1/2 gives 0.467 at z = -1)."""
    nx = 8
    S = _sim(O, model=0, nx=nx, bc=(PER, PER, PER), xlim=(0.0, 1.0), cfl=0.4, sigma=20.0, kappa=3.0, gamma=G43, integrator="ssp3")
    dt = S.dt
    w = np.zeros((11, 1, 1, nx)); w[0] = 1.0; w[4] = 1.0
    w[8], w[9], w[10] = 0.01, -0.02, 0.005
    S.set_initial(w, np.zeros((1, 1, nx)))
    q0, _ = S.get_state()
    q0[11] = 0.7; q0[12] = 0.4; q0[13] = -0.3
    assert S.set_cons(q0) == 0
    S.step(1)
    q1, w1 = S.get_state()
    R = lambda z: imex_linear_map(np.zeros((1, 1)), np.array([[z]]), 1.0, AT3, WT3, A3, W3)[0, 0].real
    Rz, Rk = R(-20.0 * dt), R(-3.0 * dt)
    assert abs(Rz - 0.350440262760) < 1e-11
    for c in range(3):
        assert np.allclose(q1[8 + c], Rz * q0[8 + c], rtol=1e-11, atol=1e-16)
    assert np.allclose(q1[13], Rk * q0[13], rtol=1e-12)
    assert np.allclose(q1[12] - 0.7 / 3.0, Rk * (q0[12] - 0.7 / 3.0), rtol=1e-12)
    assert np.allclose(q1[4], q0[4], rtol=1e-14) and np.abs(w1[1:4]).max() < 1e-14


def _smooth_prims(nx, ny, seed):
    rng = np.random.default_rng(seed)
    x = (np.arange(nx) + 0.5) / nx; y = (np.arange(ny) + 0.5) / ny
    Y, X = np.meshgrid(y, x, indexing="ij")

    def fld(amp):
        return amp * (rng.uniform(-1, 1) * np.sin(2 * np.pi * X + rng.uniform(0, 6)) + rng.uniform(-1, 1) * np.cos(2 * np.pi * Y + rng.uniform(0, 6)))
    w = np.zeros((11, 1, ny, nx))
    w[0] = 1.0 + fld(0.2); w[4] = 1.0 + fld(0.2)
    for c in range(3):
        w[1 + c] = fld(0.2); w[5 + c] = fld(0.3); w[8 + c] = fld(0.1)
    return w


def test_source_free_ssp3_is_shu_osher_rk3(O):
    """sigma = 0, rhoc = 0, kappa = 0 => Psi == 0 and the scheme is its explicit part, which for Table 3 is the
    Shu-Osher SSP-RK3.  Recompose it in its convex-combination form from eval_L calls:
      u1 = u + dt L(u);  u2 = 3/4 u + 1/4 (u1 + dt L(u1));  u' = 1/3 u + 2/3 (u2 + dt L(u2))."""
    nx, ny = 16, 12
    kw = dict(model=0, nx=nx, ny=ny, bc=(PER, PER, PER), cfl=0.3, sigma=0.0, kappa=0.0, gamma=G43)
    w = _smooth_prims(nx, ny, 5)
    S = _sim(O, integrator="ssp3", **kw)
    S.set_initial(w, np.zeros((1, ny, nx)))
    u, _ = S.get_state()
    dt = S.dt
    S.step(1)
    q_oracle, _ = S.get_state()
    S.close()
    T = _sim(O, **kw)

    def L(q):
        assert T.set_cons(q) == 0
        return T.eval_L()
    u1 = u + dt * L(u)
    u2 = 0.75 * u + 0.25 * (u1 + dt * L(u1))
    un = u / 3 + 2 / 3 * (u2 + dt * L(u2))
    T.close()
    assert np.abs(un - u).max() > 1e-3
    assert np.abs(q_oracle - un).max() < 1e-13
    # and it is NOT what two stages give
    S2 = _sim(O, integrator="ssp2", **kw); S2.set_initial(w, np.zeros((1, ny, nx))); S2.step(1); q2, _ = S2.get_state(); S2.close()
    assert np.abs(q2 - un).max() > 1e-7


def _telegraph_case(O, integrator, at, wt, a, w):
    """(B_x, phi) with sigma = 0, E = 0, rhoc = 0, fluid at rest is the linear telegraph system
        d_t B_x = -d_x phi,  d_t phi = -d_x B_x - kappa phi            (eq 1: flux of B_x is phi, of phi is B_x)
    and decouples from the fluid (the Lorentz force is O(A^2)).  At amplitude A = 1e-9 the WENO3 smoothness indicators are
    ~1e-19 << eps = 1e-6, so the reconstruction is its linear-weight limit u^ = -a/6 + 5b/6 + c/3 and one Fourier mode
    is an eigenfunction: the step is a 2x2 complex matrix built here from the tableau, the LF split (alpha = 1) and
    the linear-weight symbol.  The explicit and implicit parts do not commute, so every coefficient matters."""
    nx, kappa, A = 16, 5.0, 1e-9
    S = _sim(O, model=0, nx=nx, bc=(PER, PER, PER), xlim=(0.0, 1.0), cfl=0.4, sigma=0.0, kappa=kappa, gamma=G43, integrator=integrator)
    dt, dx = S.dt, 1.0 / nx
    x = (np.arange(nx) + 0.5) * dx
    k = 2 * np.pi
    cB, cP = A * np.exp(0.3j), 0.6 * A * np.exp(-1.1j)
    wp = np.zeros((11, 1, 1, nx)); wp[0] = 1.0; wp[4] = 1.0
    S.set_initial(wp, np.zeros((1, 1, nx)))
    q0, _ = S.get_state()
    q0[5] = (cB * np.exp(1j * k * x)).real
    q0[13] = (cP * np.exp(1j * k * x)).real
    assert S.set_cons(q0) == 0
    S.step(1)
    q1, _ = S.get_state()
    S.close()
    th = k * dx
    sp = -np.exp(-1j * th) / 6 + 5 / 6 + np.exp(1j * th) / 3            # left-biased, cells i-1, i, i+1
    sm = -np.exp(2j * th) / 6 + 5 * np.exp(1j * th) / 6 + 1 / 3         # right-biased, cells i+2, i+1, i
    M = np.array([[0, 1], [1, 0]], complex)                             # f = M q
    I2 = np.eye(2)
    Le = -(1 - np.exp(-1j * th)) / dx * (sp * 0.5 * (M + I2) + sm * 0.5 * (M - I2))
    Li = np.diag([0.0, -kappa]).astype(complex)
    c1 = imex_linear_map(Le, Li, dt, at, wt, a, w) @ np.array([cB, cP])
    Bx = (c1[0] * np.exp(1j * k * x)).real
    ph = (c1[1] * np.exp(1j * k * x)).real
    assert np.abs(q1[5, 0, 0] - Bx).max() < 2e-9 * A, np.abs(q1[5, 0, 0] - Bx).max() / A
    assert np.abs(q1[13, 0, 0] - ph).max() < 2e-9 * A, np.abs(q1[13, 0, 0] - ph).max() / A
    return c1


def test_telegraph_mode_pins_the_joint_stage_structure(O):
    c3 = _telegraph_case(O, "ssp3", AT3, WT3, A3, W3)
    c2 = _telegraph_case(O, "ssp2", AT2, WT2, A2, W2)      # the same pin for the SSP2(222) path
    assert abs(c3[0] - c2[0]) > 1e-5 * abs(c2[0])          # the two schemes are distinguishable at this accuracy


def test_general_stepper_with_table2_reproduces_the_ssp222_path(O, synth):
    """step_imex (eq 10-11 written generally) with Table 2 against the hand-written SSP2(222) step: same arithmetic up to
    summation order.  Brio-Wu-like tube (stiff, discontinuous) and a two-fluid periodic box."""
    c = synth.config1()
    kw = dict(c["params"])
    outs = []
    for integ in (0, 2):
        kw["integrator"] = integ
        S = O.OracleSim(O.make_params(**kw)); S.set_initial(c["prims"], c.get("rho_charge")); S.step(10)
        outs.append(S.get_state()[0]); S.close()
    assert np.abs(outs[0] - outs[1]).sum() / np.abs(outs[0]).sum() < 1e-13
    c = synth.config4(nx=24, ny=24, nsteps=4)
    kw = dict(c["params"])
    outs = []
    for integ in (0, 2):
        kw["integrator"] = integ
        S = O.OracleSim(O.make_params(**kw)); S.set_initial(c["prims"]); S.step(4)
        outs.append(S.get_state()[0]); S.close()
    assert np.abs(outs[0] - outs[1]).sum() / np.abs(outs[0]).sum() < 1e-13


def test_ssp3_second_order_in_time_with_stiff_source(O):
    """0-D resistive relaxation with a moving, magnetised fluid (uniform periodic state, L == 0, nonlinear Psi through
    con2prim): SSP3(332) is second order as an IMEX scheme (p = 2 in SSP3(332)); error ratio ~4 when dt halves."""
    errs = []
    ref = None
    for cfl in (0.4 / 256, 0.1, 0.05, 0.025):
        nx = 4
        S = _sim(O, model=0, nx=nx, bc=(PER, PER, PER), xlim=(0.0, 1.0), cfl=cfl, sigma=30.0, kappa=1.0, gamma=G43, integrator="ssp3")
        w = np.zeros((11, 1, 1, nx)); w[0] = 1.0; w[4] = 2.0
        w[1], w[2] = 0.3, -0.2
        w[5], w[6], w[7] = 0.5, 0.4, -0.3
        w[8], w[9], w[10] = 0.2, -0.1, 0.15
        S.set_initial(w, np.zeros((1, 1, nx)))
        n = int(round(0.2 / S.dt))
        assert abs(n * S.dt - 0.2) < 1e-12
        S.step(n)
        q, _ = S.get_state(); S.close()
        if ref is None:
            ref = q
        else:
            errs.append(np.abs(q[8:11] - ref[8:11]).max())
    assert errs[0] > 1e-7
    r1, r2 = errs[0] / errs[1], errs[1] / errs[2]
    assert 3.3 < r1 < 4.8 and 3.5 < r2 < 4.5, (errs, r1, r2)
