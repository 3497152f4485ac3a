"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU).

Each test checks the oracle against something other than itself: hand-computed textbook
values, closed forms, invariants, brute force.  Citations: PAPER.md line numbers ("P:L..")
and the readings G1..G19 of DESIGN.md.
"""
import math
import os

import numpy as np
import pytest

G43 = 4.0 / 3.0
GOLD = os.path.join(os.path.dirname(__file__), "golden")


# ------------------------------------------------------------------------------------------
# prim <-> cons
# ------------------------------------------------------------------------------------------
def test_prim2cons_hand_values_resistive(O):
    """eq (2)-(4) P:L63-71 on a state worked by hand: rho=1, p=1, Gamma=2, v=(0.8,0,0),
    E=(0,1,0), B=(0,0,2): W=5/3, h=3, Z=25/3, D=5/3, ExB=(2,0,0), (E^2+B^2)/2=5/2."""
    P = O.make_params(model=0, gamma=2.0)
    w = np.array([[1.0], [0.8], [0.0], [0.0], [1.0], [0.0], [0.0], [2.0], [0.0], [1.0], [0.0]])
    q = O.prim2cons(P, w, np.array([0.25]))[:, 0]
    expect = [5 / 3, 0.8 * 25 / 3 + 2.0, 0.0, 0.0, 25 / 3 - 1.0 + 2.5 - 5 / 3, 0, 0, 2, 0, 1, 0, 0.25, 0, 0]
    assert np.allclose(q, expect, rtol=1e-14, atol=1e-15)


def test_con2prim_closed_form_zero_momentum(O):
    """S~ = 0 => v = 0, Z = D + Gamma tau~, p = (Gamma-1) tau~, rho = D (SURVEY 8(c) pins)."""
    rng = np.random.default_rng(3)
    n = 2000
    for gam in (G43, 5.0 / 3.0, 2.0):
        P = O.make_params(model=0, gamma=gam)
        D = 10 ** rng.uniform(-2, 2, n)
        taut = 10 ** rng.uniform(-3, 2, n)
        E = rng.standard_normal((3, n)); B = rng.standard_normal((3, n))
        S = np.cross(E.T, B.T).T
        tau = taut + 0.5 * ((E ** 2).sum(0) + (B ** 2).sum(0))
        q = np.concatenate([D[None], S, tau[None], B, E, np.zeros((3, n))])
        w, it, fail = O.con2prim(P, q)
        assert not fail.any()
        assert np.allclose(w[0], D, rtol=1e-13)
        assert np.abs(w[1:4]).max() < 1e-13
        assert np.allclose(w[4], (gam - 1) * taut, rtol=1e-12)


def test_round_trip_resistive(O, synth):
    """con2prim(prim2cons(w)) == w on 2e5 random admissible states (north_star check)."""
    n = 200000
    w = synth.random_resistive_prims(n, seed=11, vmax=0.99)
    P = O.make_params(model=0, gamma=G43)
    rc = np.random.default_rng(5).standard_normal(n)
    q = O.prim2cons(P, w, rc)
    w2, it, fail = O.con2prim(P, q)
    assert not fail.any()
    assert it.max() <= 30
    # conserved variables reproduced to round-off (well conditioned direction)
    q2 = O.prim2cons(P, w2, rc)
    scale = np.abs(q[:5]).max(axis=0)
    assert (np.abs(q2[:5] - q[:5]) / scale).max() < 1e-13
    # primitives: conditioning grows with W^2 and rho/p; bound accordingly
    W2 = 1.0 / (1.0 - (w[1:4] ** 2).sum(0))
    h = 1 + G43 / (G43 - 1) * w[4] / w[0]
    cond = W2 * (1.0 + w[0] * h / w[4])
    assert (np.abs(w2[4] - w[4]) / w[4] / cond).max() < 1e-13
    assert (np.abs(w2[0] - w[0]) / w[0] / cond).max() < 1e-13
    assert (np.abs(w2[1:4] - w[1:4]).max(axis=0) / cond).max() < 1e-13
    assert np.array_equal(w2[5:], w[5:])


def test_round_trip_two_fluid(O, synth):
    n = 100000
    w = synth.random_two_fluid_prims(n, seed=12, vmax=0.9)
    P = O.make_params(model=1, gamma=G43, mu_e=-100.0, mu_p=100.0)
    q = O.prim2cons(P, w)
    w2, it, fail = O.con2prim(P, q)
    assert not fail.any()
    q2 = O.prim2cons(P, w2)
    scale = np.abs(q[:10]).max(axis=0)
    assert (np.abs(q2[:10] - q[:10]) / scale).max() < 1e-12
    for s in range(2):
        ws, w2s = w[5 * s:5 * s + 5], w2[5 * s:5 * s + 5]
        W2 = 1.0 / (1.0 - (ws[1:4] ** 2).sum(0))
        cond = W2 * (1.0 + ws[0] / ws[4] + 5.0) * 20.0   # species split loses ~ |x|/|x_s| digits
        assert (np.abs(w2s[4] - ws[4]) / ws[4] / cond).max() < 1e-12
        assert (np.abs(w2s[1:4] - ws[1:4]).max(axis=0) / cond).max() < 1e-12


def test_two_fluid_prim2cons_hand_values(O):
    """eq (6) P:L95-108 with G2.  Species at rest: rho_e=0.5,p_e=0.5; rho_p=2,p_p=1; Gamma=4/3:
    h_e = 1+4*0.5/0.5 = 5, Z_e = 2.5; h_p = 1+4*1/2 = 3, Z_p = 6.  mu_e=-3, mu_p=2."""
    P = O.make_params(model=1, gamma=G43, mu_e=-3.0, mu_p=2.0)
    w = np.zeros((16, 1))
    w[0], w[4], w[5], w[9] = 0.5, 0.5, 2.0, 1.0
    w[10:13, 0] = (0.0, 0.0, 2.0)
    w[13:16, 0] = (0.0, 1.0, 0.0)
    q = O.prim2cons(P, w)[:, 0]
    D = 2.5; tau = (2.5 - 0.5 - 0.5) + (6 - 1 - 2) + 2.5
    Dbar = -3 * 0.5 + 2 * 2.0; taubar = -3 * (2.5 - 0.5 - 0.5) + 2 * (6 - 1 - 2)
    expect = [D, 2.0, 0, 0, tau, Dbar, 0, 0, 0, taubar, 0, 0, 2, 0, 1, 0, 0, 0]
    assert np.allclose(q, expect, rtol=1e-14, atol=1e-15)
    # moving electrons: v_e = (0.6,0,0): W=1.25, Z_e = 0.5*5*1.5625 = 3.90625
    w[1] = 0.6
    q = O.prim2cons(P, w)[:, 0]
    assert math.isclose(q[0], 0.5 * 1.25 + 2.0, rel_tol=1e-14)
    assert math.isclose(q[1], 3.90625 * 0.6 + 2.0, rel_tol=1e-14)           # S_x incl. ExB
    assert math.isclose(q[6], -3.0 * 3.90625 * 0.6, rel_tol=1e-14)          # Sbar_x carries h_s (G2)
    assert math.isclose(q[5], -3 * 0.5 * 1.25 + 4.0, rel_tol=1e-14)


def test_species_split_is_inverse_of_sums(O):
    """eq (7),(8) P:L128-133: split(sum, weighted sum) returns the species parts."""
    rng = np.random.default_rng(0)
    xe, xp = rng.standard_normal(1000), rng.standard_normal(1000)
    for mu_e, mu_p in ((-100.0, 100.0), (-1836.0, 1.0), (-2.0, 5.0)):
        ge, gp = O.species_split(mu_e, mu_p, xe + xp, mu_e * xe + mu_p * xp)
        assert np.allclose(ge, xe, rtol=1e-11, atol=1e-12) and np.allclose(gp, xp, rtol=1e-11, atol=1e-12)
    with pytest.raises(ValueError):
        O.species_split(3.0, 3.0, xe, xp)


# ------------------------------------------------------------------------------------------
# flux and source vectors
# ------------------------------------------------------------------------------------------
def test_flux_vector_hydro_and_maxwell_parts(O):
    """Textbook limits of eq (1)-(2) P:L57-63.  Pure hydro (E=B=0): f(D)=D v_k,
    f(S_i)=S_i v_k + p delta_ik, f(tau)=(tau+p) v_k.  Fluid at rest: f(tau)=Poynting (ExB)_k,
    f(S_i)=Maxwell stress, f(B)=-curl structure (Faraday), f(E)=+curl structure (Ampere)."""
    P = O.make_params(model=0, gamma=2.0, sigma=7.0)
    w = np.array([[1.0], [0.3], [-0.4], [0.5], [2.0]] + [[0.0]] * 6)
    q = O.prim2cons(P, w, np.array([0.0]))
    for k in range(3):
        f = O.flux_vector(P, k, q, w)[:, 0]
        v = w[1:4, 0]
        assert math.isclose(f[0], q[0, 0] * v[k], rel_tol=1e-14)
        for i in range(3):
            assert math.isclose(f[1 + i], q[1 + i, 0] * v[k] + (2.0 if i == k else 0.0), rel_tol=1e-13, abs_tol=1e-15)
        assert math.isclose(f[4], (q[4, 0] + 2.0) * v[k], rel_tol=1e-13)
    # fluid at rest with fields; psi, phi = 0
    E = np.array([0.3, -0.2, 0.5]); B = np.array([-0.1, 0.7, 0.4])
    w = np.concatenate([[1.0, 0, 0, 0, 1.0], B, E])[:, None]
    q = O.prim2cons(P, w, np.array([0.6]))
    em = 0.5 * (E @ E + B @ B)
    ExB = np.cross(E, B)
    for k in range(3):
        f = O.flux_vector(P, k, q, w)[:, 0]
        assert f[0] == 0.0
        assert math.isclose(f[4], ExB[k], rel_tol=1e-14)
        for i in range(3):
            assert math.isclose(f[1 + i], (1.0 + em if i == k else 0.0) - E[i] * E[k] - B[i] * B[k], rel_tol=1e-13)
        # dB/dt = -curl E  <=>  dB_i/dt + d_k ( -eps_ijk E_j ) = 0 ; e.g. k=y: f(B_x) = +E_z
        a, b = (k + 1) % 3, (k + 2) % 3
        assert f[5 + k] == 0.0 and f[5 + a] == -E[b] and f[5 + b] == E[a]
        assert f[8 + k] == 0.0 and f[8 + a] == B[b] and f[8 + b] == -B[a]
        assert math.isclose(f[11], 7.0 * E[k], rel_tol=1e-14)      # J = sigma E at rest (+ rhoc v = 0)
        assert f[12] == E[k] and f[13] == B[k]


def test_resistive_source_rows(O):
    """eq (1) P:L57 rhs: only E, psi, phi rows are non-zero; J from P:L75 evaluated by hand."""
    P = O.make_params(model=0, gamma=G43, sigma=3.0, kappa=2.0)
    v = np.array([0.5, 0.0, 0.0]); B = np.array([0.0, 1.0, 0.0]); E = np.array([0.2, 0.0, 0.3])
    w = np.concatenate([[1.0], v, [1.0], B, E])[:, None]
    q = O.prim2cons(P, w, np.array([0.4]))
    q[12], q[13] = 0.7, -0.2
    s = O.source(P, q, w)[:, 0]
    W = 1 / math.sqrt(0.75)
    vxB = np.cross(v, B); vE = v @ E
    J = 0.4 * v + W * 3.0 * (E + vxB - vE * v)
    assert np.all(s[:8] == 0.0) and s[11] == 0.0
    assert np.allclose(s[8:11], -J, rtol=1e-14)
    assert math.isclose(s[12], 0.4 - 2.0 * 0.7, rel_tol=1e-14) and math.isclose(s[13], 0.4, rel_tol=1e-14)


def test_two_fluid_source_is_weighted_lorentz_force(O, synth):
    """(A2)-(A3) P:L445-451 with G2: at eta = 0 the Sbar / taubar sources must equal the
    mu-weighted sums of the per-species Lorentz force and Joule work,
    sum_s mu_s (mu_s rho_s W_s)(E + v_s x B) and sum_s mu_s (mu_s rho_s W_s) v_s.E."""
    n = 500
    w = synth.random_two_fluid_prims(n, seed=4)
    P = O.make_params(model=1, gamma=G43, mu_e=-7.0, mu_p=3.0, eta=0.0, kappa=1.0)
    q = O.prim2cons(P, w)
    s = O.source(P, q, w)
    B, E = w[10:13], w[13:16]
    F = np.zeros((3, n)); Wk = np.zeros(n); J = np.zeros((3, n)); rhoc = np.zeros(n)
    for sp, mu in ((0, -7.0), (1, 3.0)):
        rho, v = w[5 * sp], w[5 * sp + 1:5 * sp + 4]
        W = 1 / np.sqrt(1 - (v ** 2).sum(0))
        qd = mu * rho * W
        F += mu * qd * (E + np.cross(v.T, B.T).T)
        Wk += mu * qd * (v * E).sum(0)
        J += qd * v; rhoc += qd
    assert np.allclose(s[6:9], F, rtol=1e-12, atol=1e-12)
    assert np.allclose(s[9], Wk, rtol=1e-12, atol=1e-12)
    assert np.allclose(s[13:16], -J, rtol=1e-13, atol=1e-13)
    assert np.allclose(s[16], rhoc - q[16], rtol=1e-13, atol=1e-13)
    assert np.all(s[:6] == 0.0) and np.all(s[10:13] == 0.0)


def test_two_fluid_friction_vanishes_and_opposes_current(O):
    """Friction -eta wp^2 (J - rho0 u): zero for co-moving species; in the frame u = 0 it is
    -eta wp^2 J (opposes the current)."""
    mu = 50.0
    P0 = O.make_params(model=1, gamma=G43, mu_e=-mu, mu_p=mu, eta=0.0)
    P1 = O.make_params(model=1, gamma=G43, mu_e=-mu, mu_p=mu, eta=0.01)
    w = np.zeros((16, 1)); w[0] = w[5] = 0.5; w[4] = w[9] = 0.5
    w[1] = w[6] = 0.3                      # co-moving
    q = O.prim2cons(P0, w)
    assert np.allclose(O.source(P1, q, w), O.source(P0, q, w), atol=1e-12)
    w[1], w[6] = -0.3, 0.3                 # counter-streaming: u = 0, J_x = 2 mu rho W v
    q = O.prim2cons(P0, w)
    d = (O.source(P1, q, w) - O.source(P0, q, w))[:, 0]
    W = 1 / math.sqrt(1 - 0.09)
    Jx = 2 * mu * 0.5 * W * 0.3; wp2 = 2 * mu * mu * 0.5
    assert math.isclose(d[6], -0.01 * wp2 * Jx, rel_tol=1e-12)
    assert abs(d[7]) < 1e-12 and abs(d[8]) < 1e-12


# ------------------------------------------------------------------------------------------
# WENO3
# ------------------------------------------------------------------------------------------
def test_weno3_linear_exact_and_equal_beta(O):
    rng = np.random.default_rng(1)
    a0, s = rng.standard_normal(100), rng.standard_normal(100)
    # linear data u_j = a0 + s j at j=-1,0,1: face value at +1/2 is a0 + s/2
    out = O.weno3(a0 - s, a0, a0 + s)
    assert np.allclose(out, a0 + 0.5 * s, rtol=1e-14, atol=1e-15)
    # equal smoothness indicators (c-b = -(b-a)) -> optimal weights: -a/6 + 5b/6 + c/3
    a, b = rng.standard_normal(100), rng.standard_normal(100)
    c = a.copy()   # symmetric extremum: beta0 == beta1 exactly
    out = O.weno3(a, b, c)
    assert np.allclose(out, -a / 6 + 5 * b / 6 + c / 3, rtol=1e-13, atol=1e-14)
    # constant data reproduced to an ulp
    assert np.allclose(O.weno3(b, b, b), b, rtol=4e-16, atol=0)


def test_weno3_third_order_on_smooth_data(O):
    """Cell averages of sin(x): face value error falls as h^3 away from critical points."""
    errs = []
    for n in (20, 40, 80):
        h = 1.0 / n
        x0 = 0.3
        avg = lambda xc: (np.cos(xc - h / 2) - np.cos(xc + h / 2)) / h
        out = O.weno3(np.array([avg(x0 - h)]), np.array([avg(x0)]), np.array([avg(x0 + h)]))[0]
        errs.append(abs(out - math.sin(x0 + h / 2)))
    assert math.log2(errs[0] / errs[1]) > 2.7 and math.log2(errs[1] / errs[2]) > 2.7


def test_weno3_discontinuity_picks_smooth_stencil(O):
    # step between b and c: left-biased value stays near the smooth stencil {a,b} -> ~ (3b-a)/2
    out = O.weno3(np.array([1.0]), np.array([1.0]), np.array([0.0]))[0]
    assert abs(out - 1.0) < 1e-9
    out = O.weno3(np.array([0.0]), np.array([1.0]), np.array([1.0]))[0]
    assert abs(out - 1.0) < 1e-9


# ------------------------------------------------------------------------------------------
# implicit stage
# ------------------------------------------------------------------------------------------
def _stage_R(z):
    g = 1 - 1 / math.sqrt(2)
    k1 = 1 / (1 - g * z)
    k2 = (1 + (1 - 2 * g) * z * k1) / (1 - g * z)
    return 1 + 0.5 * z * (k1 + k2)


def test_golden_stability_function_value():
    val = None
    for line in open(os.path.join(GOLD, "ssp222_table2.txt")):
        if line.startswith("R(-1)"):
            val = float(line.split()[1])
    assert abs(_stage_R(-1.0) - val) < 1e-12
    assert abs(_stage_R(-1e12)) < 1e-10          # L-stable


def test_stage_closed_form_fluid_at_rest(O):
    """B = 0, rhoc = 0, S = 0  =>  v = 0, J = sigma E,  E* = E_ex/(1 + a sigma);
    psi* = (psi_ex + a rhoc)/(1 + a kappa), phi* = phi_ex/(1 + a kappa)."""
    n = 64
    rng = np.random.default_rng(9)
    P = O.make_params(model=0, gamma=G43, kappa=1.5)
    sig = 10 ** rng.uniform(0, 6, n)
    E = 0.1 * rng.standard_normal((3, n))
    w = np.concatenate([np.ones((1, n)), np.zeros((3, n)), np.ones((1, n)), np.zeros((3, n)), E])
    rhoc = np.zeros(n)
    q_ex = O.prim2cons(P, w, rhoc)
    q_ex[12] = rng.standard_normal(n); q_ex[13] = rng.standard_normal(n)
    a = 2.0e-3
    q, wout, it, fail = O.stage_batch(P, q_ex, w, a, sig)
    assert not fail.any()
    assert np.allclose(q[8:11], q_ex[8:11] / (1 + a * sig), rtol=1e-12, atol=1e-16)
    assert np.allclose(q[12], q_ex[12] / (1 + a * 1.5), rtol=1e-13)
    assert np.allclose(q[13], q_ex[13] / (1 + a * 1.5), rtol=1e-13)
    assert np.array_equal(q[:8], q_ex[:8]) or np.allclose(q[:8], q_ex[:8], rtol=1e-15, atol=1e-16)
    # with charge: v = 0 still (S = 0, B = 0): psi* = (psi_ex + a rhoc)/(1 + a kappa)
    rhoc = rng.standard_normal(n)
    q_ex[11] = rhoc
    q, wout, it, fail = O.stage_batch(P, q_ex, w, a, sig)
    assert np.allclose(q[12], (q_ex[12] + a * rhoc) / (1 + a * 1.5), rtol=1e-12, atol=1e-15)


def test_stage_guess_equals_sherman_morrison(O, synth):
    """I.3: frozen-(v,W) solve M E = b equals the closed-form inverse (Sherman-Morrison)."""
    c = synth.config2(2000, seed=3)
    P = O.make_params(**c["params"])
    w = c["prims"]; sig = c["sigma_cell"]; a = c["a_dt"]
    rc = np.random.default_rng(1).standard_normal(w.shape[1])
    q_ex = O.prim2cons(P, w, rc)
    Eg = O.stage_guess(P, q_ex, w, a, sig)
    v, B = w[1:4], w[5:8]
    W = 1 / np.sqrt(1 - (v ** 2).sum(0)); s = a * W * sig
    b = q_ex[8:11] - a * rc * v - s * np.cross(v.T, B.T).T
    Esm = (b + s * v * (v * b).sum(0) / (1 + s - s * (v ** 2).sum(0))) / (1 + s)
    assert np.allclose(Eg, Esm, rtol=1e-11, atol=1e-13)


def test_stage_solution_satisfies_eq10_by_independent_residual(O, synth):
    """Residual of eq (10) P:L152 recomputed in numpy from the returned (q*, prims*)."""
    c = synth.config2(4000, seed=0)
    P = O.make_params(**c["params"])
    w = c["prims"]; sig = c["sigma_cell"]; a = c["a_dt"]
    q_ex = O.prim2cons(P, w)
    q, ws, it, fail = O.stage_batch(P, q_ex, w, a, sig)
    assert fail.sum() == 0
    v, B, E = ws[1:4], ws[5:8], q[8:11]
    W = 1 / np.sqrt(1 - (v ** 2).sum(0))
    J = q[11] * v + W * sig * (E + np.cross(v.T, B.T).T - (v * E).sum(0) * v)
    R = E - q_ex[8:11] + a * J
    scale = 1 + a * W * sig * (np.abs(E) + np.abs(np.cross(v.T, B.T).T)).max(0)
    assert (np.abs(R).max(0) / scale).max() < 5e-14
    # returned prims are the con2prim of the returned q*
    q_chk = O.prim2cons(P, ws, q[11])
    assert (np.abs(q_chk[:5] - q[:5]).max(0) / np.abs(q[:5]).max(0)).max() < 1e-12
    # zero-source rows untouched
    assert np.allclose(q[:8], q_ex[:8], rtol=1e-14, atol=1e-15) and np.allclose(q[11], q_ex[11])
    assert it.max() <= 12


def test_stage_root_is_unique_from_random_guesses(O, synth):
    """G19: Newton from 20 perturbed guesses lands on one root (64 cells)."""
    c = synth.config2(64, seed=5)
    P = O.make_params(**c["params"])
    w = c["prims"]; sig = c["sigma_cell"]; a = c["a_dt"]
    q_ex = O.prim2cons(P, w)
    q0, w0, _, fail0 = O.stage_batch(P, q_ex, w, a, sig)
    assert not fail0.any()
    rng = np.random.default_rng(0)
    for t in range(20):
        wg = w.copy()
        wg[0] *= 10 ** rng.uniform(-0.3, 0.3, 64)
        wg[4] *= 10 ** rng.uniform(-0.3, 0.3, 64)
        wg[1:4] *= rng.uniform(0.0, 1.05, 64)
        wg[1:4] += 0.02 * rng.standard_normal((3, 64))
        q1, w1, _, fail1 = O.stage_batch(P, q_ex, wg, a, sig)
        ok = fail1 == 0
        assert ok.mean() > 0.9
        assert np.abs(q1[:, ok] - q0[:, ok]).max() < 1e-10


def test_two_fluid_stage_residual_and_fixed_rows(O, synth):
    n = 500
    w = synth.random_two_fluid_prims(n, seed=8, vmax=0.5)
    w[10:16] *= 0.1    # N(0,1) fields with mu = 100 fling the light species out of the admissible set
    P = O.make_params(model=1, gamma=G43, mu_e=-100.0, mu_p=100.0, eta=1e-3)
    q_ex = O.prim2cons(P, w)
    a = 1e-4
    q, ws, it, fail = O.stage_batch(P, q_ex, w, a)
    assert fail.sum() == 0
    # rows D, S, tau, Dbar, B have zero source (A2 P:L445)
    for r in (0, 1, 2, 3, 4, 5, 10, 11, 12):
        assert np.allclose(q[r], q_ex[r], rtol=1e-14, atol=1e-14)
    s = O.source(P, q, ws)
    R = q - q_ex - a * s
    scale = np.abs(q).max(0) + a * np.abs(s).max(0)
    assert (np.abs(R).max(0) / scale).max() < 1e-12
    # psi*, phi* closed forms with rhoc = Dbar
    assert np.allclose(q[16], (q_ex[16] + a * q_ex[5]) / (1 + a), rtol=1e-12, atol=1e-14)


def test_two_fluid_flux_is_sum_of_single_fluid_hydro_fluxes(O, synth):
    """(A1) P:L443 with G2: without fields the two-fluid flux rows are the plain / mu-weighted
    sums of the two species' single-fluid hydro fluxes (computed by the resistive model, itself
    pinned against textbook values above); with the fluid at rest they are the Maxwell rows."""
    n = 300
    w = synth.random_two_fluid_prims(n, seed=21, vmax=0.8)
    w[10:16] = 0.0
    mu_e, mu_p = -7.0, 3.0
    P2 = O.make_params(model=1, gamma=G43, mu_e=mu_e, mu_p=mu_p)
    P1 = O.make_params(model=0, gamma=G43, sigma=0.0)
    q2 = O.prim2cons(P2, w)
    zeros = np.zeros((6, n))
    fs = []
    for s in range(2):
        w1 = np.concatenate([w[5 * s:5 * s + 5], zeros])
        q1 = O.prim2cons(P1, w1)
        fs.append([O.flux_vector(P1, k, q1, w1) for k in range(3)])
    for k in range(3):
        f = O.flux_vector(P2, k, q2, w)
        fe, fp = fs[0][k], fs[1][k]
        assert np.allclose(f[0:5], fe[0:5] + fp[0:5], rtol=1e-12, atol=1e-13)
        assert np.allclose(f[5:10], mu_e * fe[0:5] + mu_p * fp[0:5], rtol=1e-12, atol=1e-12)
        assert np.all(f[10:] == 0.0)
    # fields only, species at rest: Maxwell rows identical to the resistive model's
    rng = np.random.default_rng(2)
    E = rng.standard_normal((3, n)); B = rng.standard_normal((3, n))
    w[1:4] = 0.0; w[6:9] = 0.0; w[10:13] = B; w[13:16] = E
    q2 = O.prim2cons(P2, w); q2[16] = rng.standard_normal(n); q2[17] = rng.standard_normal(n)
    w1 = np.concatenate([w[0:1] + w[5:6], np.zeros((3, n)), w[4:5] + w[9:10], B, E])
    q1 = O.prim2cons(P1, w1); q1[12] = q2[16]; q1[13] = q2[17]
    for k in range(3):
        f = O.flux_vector(P2, k, q2, w); f1 = O.flux_vector(P1, k, q1, w1)
        assert np.allclose(f[1:5], f1[1:5], rtol=1e-12, atol=1e-13)      # stress + Poynting
        assert np.array_equal(f[10:16], f1[5:11])                          # Faraday / Ampere rows
        assert np.array_equal(f[16], f1[12]) and np.array_equal(f[17], f1[13])
