"""Parity of the CUDA path (through the C-ABI) against the CPU oracle, element by element on
the same seeded inputs.  Run on the B200 box:  python -m pytest tests -m gpu

Tolerances: per-cell algebra 1e-12..1e-13 relative; config
runs use BASELINE.json's rel-L1 bounds (cfg1 1e-9, cfg2 1e-10, cfg3/4/5 1e-8), where
rel-L1 = sum |q_gpu - q_oracle| / sum |q_oracle| over all conserved variables and cells, AND, per conserved variable,
sum |q_gpu - q_oracle| / max(sum |q_oracle|, N 1e-8) <= 1e-11: the global sum is dominated by tau and B,
a defect in a small row (psi, phi, rho_charge) would not show in it.
"""
import json
import os
import time

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

G43 = 4.0 / 3.0


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device (there is no CPU fallback)")
    from paper_1808_09721_b200 import build, binding
    build.build()
    binding.lib()
    return binding


def rel_l1(a, b):
    return np.abs(a - b).sum() / np.abs(b).sum()


PER_VAR_TOL = 1e-11            # resistive model (measured: <= 5e-13)
PER_VAR_TOL_TWO_FLUID = 1e-13  # x mu^2, capped at the case's global bound: two-fluid model, 1e-9 for |mu| = 100 (measured: <= 2.6e-10), see rel_l1_per_var


def two_fluid_per_var_tol(mu, tol):
    """1e-13 mu^2, but never looser than the global rel-L1 bound `tol` of the case: at |mu| >= 316 the mu^2 law would allow more
    in one row than BASELINE.json allows in the sum over all rows (mu = 1e3: 1e-7 against 1e-8), and the check would say nothing."""
    return min(PER_VAR_TOL_TWO_FLUID * mu ** 2, tol)


def rel_l1_per_var(a, b, mu=None):
    """per conserved variable, sum |a - b| / max(sum |b|, N 1e-8) (several rows are identically ~0 in cfg1 / cfg5).
    Two-fluid model (18 rows, `mu` = max |mu_s|): the barred rows Dbar, Sbar, taubar are sums over species weighted by
    mu_s = -+mu that cancel for a neutral pair plasma (they are identically ~0 in cfg4), so their round-off is mu eps times
    the unbarred row: the denominator of row v in 5..9 is max(sum |b_v|, mu sum |b_{v-5}|); the cleaning fields psi, phi vanish
    identically there too and are measured against 1e-6 of the field they clean (E, B).  That noise is fed back through the
    source with omega_p^2 = sum mu_s^2 rho_s ~ mu^2 (A2 P:L445): the FMA / no-FMA difference of the two sides shows up at
    ~mu^2 eps per step in E and psi, which is why the two-fluid bound is 1e-13 mu^2 (1e-9 for cfg4) and not 1e-11."""
    n = b[0].size
    out = []
    for v in range(b.shape[0]):
        den = max(np.abs(b[v]).sum(), n * 1e-8)
        if mu is not None and 5 <= v <= 9:
            den = max(den, mu * np.abs(b[v - 5]).sum())
        if mu is not None and v >= 16:      # psi, phi vanish identically in cfg4: their round-off is eps |E|, eps |B| per step
            den = max(den, 1e-6 * np.abs(b[13:16] if v == 16 else b[10:13]).sum() / 3.0)
        out.append(np.abs(a[v] - b[v]).sum() / den)
    return np.array(out)


def check_state(name, q, qo, tol, params=None, per_var_tol=None):
    """Global rel-L1 <= the BASELINE.json bound and every variable's rel-L1 <= 1e-11 (two-fluid: min(1e-13 mu^2, tol), mu = the larger
    |mu_s| of the case's own `params`, which a two-fluid case must pass); the measured values go to
    gpurun_out/parity_values.jsonl when RMHD_PARITY_LOG is set (they are quoted in BASELINE.md section 4)."""
    two_fluid = qo.shape[0] == 18
    mu = None
    if two_fluid:
        assert params is not None and "mu_e" in params and "mu_p" in params, "two-fluid case: pass the case's params (mu_e, mu_p)"
        mu = max(abs(params["mu_e"]), abs(params["mu_p"]))
    if per_var_tol is None:
        per_var_tol = two_fluid_per_var_tol(mu, tol) if two_fluid else PER_VAR_TOL
    g = float(rel_l1(q, qo)); pv = rel_l1_per_var(q, qo, mu)
    if os.environ.get("RMHD_PARITY_LOG"):
        os.makedirs("gpurun_out", exist_ok=True)
        with open("gpurun_out/parity_values.jsonl", "a") as f:
            f.write(json.dumps({"case": name, "rel_l1": g, "per_var_max": float(pv.max()), "per_var_tol": per_var_tol,
                                "per_var": [float(x) for x in pv]}) + "\n")
    assert g <= tol, (name, g)
    assert pv.max() <= per_var_tol, (name, int(pv.argmax()), pv)
    return g, pv


def run_gpu(B, cfg, nsteps=None, params_override=None):
    kw = dict(cfg["params"])
    if params_override:
        kw.update(params_override)
    sim = B.Rmhd(**kw)
    sim.set_initial(np.ascontiguousarray(cfg["prims"]), cfg.get("rho_charge"))
    sim.step(cfg["nsteps"] if nsteps is None else nsteps)
    cons, prims = sim.get_state()
    stats = sim.stats()
    sim.close()
    return cons, prims, stats


def run_oracle(O, cfg, nsteps=None, params_override=None):
    kw = dict(cfg["params"])
    if params_override:
        kw.update(params_override)
    S = O.OracleSim(O.make_params(**kw))
    S.set_initial(cfg["prims"], cfg.get("rho_charge"))
    rc = S.step(cfg["nsteps"] if nsteps is None else nsteps)
    cons, prims = S.get_state()
    stats = S.get_stats()
    S.close()
    assert rc == 0
    return cons, prims, stats


# ------------------------------------------------------------------------------------------
# per-cell kernels
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n", [0, 1, 33, 4099])
def test_prim2cons_con2prim_batch_resistive(B, O, synth, n):
    w = synth.random_resistive_prims(n, seed=3, vmax=0.99)
    rc = np.random.default_rng(1).standard_normal(n)
    P = B.make_params(model=0, gamma=G43)
    PO = O.make_params(model=0, gamma=G43)
    q = np.empty((14, n))
    B.rmhd_prim2cons_batch(P, w, q, rc)
    if n == 0:
        return
    qo = O.prim2cons(PO, w, rc)
    assert rel_l1(q, qo) < 1e-14
    assert (np.abs(q - qo) / np.abs(qo[:5]).max(axis=0)).max() < 1e-14
    # con2prim on the oracle's conserved state, no guess
    w2 = np.empty((11, n)); it = np.zeros(n, np.int32); fl = np.zeros(n, np.int32)
    B.rmhd_con2prim_batch(P, qo, w2, None, it, fl)
    wo, ito, flo = O.con2prim(PO, qo)
    assert not fl.any() and not flo.any()
    W2 = 1.0 / (1.0 - (w[1:4] ** 2).sum(0))
    cond = W2 * (1.0 + w[0] * (1 + 4 * w[4] / w[0]) / w[4])
    err = (np.abs(w2[:5] - wo[:5]) / np.maximum(np.abs(wo[:5]), 1e-3) / cond).max()
    if os.environ.get("RMHD_PARITY_LOG"):
        os.makedirs("gpurun_out", exist_ok=True)
        with open("gpurun_out/parity_values.jsonl", "a") as f:
            f.write(json.dumps({"case": "con2prim batch n=%d" % n, "max_err_over_cond": float(err)}) + "\n")
    assert err < 1e-12       # both sides stop at |dZ| <= 1e-13 Z with the update applied; measured 3.3e-13
    assert np.array_equal(w2[5:], wo[5:])
    assert np.abs(it - ito).max() <= 1


def test_prim2cons_con2prim_batch_two_fluid(B, O, synth):
    n = 5000
    w = synth.random_two_fluid_prims(n, seed=5, vmax=0.9)
    kw = dict(model=1, gamma=G43, mu_e=-100.0, mu_p=100.0)
    P, PO = B.make_params(**kw), O.make_params(**kw)
    q = np.empty((18, n))
    B.rmhd_prim2cons_batch(P, w, q)
    qo = O.prim2cons(PO, w)
    assert (np.abs(q - qo) / np.abs(qo[:10]).max(axis=0)).max() < 1e-14
    w2 = np.empty((16, n)); it = np.zeros(n, np.int32); fl = np.zeros(n, np.int32)
    B.rmhd_con2prim_batch(P, qo, w2, w, it, fl)
    wo, ito, flo = O.con2prim(PO, qo, w)
    assert not fl.any() and not flo.any()
    assert (np.abs(w2 - wo) / np.maximum(np.abs(wo), 1e-2)).max() < 1e-9      # both sit at the same root
    assert rel_l1(w2, wo) < 1e-13


@pytest.mark.parametrize("gamma", [4.0 / 3.0, 2.0])
def test_con2prim_hard_tail_parity(B, O, synth, gamma):
    """2^20 states with W up to 100, p/rho in [1e-8, 1e4], B^2/rho up to 1e4, E near -v x B,
    no guess.  Both sides recover every cell; failure flags are identical; iteration counts agree to +-1 where the first
    residual converges; for Gamma = 2 some cells take the second residual (quartic in W) on both sides.  The recovered
    states are compared through the conserved state they reproduce (oracle prim2cons), in units of eps W^2."""
    n = 1 << 20
    w0 = synth.stress_resistive_prims(n, seed=11)
    P, PO = B.make_params(model=0, gamma=gamma), O.make_params(model=0, gamma=gamma)
    q = O.prim2cons(PO, w0)
    w = np.empty((11, n)); it = np.zeros(n, np.int32); fl = np.zeros(n, np.int32)
    B.rmhd_con2prim_batch(P, q, w, None, it, fl)
    wo, ito, flo = O.con2prim(PO, q)
    assert not fl.any() and not flo.any()
    first = (it <= 20) & (ito <= 20)
    # where the first residual is far from its round-off floor both sides take the same path; in the stalled tail (Gamma = 2, W > 28,
    # p/rho > 600: the Newton update hovers around the tolerance) the counts differ by a few iterations on a handful of cells
    if gamma < 1.9:
        assert np.abs(it - ito).max() <= 1
    assert (np.abs(it - ito) > 1).mean() < 0.02 and np.abs(it - ito).max() <= 45     # measured 0.8 %, max 32 (Gamma = 2: one side converges at the tolerance, the other stalls into the fall-back)
    assert first.mean() > 0.9999 and it.max() <= 45
    if gamma > 1.9:
        assert (it > 20).sum() >= 1 and (ito > 20).sum() >= 1            # the fall-back runs on both sides (not on identical cells:
        #                                                                  which cells stall at the tolerance is round-off dependent)
    W = 1 / np.sqrt(1 - (w0[1:4] ** 2).sum(0))
    eps = np.finfo(float).eps
    scale = np.abs(q[4]) + q[0] + np.sqrt((q[1:4] ** 2).sum(0))
    for ww in (w, wo):
        q2 = O.prim2cons(PO, ww, q[11])
        assert ((np.abs(q2[:5] - q[:5]).max(0) / scale) / (eps * W ** 2)).max() < 64
    # element-wise where the problem is well conditioned (W < 10, 1e-4 < p/rho < 1e2, B^2 < rho: no large E x B to subtract)
    good = (W < 10) & (w0[4] / w0[0] > 1e-4) & (w0[4] / w0[0] < 1e2) & ((w0[5:8] ** 2).sum(0) < w0[0])
    assert (np.abs(w[:5] - wo[:5]) / np.maximum(np.abs(wo[:5]), 1e-300))[:, good].max() < 1e-9


# ------------------------------------------------------------------------------------------
# config 2: batched implicit stage
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n", [1, 31, 2 ** 16 + 37, 2 ** 20])      # 2^20 = BASELINE.json configs[1] in full
def test_config2_stage_batch_parity(B, O, synth, n):
    c = synth.config2(n, seed=0)
    P = B.make_params(**c["params"]); PO = O.make_params(**c["params"])
    w = c["prims"]; sig = c["sigma_cell"]; a = c["a_dt"]
    q_ex = O.prim2cons(PO, w)       # identical input to both sides
    qo, wo, ito, flo = O.stage_batch(PO, q_ex, w, a, sig)
    q = np.empty_like(q_ex); wg = np.empty_like(w); it = np.zeros(n, np.int32); fl = np.zeros(n, np.int32)
    B.rmhd_stage_batch(P, q_ex, w, a, q, wg, sig, it, fl)
    ok = (fl == 0) & (flo == 0)
    assert (fl != 0).sum() <= max(1, 1e-5 * n) and (flo != 0).sum() <= max(1, 1e-5 * n)
    assert ((fl != 0) != (flo != 0)).sum() <= max(1, 1e-5 * n)
    assert rel_l1(q[:, ok], qo[:, ok]) <= 1e-10          # BASELINE.json configs[1] tolerance
    assert rel_l1(q[:, ok], qo[:, ok]) <= 1e-14          # in fact both sit at round-off
    assert np.abs(q[8:11, ok] - qo[8:11, ok]).max() < 1e-12
    assert rel_l1(wg[:, ok], wo[:, ok]) < 1e-13
    assert it[ok].min() >= 1 and it[ok].max() <= 12


def test_config2_device_buffers_and_own_prim2cons(B, O, synth):
    """Same call with torch CUDA tensors (the launch configuration bench.py times), q_ex made by the
    library's own prim2cons."""
    import torch
    n = 2 ** 16
    c = synth.config2(n, seed=0)
    P = B.make_params(**c["params"]); PO = O.make_params(**c["params"])
    dev = torch.device("cuda", 0)
    w = torch.from_numpy(c["prims"]).to(dev); sig = torch.from_numpy(c["sigma_cell"]).to(dev)
    q_ex = torch.empty((14, n), dtype=torch.float64, device=dev)
    B.rmhd_prim2cons_batch(P, w, q_ex)
    q = torch.empty_like(q_ex); wg = torch.empty_like(w)
    it = torch.zeros(n, dtype=torch.int32, device=dev); fl = torch.zeros(n, dtype=torch.int32, device=dev)
    B.rmhd_stage_batch(P, q_ex, w, c["a_dt"], q, wg, sig, it, fl)
    torch.cuda.synchronize()
    qo, wo, ito, flo = O.stage_batch(PO, O.prim2cons(PO, c["prims"]), c["prims"], c["a_dt"], c["sigma_cell"])
    ok = (fl.cpu().numpy() == 0) & (flo == 0)
    assert ok.mean() > 1 - 1e-5
    assert rel_l1(q.cpu().numpy()[:, ok], qo[:, ok]) <= 1e-10


@pytest.mark.parametrize("n,mu,eta,a", [(1, 100.0, 1e-4, 2e-4), (37, 100.0, 1e-4, 2e-4), (2 ** 14 + 5, 100.0, 1e-4, 2e-4),
                                        (4099, 1e3, 1e-2, 3e-4), (4099, 1e4, 1e-3, 3e-4), (4099, 1e3, 1.0, 3e-3),
                                        (4099, 10.0, 0.0, 1e-2)])
def test_two_fluid_stage_batch_parity(B, O, synth, n, mu, eta, a):
    """Two-fluid implicit stage (7+2 unknowns on the GPU, full N=18 Newton in the oracle) on random
    admissible states; mu = 1e3, 1e4 are the paper's stiff regimes (a wp ~ 0.3..30)."""
    w = synth.random_two_fluid_prims(n, seed=11, vmax=0.8)
    w[10:] *= 0.3
    if mu >= 1e3:     # stiff: start near the quasi-neutral, drift-free, ideal-Ohm state (else most cells have no root)
        rng = np.random.default_rng(12)
        w[5] = w[0] * (1 + 1e-4 * rng.standard_normal(n))
        w[6:9] = w[1:4] + 1e-4 * rng.standard_normal((3, n))
        w[13:16] = -np.cross(w[1:4], w[10:13], axis=0) + 1e-3 * rng.standard_normal((3, n))
    kw = dict(model=1, gamma=G43, mu_e=-mu, mu_p=mu, eta=eta)
    P, PO = B.make_params(**kw), O.make_params(**kw)
    q_ex = O.prim2cons(PO, w)
    qo, wo, ito, flo = O.stage_batch(PO, q_ex, w, a)
    q = np.empty_like(q_ex); wg = np.empty_like(w); it = np.zeros(n, np.int32); fl = np.zeros(n, np.int32)
    B.rmhd_stage_batch(P, q_ex, w, a, q, wg, None, it, fl)
    ok = (fl == 0) & (flo == 0)
    assert ((fl != 0) != (flo != 0)).sum() <= max(1, 1e-3 * n), ((fl != 0).sum(), (flo != 0).sum())
    assert ok.sum() >= 0.95 * n          # the random non-neutral case has ~3 % cells with no admissible root (both sides flag them)
    assert rel_l1(q[:, ok], qo[:, ok]) <= 1e-10, rel_l1(q[:, ok], qo[:, ok])
    assert rel_l1(wg[:, ok], wo[:, ok]) <= 1e-10
    # rows without a source are copied through unchanged
    for r in (0, 1, 2, 3, 4, 5, 10, 11, 12):
        assert np.array_equal(q[r], q_ex[r])
    assert it[ok].min() >= 1 and np.percentile(it[ok], 99) <= 8 and it[ok].max() <= 50


# ------------------------------------------------------------------------------------------
# L(q): flux-vector splitting + WENO3 + divergence, virtual ghost zones
# ------------------------------------------------------------------------------------------
def _random_state(model, shape, seed):
    rng = np.random.default_rng(seed)
    nz, ny, nx = shape
    np_ = 11 if model == 0 else 16
    w = np.zeros((np_, nz, ny, nx))
    for s in range(1 if model == 0 else 2):
        w[5 * s] = 10 ** rng.uniform(-0.5, 0.5, shape)
        w[5 * s + 4] = 10 ** rng.uniform(-1, 0.5, shape)
        w[5 * s + 1:5 * s + 4] = rng.uniform(-0.5, 0.5, (3,) + shape)
    w[-6:] = 0.3 * rng.standard_normal((6,) + shape)
    return w


@pytest.mark.parametrize("model,shape,bc", [
    (0, (1, 1, 67), (0, 0, 0)), (0, (1, 1, 130), (1, 1, 1)), (0, (1, 9, 70), (1, 0, 0)), (0, (1, 33, 5), (0, 1, 0)),
    (0, (7, 10, 35), (0, 1, 0)), (0, (11, 3, 66), (1, 0, 1)), (0, (9, 1, 40), (0, 0, 1)),
    (0, (37, 6, 33), (1, 1, 1)), (0, (50, 5, 40), (0, 0, 0)), (0, (2, 2, 2), (1, 0, 1)), (1, (35, 6, 33), (0, 1, 1)),
    # even nx, 3-D, resistive: partial x / y tiles and several z segments of k_flux_hm with 8-row tiles (ny >= 8) and 4-row tiles, both BCs
    (0, (7, 10, 34), (0, 1, 0)), (0, (20, 19, 70), (1, 0, 1)), (0, (5, 8, 32), (0, 0, 0)), (0, (40, 16, 64), (1, 1, 1)),
    (0, (3, 2, 4), (1, 1, 0)), (0, (33, 9, 30), (0, 0, 1)),
    (1, (1, 1, 67), (1, 0, 0)), (1, (1, 12, 37), (0, 1, 0)), (1, (6, 9, 34), (1, 1, 0)),
])
def test_flux_divergence_parity(B, O, model, shape, bc):
    nz, ny, nx = shape
    w = _random_state(model, shape, seed=nx + 7 * ny + 13 * nz)
    kw = dict(model=model, nx=nx, ny=ny, nz=nz, bc=bc, xlim=(0.0, 1.0), ylim=(-1.0, 0.5), zlim=(0.0, 0.7), gamma=G43,
              sigma=25.0, eta=1e-3, mu_e=-20.0, mu_p=10.0)
    rc = np.random.default_rng(0).standard_normal(shape) if model == 0 else None
    sim = B.Rmhd(**kw); sim.set_initial(w, rc)
    L = sim.flux_divergence()
    q, _ = sim.get_state()
    sim.close()
    S = O.OracleSim(O.make_params(**kw)); S.set_initial(w, rc)
    Lo = S.eval_L(); qo, _ = S.get_state()
    assert (np.abs(q - qo) / (np.abs(qo).max() + 1)).max() < 1e-14
    scale = np.abs(Lo).max(axis=(1, 2, 3), keepdims=True) + 1e-30
    assert (np.abs(L - Lo) / scale).max() < 1e-12, np.unravel_index(np.argmax(np.abs(L - Lo) / scale), L.shape)


def test_gauss_law_initialisation_matches(B, O, synth):
    c = synth.config3(nx=48, ny=40, nsteps=1)
    q, _, _ = run_gpu(B, c, nsteps=0)
    qo, _, _ = run_oracle(O, c, nsteps=0)
    assert np.abs(qo[11]).max() > 1.0          # the shear layer carries charge (G10)
    assert np.abs(q[11] - qo[11]).max() < 1e-12 * np.abs(qo[11]).max()


# ------------------------------------------------------------------------------------------
# full configs
# ------------------------------------------------------------------------------------------
def test_config1_riemann_tube_full(B, O, synth):
    c = synth.config1()
    q, w, st = run_gpu(B, c)
    qo, wo, sto = run_oracle(O, c)
    assert st["n_failed"] == 0
    check_state("cfg1 128 cells x 128 steps", q, qo, 1e-9, c["params"])
    assert st["hist_stage"].sum() == 2 * 128 * 128 and st["hist_c2p"].sum() == 128 * 128
    assert st["hist_stage"][0] == 0


def test_config3_shear_layer_reduced(B, O, synth):
    c = synth.config3(nx=96, ny=128, nsteps=60)
    q, w, st = run_gpu(B, c)
    qo, wo, _ = run_oracle(O, c)
    assert st["n_failed"] == 0
    check_state("cfg3 96 x 128 x 60 steps", q, qo, 1e-8, c["params"])
    assert rel_l1(w[:5], wo[:5]) <= 1e-8


def test_config3_shear_layer_full_size(B, O, synth):
    """BASELINE.json configs[2] as stated: 512 x 512, 200 steps, whole grid against the oracle (about a minute of
    oracle time on 16 cores)."""
    c = synth.config3()
    assert c["prims"].shape[1:] == (1, 512, 512) and c["nsteps"] == 200
    q, w, st = run_gpu(B, c)
    qo, wo, _ = run_oracle(O, c)
    assert st["n_failed"] == 0
    check_state("cfg3 512 x 512 x 200 steps", q, qo, 1e-8, c["params"])
    assert rel_l1(w[:5], wo[:5]) <= 1e-8


def test_config5_blast_reduced(B, O, synth):
    c = synth.config5(n=40, nsteps=20)
    q, w, st = run_gpu(B, c)
    qo, wo, _ = run_oracle(O, c)
    assert st["n_failed"] == 0
    check_state("cfg5 40^3 x 20 steps", q, qo, 1e-8, c["params"])


def test_config5_full_size_full_length(B, O, synth):
    """BASELINE.json configs[4] as stated: 256^3, 20 steps, the WHOLE grid against the oracle, in the launch configuration
    bench.py times.  Cost: 256^3 x 20 = 3.4e8 oracle zone-updates, about 6 minutes at the 9e5 zone-updates/s the oracle
    reaches on the GPU box's 16 host threads, and about 25 GB of host memory (the oracle keeps 120 ghosted rows of
    264^3 doubles)."""
    n = 256
    c = synth.config5(n=n, nsteps=20)
    assert c["nsteps"] == 20
    t0 = time.time()
    q, w, st = run_gpu(B, c)
    del w
    qo, wo, sto = run_oracle(O, c)
    del wo
    assert st["n_failed"] == 0 and sto["n_failed"] == 0
    g, pv = check_state("cfg5 %d^3 x 20 steps (whole grid)" % n, q, qo, 1e-8, c["params"])
    assert st["hist_stage"].sum() == 2 * n ** 3 * 20
    print("cfg5 full: %.0f s, rel-L1 %.2e, per-variable max %.2e" % (time.time() - t0, g, pv.max()))


def test_config5_full_size_sampled_against_oracle(B, O, synth):
    """256^3, the launch configuration bench.py times.  Two steps; the oracle recomputes a
    sub-box (24^3 + 8 halo cells per side, enough for 2 steps x 2 stages x 2-cell stencil) that
    straddles the blast edge, from the same initial data; plus properties that hold at any size."""
    n = 256
    c = synth.config5(n=n, nsteps=2)
    sim = B.Rmhd(**c["params"])
    sim.set_initial(c["prims"])
    q0, _ = sim.get_state()
    sim.step(2)
    q, w = sim.get_state()
    st = sim.stats()
    sim.close()
    assert st["n_failed"] == 0
    lo, m, h = 136, 24, 8            # box [136,160)^3 ; blast edge at 128 + 25.6 cells
    sl = slice(lo - h, lo + m + h)
    sub = dict(c); P = dict(c["params"]); dx = 1.0 / n
    P.update(nx=m + 2 * h, ny=m + 2 * h, nz=m + 2 * h,
             xlim=(-0.5 + (lo - h) * dx, -0.5 + (lo + m + h) * dx),
             ylim=(-0.5 + (lo - h) * dx, -0.5 + (lo + m + h) * dx),
             zlim=(-0.5 + (lo - h) * dx, -0.5 + (lo + m + h) * dx))
    sub["params"] = P
    sub["prims"] = np.ascontiguousarray(c["prims"][:, sl, sl, sl])
    qo, wo, _ = run_oracle(O, sub, nsteps=2)
    inner = slice(h, h + m)
    a = q[:, lo:lo + m, lo:lo + m, lo:lo + m]; b = qo[:, inner, inner, inner]
    assert np.abs(b[1]).max() > 1e-4                     # the box does see the blast wave
    assert rel_l1(a, b) <= 1e-8, rel_l1(a, b)
    # properties at full size: source-free rows conserved (nothing reaches the boundary) ...
    for r in (0, 4, 5):
        assert abs(q[r].sum() - q0[r].sum()) <= 1e-12 * np.abs(q0[r]).sum()
    # ... and x-mirror symmetry (B_x even): S_x odd, D even
    assert np.abs(q[0] - q[0][:, :, ::-1]).max() < 1e-11
    assert np.abs(q[1] + q[1][:, :, ::-1]).max() < 1e-11


def test_config4_two_fluid_reduced(B, O, synth):
    c = synth.config4(nx=64, ny=48, nsteps=50)
    q, w, st = run_gpu(B, c)
    qo, wo, _ = run_oracle(O, c)
    assert st["n_failed"] == 0
    check_state("cfg4 64 x 48 x 50 steps", q, qo, 1e-8, c["params"])
    assert rel_l1(w[:10], wo[:10]) <= 1e-8
    assert st["hist_stage"].sum() == 2 * 64 * 48 * 50


def test_config4_full_size_full_length(B, O, synth):
    """BASELINE.json configs[3] as stated: two-fluid, 1024 x 1024, 50 steps, the WHOLE grid against the oracle
    (5.2e7 two-fluid oracle zone-updates: a few minutes on the GPU box's host threads)."""
    c = synth.config4()
    assert c["prims"].shape[1:] == (1, 1024, 1024) and c["nsteps"] == 50
    t0 = time.time()
    q, w, st = run_gpu(B, c)
    qo, wo, sto = run_oracle(O, c)
    assert st["n_failed"] == 0 and sto["n_failed"] == 0
    g, pv = check_state("cfg4 1024 x 1024 x 50 steps (whole grid)", q, qo, 1e-8, c["params"])
    assert rel_l1(w[:10], wo[:10]) <= 1e-8
    assert st["hist_stage"].sum() == 2 * 1024 * 1024 * 50
    print("cfg4 full: %.0f s, rel-L1 %.2e, per-variable max %.2e" % (time.time() - t0, g, pv.max()))


def test_config4_full_size_sampled_against_oracle(B, O, synth):
    """1024^2 two-fluid (BASELINE.json configs[3]), two steps; the oracle recomputes a 32^2 box with
    8 halo cells per side (2 steps x 2 stages x 2-cell stencil) from the same initial data."""
    c = synth.config4(nsteps=2)
    sim = B.Rmhd(**c["params"])
    sim.set_initial(c["prims"])
    q0, _ = sim.get_state()
    sim.step(2)
    q, w = sim.get_state()
    st = sim.stats()
    sim.close()
    assert st["n_failed"] == 0
    n, lo, m, h = 1024, 300, 32, 8
    sl = slice(lo - h, lo + m + h)
    sub = dict(c); P = dict(c["params"]); dx = 1.0 / n
    P.update(nx=m + 2 * h, ny=m + 2 * h, bc=(0, 0, 0), xlim=((lo - h) * dx, (lo + m + h) * dx), ylim=((lo - h) * dx, (lo + m + h) * dx))
    sub["params"] = P
    sub["prims"] = np.ascontiguousarray(c["prims"][:, :, sl, sl])
    qo, wo, _ = run_oracle(O, sub, nsteps=2)
    inner = slice(h, h + m)
    a = q[:, :, lo:lo + m, lo:lo + m]; b = qo[:, :, inner, inner]
    assert rel_l1(a, b) <= 1e-8, rel_l1(a, b)
    # periodic grid: the source-free rows D, S, tau, Dbar, B are conserved to round-off
    for r in (0, 1, 2, 4, 5, 10):
        assert abs(q[r].sum() - q0[r].sum()) <= 1e-11 * max(np.abs(q0[r]).sum(), 1.0), r


# ------------------------------------------------------------------------------------------
# API behaviour
# ------------------------------------------------------------------------------------------
def test_unphysical_input_is_reported(B, synth):
    c = synth.config1(nx=16)
    w = c["prims"].copy(); w[4, 0, 0, 3] = -1.0
    sim = B.Rmhd(**c["params"])
    with pytest.raises(B.RmhdError) as e:
        sim.set_initial(w)
    assert e.value.code == B.RMHD_ERR_UNPHYSICAL_INPUT
    sim.close()


def test_graph_replay_equals_plain_launches_bitwise(B, synth):
    """rmhd_step replays one captured step as a CUDA graph on grids of up to 2^21 cells; profiling mode uses plain launches.
    Same kernels, same arguments: the states must be bitwise equal (1-D, 2-D and 3-D, both integrators), and
    rmhd_get_kernel_times must count the same launches on both paths (a replayed step counts its kernels, the capture itself none)."""
    for c, kw in ((synth.config1(nx=100), {}), (synth.config3(nx=64, ny=40, nsteps=6), {}), (synth.config5(n=24, nsteps=6), {}),
                  (synth.config5(n=24, nsteps=6), {"integrator": "ssp3"}), (synth.config4(nx=40, ny=24, nsteps=6), {})):
        p = dict(c["params"]); p.update(kw)
        a = B.Rmhd(**p); a.set_initial(np.ascontiguousarray(c["prims"]), c.get("rho_charge"))
        B.rmhd_set_profiling(a.ctx, False)      # zeroes the counters; set_initial's launch is not a step's
        a.step(1); a.step(5)
        la = {k: v["launches"] for k, v in B.rmhd_get_kernel_times(a.ctx).items()}
        qa, wa = a.get_state(); sa = a.stats(); a.close()
        b = B.Rmhd(**p); b.set_initial(np.ascontiguousarray(c["prims"]), c.get("rho_charge"))
        B.rmhd_set_profiling(b.ctx, True)
        b.step(6)
        lb = {k: v["launches"] for k, v in B.rmhd_get_kernel_times(b.ctx).items()}
        qb, wb = b.get_state(); sb = b.stats(); b.close()
        assert la == lb and sum(la.values()) == 6 * (7 if kw else 5), (la, lb)
        assert np.array_equal(qa, qb) and np.array_equal(wa, wb)
        assert np.array_equal(sa["hist_stage"], sb["hist_stage"]) and np.array_equal(sa["hist_c2p"], sb["hist_c2p"])


def test_degenerate_calls(B, synth):
    """nsteps = 0 is a no-op; an empty batch is accepted; a grid of 2^31 cells is refused before anything is allocated; set_cons
    resets the statistics so that its return code is its own."""
    c = synth.config5(n=16, nsteps=1)
    sim = B.Rmhd(**c["params"]); sim.set_initial(c["prims"])
    q0, _ = sim.get_state()
    assert sim.step(0) == B.RMHD_OK and sim.time == 0.0
    q1, _ = sim.get_state()
    assert np.array_equal(q0, q1)
    sim.step(2)
    assert sim.stats()["hist_stage"].sum() == 2 * 2 * 16 ** 3
    assert sim.set_cons(q0) == 0
    st = sim.stats()
    assert st["hist_stage"].sum() == 0 and st["hist_c2p"].sum() == 16 ** 3 and st["n_failed"] == 0
    assert abs(sim.time - 2 * sim.dt) < 1e-18          # the step counter is untouched
    sim.close()
    P = B.make_params(model=0, gamma=G43, sigma=1.0)
    e = np.empty((14, 0)); w = np.empty((11, 0))
    B.rmhd_stage_batch(P, e, w, 1e-3, e.copy(), w.copy())
    B.rmhd_con2prim_batch(P, e, w.copy())
    with pytest.raises(B.RmhdError) as ex:
        B.Rmhd(model=0, nx=2048, ny=2048, nz=512, sigma=1.0)
    assert ex.value.code == B.RMHD_ERR_BAD_PARAM


def test_host_batches_reuse_one_staging_area(B, synth):
    """Host-buffer batch calls stage through one grow-only device allocation (rmhd_release_staging, rmhd.h): a small call, a larger
    one (the area grows), the small one again (stale contents of the larger call behind it), and once more after a release must all
    give what the device-buffer path gives, bit for bit."""
    import torch
    def run(n, host):
        c = synth.config2(n, seed=4)
        P = B.make_params(**c["params"])
        q_ex = np.empty((14, n)); B.rmhd_prim2cons_batch(P, c["prims"], q_ex)
        if host:
            q = np.empty_like(q_ex); w = np.empty_like(c["prims"]); it = np.zeros(n, np.int32); fl = np.zeros(n, np.int32)
            B.rmhd_stage_batch(P, q_ex, c["prims"], c["a_dt"], q, w, c["sigma_cell"], it, fl)
            w2 = np.empty_like(w); B.rmhd_con2prim_batch(P, q, w2, w)
            return q, w, it, fl, w2
        d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
        q = torch.empty(14, n, dtype=torch.float64, device="cuda"); w = torch.empty(11, n, dtype=torch.float64, device="cuda")
        it = torch.zeros(n, dtype=torch.int32, device="cuda"); fl = torch.zeros(n, dtype=torch.int32, device="cuda")
        B.rmhd_stage_batch(P, d(q_ex), d(c["prims"]), c["a_dt"], q, w, d(c["sigma_cell"]), it, fl)
        w2 = torch.empty_like(w); B.rmhd_con2prim_batch(P, q, w2, w)
        torch.cuda.synchronize()
        return tuple(x.cpu().numpy() for x in (q, w, it, fl, w2))
    ref = {n: run(n, host=False) for n in (1000, 70001)}
    for n in (1000, 70001, 1000):
        for a, b in zip(run(n, host=True), ref[n]):
            assert np.array_equal(a, b, equal_nan=True)
    B.rmhd_release_staging(0)
    B.rmhd_release_staging(-1)          # nothing left: still fine
    for a, b in zip(run(1000, host=True), ref[1000]):
        assert np.array_equal(a, b, equal_nan=True)


def test_set_cons_get_state_round_trip_and_device_buffers(B, O, synth):
    import torch
    c = synth.config3(nx=32, ny=24, nsteps=3)
    sim = B.Rmhd(**c["params"]); sim.set_initial(c["prims"]); sim.step(3)
    q, w = sim.get_state()
    qd, wd = sim.get_state(device=True)
    assert np.array_equal(qd.cpu().numpy(), q) and np.array_equal(wd.cpu().numpy(), w)
    # restart from the checkpoint on a new context: same continuation
    sim.step(2); q5, _ = sim.get_state(); sim.close()
    sim2 = B.Rmhd(**c["params"]); assert sim2.set_cons(q, w) == 0; sim2.step(2); q5b, _ = sim2.get_state(); sim2.close()
    assert rel_l1(q5b, q5) < 1e-13
    assert abs(B.Rmhd(**c["params"]).dt - 0.4 / (32 / 1.0 + 24 / 2.0)) < 1e-16


# ------------------------------------------------------------------------------------------
# SSP3(332) (Table 3): same kernels, three stages
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("case", ["tube_1d", "shear_2d", "blast_3d", "two_fluid_2d", "blast_3d_split"])
def test_ssp3_332_parity(B, O, synth, case, monkeypatch):
    if case == "tube_1d":                 # per-axis flux kernels + k_final_A
        c = synth.config1(); nsteps, tol = 128, 1e-9
    elif case == "shear_2d":              # fused two-role flux kernel, 2-D, partial tiles
        c = synth.config3(nx=80, ny=72, nsteps=40); nsteps, tol = 40, 1e-8
    elif case in ("blast_3d", "blast_3d_split"):
        c = synth.config5(n=40, nsteps=12); nsteps, tol = 12, 1e-8
        if case == "blast_3d_split":
            monkeypatch.setenv("RMHD_FLUX", "split")
    else:
        c = synth.config4(nx=48, ny=40, nsteps=30); nsteps, tol = 30, 1e-8
    q, w, st = run_gpu(B, c, nsteps=nsteps, params_override={"integrator": "ssp3"})
    qo, wo, _ = run_oracle(O, c, nsteps=nsteps, params_override={"integrator": "ssp3"})
    assert st["n_failed"] == 0
    check_state("ssp3 " + case, q, qo, tol, c["params"])
    ncell = int(np.prod(c["prims"].shape[1:]))
    assert st["hist_stage"].sum() == 3 * ncell * nsteps and st["hist_c2p"].sum() == ncell * nsteps
    # and it is a different scheme from SSP2(222)
    q2, _, _ = run_gpu(B, c, nsteps=nsteps)
    assert rel_l1(q2, qo) > 1e-7


def test_bad_integrator_is_rejected(B):
    with pytest.raises(B.RmhdError):
        B.Rmhd(model=0, nx=8, integrator=7)


# ------------------------------------------------------------------------------------------
# the paper's own set-ups (section 4), both integrators
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("integrator", ["ssp2", "ssp3"])
@pytest.mark.parametrize("case", ["brio_wu_single_fig1", "brio_wu_pair", "brio_wu_electron_proton", "khi_resistive", "khi_two_fluid"])
def test_paper_setups_parity(B, O, synth, case, integrator):
    if case == "brio_wu_single_fig1":        # Fig 1: nx = 200, T = 0.4, sigma = 1e3
        c = synth.brio_wu_single(nx=200, sigma=1e3, integrator=integrator); tol = 1e-9
    elif case == "brio_wu_pair":             # Fig 2 left: mu_p = -mu_e = 1e3
        c = synth.brio_wu_two_fluid(nx=200, mu_p=1e3, mu_e=-1e3, integrator=integrator); tol = 1e-8
    elif case == "brio_wu_electron_proton":  # Fig 2 right: mu_p = 1e3, mu_e = -1e5
        c = synth.brio_wu_two_fluid(nx=160, mu_p=1e3, mu_e=-1e5, integrator=integrator); tol = 1e-8
    elif case == "khi_resistive":            # eq (18)-(20), reduced grid, 120 steps
        c = synth.khi_paper(model=0, nx=64, ny=128, nsteps=120, integrator=integrator); tol = 1e-8
    else:
        c = synth.khi_paper(model=1, nx=48, ny=96, nsteps=60, integrator=integrator); tol = 1e-8
    q, w, st = run_gpu(B, c)
    qo, wo, sto = run_oracle(O, c)
    assert st["n_failed"] == 0 and sto["n_failed"] == 0
    check_state("paper %s %s" % (case, integrator), q, qo, tol, c["params"])
    nh = 5 if c["params"]["model"] == 0 else 10
    assert rel_l1(w[:nh], wo[:nh]) <= 10 * tol


@pytest.mark.parametrize("integrator,flux", [("ssp2", None), ("ssp3", None), ("ssp2", "split")])
def test_two_fluid_3d_blast_parity(B, O, synth, integrator, flux, monkeypatch):
    """Full steps of the 18-variable model in 3-D (two-role flux kernel, per-axis kernels)."""
    if flux:
        monkeypatch.setenv("RMHD_FLUX", flux)
    c = synth.two_fluid_blast(n=36, nsteps=8, integrator=integrator)
    q, w, st = run_gpu(B, c)
    qo, wo, sto = run_oracle(O, c)
    assert st["n_failed"] == 0 and sto["n_failed"] == 0
    check_state("two-fluid 3-D blast %s %s" % (integrator, flux), q, qo, 1e-8, c["params"])
    assert rel_l1(w[:10], wo[:10]) <= 1e-8


def test_nonconvergence_is_reported_not_hidden(B, synth):
    """max_iter_stage = 1 on a stiff tube (sigma dt = 9): the Newton loops cannot finish.  rmhd_step still advances the
    requested steps, returns RMHD_ERR_NONCONVERGED, and get_stats names the count and the first failing cell
    (include/rmhd.h error contract; SURVEY.md section 5 'failure detection')."""
    c = synth.config1()
    kw = dict(c["params"]); kw["max_iter_stage"] = 1
    sim = B.Rmhd(**kw); sim.set_initial(np.ascontiguousarray(c["prims"]))
    rc = sim.step(3, check=False)
    assert rc == B.RMHD_ERR_NONCONVERGED
    assert abs(sim.time - 3 * sim.dt) < 1e-15
    st = sim.stats()
    assert st["n_failed"] > 0 and 0 <= st["first_failed_cell"] < 128
    # every solve stopped after its single iteration (or, in a cell an earlier failure made inadmissible, before it)
    assert st["hist_stage"][:2].sum() == st["hist_stage"].sum() == 2 * 3 * 128 and st["hist_stage"][1] > 700
    with pytest.raises(B.RmhdError) as e:
        sim.step(1)
    assert e.value.code == B.RMHD_ERR_NONCONVERGED
    sim.close()
    # the same run with the default cap converges everywhere
    sim = B.Rmhd(**c["params"]); sim.set_initial(np.ascontiguousarray(c["prims"])); sim.step(3)
    assert sim.stats()["n_failed"] == 0
    sim.close()


def test_stage_batch_flags_inadmissible_cells_like_the_oracle(B, O, synth):
    """config 2 recipe with E perturbations 10x larger (std 0.1): some low-pressure, strong-field cells have no
    admissible root.  Both sides must flag (almost) the same cells and agree on all the others."""
    n = 2 ** 15
    c = synth.config2(n, seed=0)
    w = c["prims"].copy()
    rng = np.random.default_rng(123)
    w[8:11] += 0.1 * rng.standard_normal((3, n))
    P = B.make_params(**c["params"]); PO = O.make_params(**c["params"])
    q_ex = O.prim2cons(PO, w)
    qo, wo, ito, flo = O.stage_batch(PO, q_ex, w, c["a_dt"], c["sigma_cell"])
    q = np.empty_like(q_ex); wg = np.empty_like(w); it = np.zeros(n, np.int32); fl = np.zeros(n, np.int32)
    B.rmhd_stage_batch(P, q_ex, w, c["a_dt"], q, wg, c["sigma_cell"], it, fl)
    bad, bado = fl != 0, flo != 0
    assert (bad != bado).sum() <= max(2, 0.02 * max(bad.sum(), bado.sum()))      # the same cells, up to marginal ones
    ok = ~bad & ~bado
    assert ok.mean() > 0.9
    assert rel_l1(q[:, ok], qo[:, ok]) <= 1e-10
