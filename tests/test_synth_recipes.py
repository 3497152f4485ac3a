"""The seeded input recipes of BASELINE.json's five configs and of the paper's own
set-ups: shapes, parameters, time steps (reading G9), reproducibility.  synth.py holds no method arithmetic, so these are
checks of the recipe itself, not of the scheme."""
import numpy as np


def _dt(O, c, small=8):
    """dt of the config as the oracle computes it (G9), on a grid cut down to `small` cells per present axis with the
    same cell sizes (the time step depends on dx only; a 256^3 oracle context would need 17 GB)."""
    p = dict(c["params"])
    for n, lim in (("nx", "xlim"), ("ny", "ylim"), ("nz", "zlim")):
        if p[n] > small:
            dx = (p[lim][1] - p[lim][0]) / p[n]
            p[lim] = (p[lim][0], p[lim][0] + small * dx)
            p[n] = small
    S = O.OracleSim(O.make_params(**p))
    dt = S.dt
    S.close()
    return dt


def test_config1_tube(O, synth):
    c = synth.config1()
    w = c["prims"]
    assert w.shape == (11, 1, 1, 128) and c["nsteps"] == 128 and c["params"]["gamma"] == 2.0 and c["params"]["sigma"] == 1e4
    assert np.all(w[0, 0, 0, :64] == 1.0) and np.all(w[0, 0, 0, 64:] == 0.125)          # interface on the face 63|64
    assert np.all(w[4, 0, 0, :64] == 1.0) and np.all(w[4, 0, 0, 64:] == 0.1)
    assert np.all(w[5] == 0.5) and np.all(w[6, 0, 0, :64] == 1.0) and np.all(w[6, 0, 0, 64:] == -1.0)
    assert not w[1:4].any() and not w[8:11].any()
    dt = _dt(O, c)
    assert abs(dt - 0.003125) < 1e-18 and abs(128 * dt - 0.4) < 1e-15


def test_config2_batch_is_seeded_and_in_range(synth):
    a, b = synth.config2(4096, seed=0), synth.config2(4096, seed=0)
    assert np.array_equal(a["prims"], b["prims"]) and np.array_equal(a["sigma_cell"], b["sigma_cell"])
    assert not np.array_equal(a["prims"], synth.config2(4096, seed=1)["prims"])
    w, sig = a["prims"], a["sigma_cell"]
    assert w.shape == (11, 4096)
    assert 0.1 <= w[0].min() and w[0].max() <= 10 and 0.01 <= w[4].min() and w[4].max() <= 10
    assert np.sqrt((w[1:4] ** 2).sum(0)).max() < 0.9 and 1.0 <= sig.min() and sig.max() <= 1e6
    dE = w[8:11] + np.cross(w[1:4].T, w[5:8].T).T                 # E + v x B: the N(0, 0.01) perturbation (G17: std)
    assert 0.008 < dE.std() < 0.012 and abs(dE.mean()) < 1e-3
    assert abs(a["a_dt"] - (1 - 1 / np.sqrt(2)) * 1e-3) < 1e-18 and a["params"]["gamma"] == 4.0 / 3.0
    assert synth.config2()["prims"].shape == (11, 2 ** 20)


def test_config3_shear_layer(O, synth):
    c = synth.config3()
    w = c["prims"]
    assert w.shape == (11, 1, 512, 512) and c["nsteps"] == 200 and c["params"]["sigma"] == 1e3
    assert c["params"]["bc"][0] == synth.BC_PERIODIC and c["params"]["bc"][1] == synth.BC_OUTFLOW
    y = synth.cell_centres(512, -1.0, 1.0)[:, None]; x = synth.cell_centres(512, -0.5, 0.5)[None, :]
    assert np.allclose(w[1, 0], 0.5 * np.tanh(y / 0.01) + 0 * x) and np.allclose(w[2, 0], 0.1 * np.sin(2 * np.pi * x) * np.exp(-y ** 2 / 0.01))
    assert np.all(w[7] == 0.1) and np.allclose(w[8], -0.1 * w[2]) and np.allclose(w[9], 0.1 * w[1]) and not w[10].any()
    assert c["rho_charge"] is None                                  # Gauss's law by the consumer (G10)
    assert abs(_dt(O, c) - 0.4 / 768) < 1e-18


def test_config4_two_fluid(O, synth):
    c = synth.config4(nx=64, ny=64)
    w = c["prims"]
    assert w.shape == (16, 1, 64, 64) and np.all(w[0] == 0.5) and np.all(w[5] == 0.5) and np.all(w[4] == 0.5) and np.all(w[9] == 0.5)
    assert np.array_equal(w[1:4], w[6:9]) and not w[3].any()
    assert abs(np.sqrt((w[1:4] ** 2).sum(0)).max() - 0.4) < 1e-12
    assert np.all(w[10] == 0.2) and np.allclose(w[15], 0.2 * w[2]) and not w[13].any() and not w[14].any()
    p = c["params"]
    assert (p["mu_e"], p["mu_p"], p["eta"]) == (-100.0, 100.0, 1e-4) and all(b == synth.BC_PERIODIC for b in p["bc"])
    full = synth.config4()
    assert full["prims"].shape == (16, 1, 1024, 1024) and full["nsteps"] == 50 and abs(_dt(O, dict(full, prims=None)) - 0.4 / 2048) < 1e-18


def test_config5_blast(O, synth):
    c = synth.config5(n=64)
    w = c["prims"]
    x = synth.cell_centres(64, -0.5, 0.5)
    r2 = x[:, None, None] ** 2 + x[None, :, None] ** 2 + x[None, None, :] ** 2
    assert np.array_equal(w[4] == 1.0, r2 < 0.01) and set(np.unique(w[4])) == {0.01, 1.0}
    assert np.all(w[0] == 1.0) and np.all(w[5] == 0.1) and not w[1:4].any() and not w[6:11].any()
    p = synth.config5()["params"]
    assert (p["nx"], p["ny"], p["nz"], p["sigma"], p["cfl"]) == (256, 256, 256, 1e5, 0.3)
    assert abs(_dt(O, dict(params=p)) - 0.1 / 256) < 1e-18


def test_paper_setups(synth):
    bw = synth.brio_wu_single(nx=200)
    assert bw["nsteps"] == 200 and bw["params"]["gamma"] == 2.0 and np.all(np.abs(bw["prims"][6]) == 0.5)
    tf = synth.brio_wu_two_fluid(nx=100, mu_p=1e3, mu_e=-1e5)
    w = tf["prims"]
    assert np.allclose(w[0] + w[5], np.where(np.arange(100) < 50, 1.0, 0.125))           # total density of eq (14)
    assert np.allclose(-1e5 * w[0] + 1e3 * w[5], 0.0, atol=1e-12)                         # charge neutral
    k = synth.khi_paper(model=0, nx=32, ny=64, nsteps=1)["prims"]
    assert abs(k[1].max() - 0.5) < 1e-6 and abs(k[0].max() - 1.0) < 1e-6 and abs(k[0].min() - 0.1) < 1e-6
    assert np.allclose(k[1, 0, 0], k[1, 0, -1], atol=1e-12)                               # periodic in y
