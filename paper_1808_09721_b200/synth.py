"""Seeded synthetic inputs for the five BASELINE.json configs.

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of the
method's arithmetic: it only writes down initial *primitive* fields (rho, v, p, B, E) and
the run parameters.  prim->cons, Gauss's law, con2prim etc. are done by whichever side
consumes the arrays.  The paper measures on its own initial data (Brio-Wu, KHI; PAPER.md
L260-354), not on a public suite; these configs are synthetic stand-ins with those shapes.

Arrays: float64, variable-major SoA, interior cells only, ``prims[var, k, j, i]`` (x fastest).
Resistive prims (11): rho, vx, vy, vz, p, Bx, By, Bz, Ex, Ey, Ez.
Two-fluid prims (16): rho_e, v_e(3), p_e, rho_p, v_p(3), p_p, B(3), E(3).
"""
import numpy as np

RESISTIVE, TWO_FLUID = 0, 1
BC_OUTFLOW, BC_PERIODIC = 0, 1

SSP2_GAMMA = 1.0 - 1.0 / np.sqrt(2.0)


def cell_centres(n, lo, hi):
    dx = (hi - lo) / n
    return lo + (np.arange(n) + 0.5) * dx


def _minus_v_cross_B(v, B):
    """E = -v x B (ideal-MHD initial electric field; initial data, not the scheme)."""
    return -np.stack([v[1] * B[2] - v[2] * B[1], v[2] * B[0] - v[0] * B[2], v[0] * B[1] - v[1] * B[0]])


def config1(nx=128):
    """1D resistive Riemann tube (BASELINE.json configs[0]); 128 steps at nx=128 reach t=0.4."""
    x = cell_centres(nx, -0.5, 0.5)
    left = x < 0.0
    w = np.zeros((11, 1, 1, nx))
    w[0, 0, 0] = np.where(left, 1.0, 0.125)
    w[4, 0, 0] = np.where(left, 1.0, 0.1)
    w[5, 0, 0] = 0.5
    w[6, 0, 0] = np.where(left, 1.0, -1.0)
    params = dict(model=RESISTIVE, nx=nx, ny=1, nz=1, ng=4, xlim=(-0.5, 0.5), ylim=(0.0, 1.0), zlim=(0.0, 1.0),
                  bc=(BC_OUTFLOW,) * 3, gamma=2.0, sigma=1e4, kappa=1.0, cfl=0.4)
    return dict(name="cfg1_tube", params=params, prims=w, rho_charge=None, nsteps=nx, tol=1e-9)


def config2(ncells=2 ** 20, seed=0):
    """Batched implicit-stage microbench (BASELINE.json configs[1]): independent resistive cells."""
    rng = np.random.default_rng(seed)
    rho = 10.0 ** rng.uniform(-1.0, 1.0, ncells)
    p = 10.0 ** rng.uniform(-2.0, 1.0, ncells)
    dirs = rng.standard_normal((3, ncells))
    dirs /= np.sqrt((dirs ** 2).sum(axis=0))
    v = dirs * (0.9 * rng.uniform(0.0, 1.0, ncells) ** (1.0 / 3.0))
    B = rng.standard_normal((3, ncells))
    E = _minus_v_cross_B(v, B) + 0.01 * rng.standard_normal((3, ncells))
    sigma = 10.0 ** rng.uniform(0.0, 6.0, ncells)
    w = np.concatenate([rho[None], v, p[None], B, E], axis=0)
    params = dict(model=RESISTIVE, nx=1, ny=1, nz=1, ng=4, gamma=4.0 / 3.0, sigma=1.0, kappa=1.0, cfl=0.4)
    return dict(name="cfg2_stage_batch", params=params, prims=np.ascontiguousarray(w), sigma_cell=sigma,
                a_dt=SSP2_GAMMA * 1e-3, tol=1e-10)


def config3(nx=512, ny=512, nsteps=200):
    """2D resistive shear layer (BASELINE.json configs[2]); periodic x / outflow y."""
    x = cell_centres(nx, -0.5, 0.5)[None, :]
    y = cell_centres(ny, -1.0, 1.0)[:, None]
    w = np.zeros((11, 1, ny, nx))
    w[0] = 1.0
    w[4] = 1.0
    vx = 0.5 * np.tanh(y / 0.01) + 0.0 * x
    vy = 0.1 * np.sin(2.0 * np.pi * x) * np.exp(-y ** 2 / 0.01)
    w[1, 0], w[2, 0] = vx, vy
    w[7] = 0.1
    w[8:11] = _minus_v_cross_B(w[1:4], w[5:8])
    params = dict(model=RESISTIVE, nx=nx, ny=ny, nz=1, ng=4, xlim=(-0.5, 0.5), ylim=(-1.0, 1.0), zlim=(0.0, 1.0),
                  bc=(BC_PERIODIC, BC_OUTFLOW, BC_OUTFLOW), gamma=4.0 / 3.0, sigma=1e3, kappa=1.0, cfl=0.4)
    return dict(name="cfg3_shear", params=params, prims=w, rho_charge=None, nsteps=nsteps, tol=1e-8)


def config4(nx=1024, ny=1024, nsteps=50, seed=0):
    """2D two-fluid pair plasma with seeded smooth velocity (BASELINE.json configs[3]); periodic."""
    rng = np.random.default_rng(seed)
    A = rng.uniform(-1.0, 1.0, (2, 4))
    th = rng.uniform(0.0, 2.0 * np.pi, (2, 4))
    kvec = [(1, 0), (0, 1), (1, 1), (1, -1)]
    x = cell_centres(nx, 0.0, 1.0)[None, :]
    y = cell_centres(ny, 0.0, 1.0)[:, None]
    v = np.zeros((3, 1, ny, nx))
    for c in range(2):
        for m, (kx, ky) in enumerate(kvec):
            v[c, 0] += A[c, m] * np.sin(2.0 * np.pi * (kx * x + ky * y) + th[c, m])
    v *= 0.4 / np.sqrt((v ** 2).sum(axis=0)).max()
    w = np.zeros((16, 1, ny, nx))
    for s in range(2):
        w[5 * s + 0] = 0.5
        w[5 * s + 1:5 * s + 4] = v
        w[5 * s + 4] = 0.5
    w[10] = 0.2
    w[13:16] = _minus_v_cross_B(v, w[10:13])
    params = dict(model=TWO_FLUID, nx=nx, ny=ny, nz=1, ng=4, xlim=(0.0, 1.0), ylim=(0.0, 1.0), zlim=(0.0, 1.0),
                  bc=(BC_PERIODIC,) * 3, gamma=4.0 / 3.0, eta=1e-4, mu_e=-100.0, mu_p=100.0, kappa=1.0, cfl=0.4)
    return dict(name="cfg4_two_fluid", params=params, prims=w, rho_charge=None, nsteps=nsteps, tol=1e-8)


def config5(n=256, nsteps=20):
    """3D resistive blast (BASELINE.json configs[4]); outflow."""
    c = cell_centres(n, -0.5, 0.5)
    r2 = c[:, None, None] ** 2 + c[None, :, None] ** 2 + c[None, None, :] ** 2
    w = np.zeros((11, n, n, n))
    w[0] = 1.0
    w[4] = np.where(r2 < 0.1 ** 2, 1.0, 0.01)
    w[5] = 0.1
    params = dict(model=RESISTIVE, nx=n, ny=n, nz=n, ng=4, xlim=(-0.5, 0.5), ylim=(-0.5, 0.5), zlim=(-0.5, 0.5),
                  bc=(BC_OUTFLOW,) * 3, gamma=4.0 / 3.0, sigma=1e5, kappa=1.0, cfl=0.3)
    return dict(name="cfg5_blast", params=params, prims=w, rho_charge=None, nsteps=nsteps, tol=1e-8)


# ---------------------------------------------------------------------------------------------------
# The paper's own set-ups: initial data as printed in PAPER.md section 4, used as
# second / third workloads.  What the paper leaves open is fixed here and listed in DESIGN.md section 12.
# ---------------------------------------------------------------------------------------------------
def brio_wu_single(nx=200, sigma=1e4, t_end=0.4, cfl=0.4, integrator="ssp2"):
    """Single-fluid resistive Brio-Wu tube, eq (13) PAPER.md L268 (set-up of Palenzuela et al. 2009): Gamma = 2,
    (rho, p, B_y) = (1, 1, 0.5) | (0.125, 0.1, -0.5) on x in [0, 1], v = 0, E = 0, B_x = B_z = 0 (not printed: G14).
    Fig 1 uses nx = 200, T = 0.4 (L287); the profile table nx = 2^17, sigma = 1e4 (L402)."""
    x = cell_centres(nx, 0.0, 1.0)
    left = x < 0.5
    w = np.zeros((11, 1, 1, nx))
    w[0, 0, 0] = np.where(left, 1.0, 0.125)
    w[4, 0, 0] = np.where(left, 1.0, 0.1)
    w[6, 0, 0] = np.where(left, 0.5, -0.5)
    params = dict(model=RESISTIVE, nx=nx, ny=1, nz=1, ng=4, xlim=(0.0, 1.0), ylim=(0.0, 1.0), zlim=(0.0, 1.0),
                  bc=(BC_OUTFLOW,) * 3, gamma=2.0, sigma=sigma, kappa=1.0, cfl=cfl, integrator=integrator)
    nsteps = int(round(t_end / (cfl / nx)))
    return dict(name="brio_wu_single", params=params, prims=w, rho_charge=None, nsteps=nsteps, tol=1e-9)


def brio_wu_two_fluid(nx=400, mu_p=1e3, mu_e=-1e3, eta=1e-3, t_end=0.4, cfl=0.4, integrator="ssp2"):
    """Two-fluid Brio-Wu tube, eq (14) PAPER.md L275 (initial data of Amano 2016):
    (rho, p, B_x, B_y) = (1, 1, 0.5, 1) | (0.125, 0.1, 0.5, -1) on x in [0, 1], both species at rest, E = 0.
    Fig 2 (L291): pair plasma mu_p = -mu_e = 1e3, and mu_p = 1e3, mu_e = -1e5, up to 1600 cells, T = 0.4.
    Species split (not printed): charge neutral (sum_s mu_s rho_s = 0) and equal number density and temperature,
    so rho_s = rho |mu_other| / (|mu_e| + |mu_p|) and p_e = p_p = p/2.  Gamma = 2 as in the single-fluid tube;
    eta = 1e-3 (the paper gives none for this test)."""
    x = cell_centres(nx, 0.0, 1.0)
    left = x < 0.5
    rho = np.where(left, 1.0, 0.125)
    pr = np.where(left, 1.0, 0.1)
    ae, ap = abs(mu_e), abs(mu_p)
    w = np.zeros((16, 1, 1, nx))
    w[0, 0, 0] = rho * ap / (ae + ap)
    w[5, 0, 0] = rho * ae / (ae + ap)
    w[4, 0, 0] = 0.5 * pr
    w[9, 0, 0] = 0.5 * pr
    w[10, 0, 0] = 0.5
    w[11, 0, 0] = np.where(left, 1.0, -1.0)
    params = dict(model=TWO_FLUID, nx=nx, ny=1, nz=1, ng=4, xlim=(0.0, 1.0), ylim=(0.0, 1.0), zlim=(0.0, 1.0),
                  bc=(BC_OUTFLOW,) * 3, gamma=2.0, eta=eta, mu_e=mu_e, mu_p=mu_p, kappa=1.0, cfl=cfl, integrator=integrator)
    nsteps = int(round(t_end / (cfl / nx)))
    return dict(name="brio_wu_two_fluid", params=params, prims=w, rho_charge=None, nsteps=nsteps, tol=1e-8)


def khi_paper(model=RESISTIVE, nx=512, ny=1024, nsteps=None, cfl=0.4, integrator="ssp2"):
    """Double-shear-layer Kelvin-Helmholtz set-up, eq (18)-(20) PAPER.md L336-352 (adapted from Mignone et al. 2009):
    x in [-0.5, 0.5], y in [-1, 1]; v_shear = 0.5, a = 0.01, (rho0, rho1) = (0.55, 0.45), A0 = 0.1, l = 0.1, p = 1,
    Gamma = 4/3, B_z = 0.1, sigma = 10, mu_p = -mu_e = 100; 512 x 1024 cells, T = 6 (L350-354).
    Not printed: boundary conditions (periodic in x and y here: the double layer is periodic in y), E (-v x B),
    the two-fluid species split (rho_s = rho/2, p_s = p/2, v_s = v) and its resistivity (eta = 1/sigma)."""
    vs, a, rho0, rho1, A0, ell = 0.5, 0.01, 0.55, 0.45, 0.1, 0.1
    x = cell_centres(nx, -0.5, 0.5)[None, :]
    y = cell_centres(ny, -1.0, 1.0)[:, None]
    up = y > 0.0
    ys = np.where(up, y - 0.5, y + 0.5)
    sgn = np.where(up, 1.0, -1.0)
    vx = sgn * vs * np.tanh(ys / a) + 0.0 * x
    vy = sgn * A0 * vs * np.sin(2.0 * np.pi * x) * np.exp(-ys ** 2 / ell ** 2)
    rho = rho0 + sgn * rho1 * np.tanh(ys / a) + 0.0 * x
    v = np.zeros((3, 1, ny, nx)); v[0, 0] = vx; v[1, 0] = vy
    B = np.zeros((3, 1, ny, nx)); B[2] = 0.1
    E = _minus_v_cross_B(v, B)
    common = dict(nx=nx, ny=ny, nz=1, ng=4, xlim=(-0.5, 0.5), ylim=(-1.0, 1.0), zlim=(0.0, 1.0),
                  bc=(BC_PERIODIC, BC_PERIODIC, BC_PERIODIC), gamma=4.0 / 3.0, kappa=1.0, cfl=cfl, integrator=integrator)
    if model == RESISTIVE:
        w = np.zeros((11, 1, ny, nx))
        w[0, 0] = rho; w[1:4] = v; w[4] = 1.0; w[5:8] = B; w[8:11] = E
        params = dict(model=RESISTIVE, sigma=10.0, **common)
    else:
        w = np.zeros((16, 1, ny, nx))
        for sp in range(2):
            w[5 * sp, 0] = 0.5 * rho; w[5 * sp + 1:5 * sp + 4] = v; w[5 * sp + 4] = 0.5
        w[10:13] = B; w[13:16] = E
        params = dict(model=TWO_FLUID, eta=0.1, mu_e=-100.0, mu_p=100.0, **common)
    dt = cfl / (nx / 1.0 + ny / 2.0)
    if nsteps is None:
        nsteps = int(round(6.0 / dt))
    return dict(name="khi_paper_" + ("resistive" if model == RESISTIVE else "two_fluid"), params=params, prims=w,
                rho_charge=None, nsteps=nsteps, tol=1e-8)


def two_fluid_blast(n=128, nsteps=10, integrator="ssp2"):
    """3-D two-fluid pair-plasma blast: the recipe of BASELINE.json configs[4] (3-D resistive blast) carried over to the
    18-variable model (not a BASELINE config; exercises the 3-D two-fluid kernels).  rho_e = rho_p = 0.5, total
    p = 1 inside r < 0.1 (cell-centre radius) and 0.01 outside split equally, both species at rest, B = (0.1, 0, 0), E = 0,
    mu_p = -mu_e = 100, eta = 1e-3, Gamma = 4/3, CFL 0.3, outflow."""
    c = cell_centres(n, -0.5, 0.5)
    r2 = c[:, None, None] ** 2 + c[None, :, None] ** 2 + c[None, None, :] ** 2
    w = np.zeros((16, n, n, n))
    for sp in range(2):
        w[5 * sp] = 0.5
        w[5 * sp + 4] = 0.5 * np.where(r2 < 0.1 ** 2, 1.0, 0.01)
    w[10] = 0.1
    params = dict(model=TWO_FLUID, nx=n, ny=n, nz=n, ng=4, xlim=(-0.5, 0.5), ylim=(-0.5, 0.5), zlim=(-0.5, 0.5),
                  bc=(BC_OUTFLOW,) * 3, gamma=4.0 / 3.0, eta=1e-3, mu_e=-100.0, mu_p=100.0, kappa=1.0, cfl=0.3,
                  integrator=integrator)
    return dict(name="two_fluid_blast", params=params, prims=w, rho_charge=None, nsteps=nsteps, tol=1e-8)


def random_resistive_prims(n, seed, vmax=0.99, with_E=True):
    """Random admissible resistive primitive states (round-trip pins, kernel unit tests)."""
    rng = np.random.default_rng(seed)
    rho = 10.0 ** rng.uniform(-2.0, 2.0, n)
    p = 10.0 ** rng.uniform(-3.0, 2.0, n)
    dirs = rng.standard_normal((3, n))
    dirs /= np.sqrt((dirs ** 2).sum(axis=0))
    v = dirs * (vmax * rng.uniform(0.0, 1.0, n))
    B = rng.standard_normal((3, n))
    E = rng.standard_normal((3, n)) if with_E else np.zeros((3, n))
    return np.ascontiguousarray(np.concatenate([rho[None], v, p[None], B, E], axis=0))


def random_two_fluid_prims(n, seed, vmax=0.9):
    rng = np.random.default_rng(seed)
    parts = []
    for _ in range(2):
        rho = 10.0 ** rng.uniform(-1.0, 1.0, n)
        p = 10.0 ** rng.uniform(-2.0, 1.0, n)
        dirs = rng.standard_normal((3, n))
        dirs /= np.sqrt((dirs ** 2).sum(axis=0))
        v = dirs * (vmax * rng.uniform(0.0, 1.0, n))
        parts += [rho[None], v, p[None]]
    B = rng.standard_normal((3, n))
    E = rng.standard_normal((3, n))
    return np.ascontiguousarray(np.concatenate(parts + [B, E], axis=0))


def stress_resistive_prims(n, seed, w_max=100.0, noise=1e-3):
    """Hard tail for con2prim: Lorentz factors log-uniform up to `w_max`, p/rho log-uniform
    in [1e-8, 1e4], B^2/rho log-uniform in [1e-4, 1e4], E = -v x B (1 + noise N(0,1)) component-wise, rho log-uniform in
    [1e-3, 1e3].  Initial data only: no method arithmetic."""
    rng = np.random.default_rng(seed)
    rho = 10.0 ** rng.uniform(-3.0, 3.0, n)
    p = rho * 10.0 ** rng.uniform(-8.0, 4.0, n)
    W = 10.0 ** rng.uniform(0.0, np.log10(w_max), n)
    dirs = rng.standard_normal((3, n))
    dirs /= np.sqrt((dirs ** 2).sum(axis=0))
    v = dirs * np.sqrt(1.0 - 1.0 / W ** 2)
    bdir = rng.standard_normal((3, n))
    bdir /= np.sqrt((bdir ** 2).sum(axis=0))
    B = bdir * np.sqrt(rho * 10.0 ** rng.uniform(-4.0, 4.0, n))
    E = _minus_v_cross_B(v, B) * (1.0 + noise * rng.standard_normal((3, n)))
    return np.ascontiguousarray(np.concatenate([rho[None], v, p[None], B, E], axis=0))
