"""How much of the GPU-vs-oracle difference is FMA contraction?  (TEST INFRASTRUCTURE; an experiment, not a test.)

The GPU path contracts a*b+c into FMAs, the oracle is built with -ffp-contract=off (the paper switches FMA off).
tests/test_gpu_parity.py bounds the per-variable rel-L1 of the two-fluid model by 1e-13 mu^2 (capped at the case's global bound)
on the argument that this round-off is fed back through the source with omega_p^2 ~ mu^2 (A2).  This script
checks the argument on the CPU alone: it builds the oracle a second time with -ffp-contract=fast -mfma and runs the same seeded
cases on both builds.  If oracle(FMA) - oracle(no FMA) is of the size of GPU - oracle(no FMA), the bound is explained by
contraction; if it were orders smaller, the GPU path would carry a defect of its own.

    python -m oracle.fma_noise            # prints one table row per case; results quoted in DESIGN.md section 6

Calls only oracle/ and the seeded input generators (paper_1808_09721_b200/synth.py, which holds none of the method's arithmetic).
"""
import os
import subprocess
import sys
import tempfile

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)


def rel_l1_per_var(a, b, mu=None):
    """The measure of tests/test_gpu_parity.py::rel_l1_per_var, restated."""
    n = b[0].size
    out = []
    for v in range(b.shape[0]):
        den = max(np.abs(b[v]).sum(), n * 1e-8)
        if mu is not None and 5 <= v <= 9:
            den = max(den, mu * np.abs(b[v - 5]).sum())
        if mu is not None and v >= 16:
            den = max(den, 1e-6 * np.abs(b[13:16] if v == 16 else b[10:13]).sum() / 3.0)
        out.append(np.abs(a[v] - b[v]).sum() / den)
    return np.array(out)


def cases(synth):
    return {
        "cfg3 96 x 128 x 60 (resistive, control)": synth.config3(nx=96, ny=128, nsteps=60),
        "cfg4 128 x 128 x 50 (two-fluid, mu = 100)": synth.config4(nx=128, ny=128, nsteps=50),
        "cfg4 64 x 48 x 50 (two-fluid, mu = 100; GPU test case)": synth.config4(nx=64, ny=48, nsteps=50),
        "Brio-Wu pair plasma nx = 200 (mu = 1e3; GPU test case)": synth.brio_wu_two_fluid(nx=200, mu_p=1e3, mu_e=-1e3),
    }


def child(which, outdir):
    sys.path.insert(0, ROOT)
    from oracle import build as obuild
    if which == "fma":
        lib = os.path.join(HERE, "liboracle_fma.so")
        subprocess.check_call(["g++", "-std=c++17", "-O2", "-ffp-contract=fast", "-mfma", "-fopenmp", "-shared", "-fPIC",
                               "-Wno-unused-parameter", "-o", lib, obuild.SRC])
        obuild.LIB = lib
        obuild.build = lambda force=False: lib
    from oracle import oracle as O
    from paper_1808_09721_b200 import synth
    for i, (name, c) in enumerate(cases(synth).items()):
        S = O.OracleSim(O.make_params(**c["params"]))
        S.set_initial(c["prims"], c.get("rho_charge"))
        assert S.step(c["nsteps"]) == 0
        q, _ = S.get_state()
        S.close()
        np.save(os.path.join(outdir, "%s_%d.npy" % (which, i)), q)


def main():
    if len(sys.argv) == 4 and sys.argv[1] == "--child":
        return child(sys.argv[2], sys.argv[3])
    sys.path.insert(0, ROOT)
    from paper_1808_09721_b200 import synth
    with tempfile.TemporaryDirectory() as d:
        for which in ("plain", "fma"):
            subprocess.check_call([sys.executable, os.path.abspath(__file__), "--child", which, d])
        print("| case | global rel-L1, oracle(FMA) vs oracle | largest per-variable rel-L1 (row) | 1e-13 mu^2 |")
        print("|---|---|---|---|")
        for i, (name, c) in enumerate(cases(synth).items()):
            a = np.load(os.path.join(d, "fma_%d.npy" % i)); b = np.load(os.path.join(d, "plain_%d.npy" % i))
            two = b.shape[0] == 18
            mu = max(abs(c["params"]["mu_e"]), abs(c["params"]["mu_p"])) if two else None
            pv = rel_l1_per_var(a, b, mu)
            g = np.abs(a - b).sum() / np.abs(b).sum()
            print("| %s | %.1e | %.1e (%d) | %s |" % (name, g, pv.max(), int(pv.argmax()), "%.0e" % (1e-13 * mu ** 2) if two else "-"))
            print("|   per row: " + " ".join("%.0e" % x for x in pv) + " | | | |")


if __name__ == "__main__":
    main()
