"""Writes tests/golden/oracle_small_case.txt: the state after 2 RK2 steps of a tiny viscous run, computed by
oracle/ ONLY (never by the CUDA path).  Regression pin: an accidental change of the oracle's arithmetic shows up
as a diff of this file; the CUDA path is compared with the same stored values in tests/test_golden.py.

    python tests/golden/make_golden.py

Case: 7 x 6 x 5 cells, dx = dy = 0.3 fm, deta = 0.3, tau0 = 0.6, dtau = 0.03, eta/s = 0.12, crossover EoS table,
Milne geometry, outflow boundaries in x and eta, periodic in y, defaults otherwise (theta 1.1, xi 1, v_max 0.999);
initial state from inputs.ic_random_smooth(7, 6, 5, seed=42, vmax=0.35) with its raw pi components."""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

from oracle import Oracle  # noqa: E402
from paper_1802_04449_b200 import inputs  # noqa: E402

CASE = dict(nx=7, ny=6, nz=5, dx=0.3, dy=0.3, deta=0.3, dtau=0.03, tau0=0.6, eta_over_s=0.12, bc=(0, 1, 0), steps=2)


def initial_T_pi(eos):
    e, v, pi = inputs.ic_random_smooth(CASE["nx"], CASE["ny"], CASE["nz"], seed=42, vmax=0.35)
    o = Oracle(1, 1, 1, 1, 1, 1, 0.1, 1.0, eos, 0.0)
    P = np.vectorize(lambda x: o.eos(x)[0])(e)
    g2 = 1.0 / (1.0 - (v ** 2).sum(0))
    T = np.stack([(e + P) * g2 - P, (e + P) * g2 * v[0], (e + P) * g2 * v[1], (e + P) * g2 * v[2]]) + pi[:4]
    return T, pi


def run():
    eos = inputs.crossover_table()
    T, pi = initial_T_pi(eos)
    o = Oracle(CASE["nx"], CASE["ny"], CASE["nz"], CASE["dx"], CASE["dy"], CASE["deta"], CASE["dtau"], CASE["tau0"],
               eos, CASE["eta_over_s"], bc=CASE["bc"])
    o.load(T, pi)
    o.step(CASE["steps"])
    e, u, p = o.read()
    return np.concatenate([e[None], u, p]).reshape(15, -1)


if __name__ == "__main__":
    out = run()
    path = os.path.join(HERE, "oracle_small_case.txt")
    with open(path, "w") as f:
        f.write("# written by tests/golden/make_golden.py from oracle/ only; rows: e, u^tau, u^x, u^y, u^eta, pi[0..9]; "
                "columns: cells [k][j][i] of the 7x6x5 case described in that script\n")
        np.savetxt(f, out, fmt="%.17e")
    print("wrote", path, out.shape)
