"""Stored oracle output (tests/golden/oracle_small_case.txt, written by tests/golden/make_golden.py from oracle/
only): the oracle must still reproduce it (CPU), and the CUDA path must match it (GPU)."""
import os
import sys

import numpy as np
import pytest

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.join(HERE, "golden"))
import make_golden  # noqa: E402

GOLD = np.loadtxt(os.path.join(HERE, "golden", "oracle_small_case.txt"))


def test_oracle_reproduces_golden():
    out = make_golden.run()
    assert out.shape == GOLD.shape == (15, 210)
    assert np.max(np.abs(out - GOLD) / (np.abs(GOLD) + 1e-30)) < 1e-12


@pytest.mark.gpu
@pytest.mark.parametrize("kernel", [1, 2, 3])
def test_cuda_matches_golden(crossover, kernel):
    from paper_1802_04449_b200 import Hydro
    c = make_golden.CASE
    T, pi = make_golden.initial_T_pi(crossover)
    g = Hydro(c["nx"], c["ny"], c["nz"], c["dx"], c["dy"], c["deta"], c["dtau"], c["tau0"], crossover,
              c["eta_over_s"], bc=c["bc"], kernel=kernel)
    g.load(np.ascontiguousarray(T), np.ascontiguousarray(pi))
    g.step(c["steps"])
    e, u, p = g.read()
    out = np.concatenate([e[None], u, p]).reshape(15, -1)
    scale = np.abs(GOLD).max(axis=1, keepdims=True)
    assert np.max(np.abs(out - GOLD) / scale) < 1e-12
