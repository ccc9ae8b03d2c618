"""Oracle pins 1-2: Bjorken flow, PAPER.md:382-392 (Eq.68, Eq.69)."""
import numpy as np
import pytest

from oracle import Oracle
from analytic_refs import bjorken_is, bjorken_w_ns, T_conformal, HBARC

E0, TAU0, TAU1 = 30.0, 0.6, 10.0


def run_cell(conformal, h, eta_s, t1=TAU1):
    o = Oracle(1, 1, 1, 1.0, 1.0, 1.0, h, TAU0, conformal, eta_s, bc=(1, 1, 1), pi_limit_xi=0.0)
    T = np.zeros((4, 1, 1, 1)); T[0] = E0
    pi = None
    if eta_s > 0:
        w0 = bjorken_w_ns(E0, TAU0, eta_s)
        pi = np.zeros((10, 1, 1, 1)); pi[9] = w0; pi[4] = pi[7] = -w0 / 2
    o.load(T, pi)
    o.step(int(round((t1 - TAU0) / h)))
    e, u, p = o.read()
    return o.diag()["tau"], e.ravel()[0], u[:, 0, 0, 0], p[:, 0, 0, 0]


def test_ideal_bjorken_1e6(conformal):
    # Eq.68 with pi=0, P=e/3: e tau^{4/3} constant.  Heun drift is O(h^2): needs h<=0.003 for 1e-6.
    tau, e, u, _ = run_cell(conformal, 0.002, 0.0)
    assert abs(tau - TAU1) < 1e-9
    assert abs(e * tau ** (4 / 3) / (E0 * TAU0 ** (4 / 3)) - 1) < 1e-6
    assert np.allclose(u, [1, 0, 0, 0], atol=1e-15)


def test_ideal_bjorken_second_order(conformal):
    errs = []
    for h in (0.04, 0.02, 0.01):
        tau, e, _, _ = run_cell(conformal, h, 0.0)
        errs.append(abs(e * tau ** (4 / 3) / (E0 * TAU0 ** (4 / 3)) - 1))
    assert 3.5 < errs[0] / errs[1] < 4.5 and 3.5 < errs[1] / errs[2] < 4.5


@pytest.mark.parametrize("eta_s", [0.08, 0.2])
def test_viscous_bjorken_vs_is_ode(conformal, eta_s):
    ref = bjorken_is(E0, TAU0, TAU1, eta_s)(TAU1)
    errs = []
    for h in (0.02, 0.01, 0.005):
        tau, e, u, p = run_cell(conformal, h, eta_s)
        errs.append((abs(e / ref[0] - 1), abs(p[9] / ref[1] - 1)))
        # pi~xx = pi~yy = -pi~etaeta/2 (A20), traceless, all other components zero
        assert abs(p[4] + p[9] / 2) < 1e-12 * abs(p[9]) and abs(p[7] - p[4]) < 1e-14
        assert np.all(np.abs(p[[0, 1, 2, 3, 5, 6, 8]]) < 1e-14)
    assert errs[-1][0] < 2e-6 and errs[-1][1] < 2e-6
    for k in (0, 1):
        assert 3.5 < errs[0][k] / errs[1][k] < 4.5 and 3.5 < errs[1][k] / errs[2][k] < 4.5


@pytest.mark.parametrize("eta_s", [0.08, 0.2])
def test_eq69_navier_stokes_sanity(conformal, eta_s):
    # Eq.69 is the Navier-Stokes solution; IS stays within 2 % of it (A19).
    T0 = T_conformal(E0)
    for t1 in (2.0, 5.0, 10.0):
        tau, e, _, _ = run_cell(conformal, 0.01, eta_s, t1)
        T_ns = T0 * (TAU0 / tau) ** (1 / 3) * (1 + (2.0 / 3.0) * eta_s * HBARC / (T0 * TAU0) * (1 - (TAU0 / tau) ** (2 / 3)))
        assert abs(T_conformal(e) / T_ns - 1) < 0.02
