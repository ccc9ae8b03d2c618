"""Oracle pins 3-4: Gubser flow, PAPER.md:394-457 (Eq.70-76; sign of Eq.75 per A21)."""
import numpy as np
import pytest

from oracle import Oracle
from analytic_refs import Gubser


def gubser_errors(conformal, eta_s, dx, t1, theta=2.0, L=5.0):
    n = int(round(2 * L / dx)) + 1
    x = (np.arange(n) - (n - 1) / 2) * dx
    Y, X = np.meshgrid(x, x, indexing="ij")
    X, Y = X[None], Y[None]
    g = Gubser(1.0, eta_s)
    h = dx / 10
    T, pi = g.T_tau_mu(1.0, X, Y)
    o = Oracle(n, n, 1, dx, dx, 1.0, h, 1.0, conformal, eta_s, pi_limit_xi=0.0, minmod_theta=theta)
    o.load(T, pi if eta_s > 0 else None)
    o.set_history(g.fields(1.0 - h, X, Y)[1][1:])
    o.step(int(round((t1 - 1.0) / h)))
    e, u, p = o.read()
    ea, ua, pa = g.fields(t1, X, Y)
    m = ea > 1e-3 * ea.max()
    l2 = lambda a, b: float(np.sqrt(((a - b)[m] ** 2).sum() / (b[m] ** 2).sum()))
    vr = np.sqrt(u[1] ** 2 + u[2] ** 2) / u[0]
    vra = np.sqrt(ua[1] ** 2 + ua[2] ** 2) / ua[0]
    out = dict(e=l2(e, ea), vr=l2(vr, vra))
    if eta_s > 0:
        out.update(pixx=l2(p[4], pa[4]), pinn=l2(p[9], pa[9]))
        # eta-components that must stay zero in a boost-invariant 2+1 D flow
        assert np.all(np.abs(p[[3, 6, 8]]) < 1e-13) and np.all(np.abs(u[3]) < 1e-13)
    return out


def test_gubser_reference_is_traceless_transverse():
    g = Gubser(1.0, 0.2)
    x = np.linspace(-5, 5, 41)
    Y, X = np.meshgrid(x, x, indexing="ij")
    e, u, pi = g.fields(1.7, X, Y)
    tr = pi[0] - pi[4] - pi[7] - pi[9]
    assert np.abs(tr).max() < 1e-14
    # u_mu pi^{mu nu} = 0 for nu = tau, x, y
    t0 = u[0] * pi[0] - u[1] * pi[1] - u[2] * pi[2]
    t1 = u[0] * pi[1] - u[1] * pi[4] - u[2] * pi[5]
    t2 = u[0] * pi[2] - u[1] * pi[5] - u[2] * pi[7]
    assert max(np.abs(t0).max(), np.abs(t1).max(), np.abs(t2).max()) < 1e-14


@pytest.mark.parametrize("eta_s", [0.0, 0.2])
def test_gubser_converges_second_order(conformal, eta_s):
    """dx, h halved together (0.1 -> 0.05, the stated resolution), tau = 1 -> 1.25: the error of e falls 4x (measured
    4.02 ideal, 4.62 viscous).  pi~xx, pi~etaeta fall 3.2-3.3x.  v_r is limited by the ultra-relativistic ring at the
    vacuum edge, where minmod clips (ratio 1.9 ideal, 2.6 viscous, measured; BASELINE.md section 4 has the same)."""
    c = gubser_errors(conformal, eta_s, 0.1, 1.25)
    f = gubser_errors(conformal, eta_s, 0.05, 1.25)
    print("gubser convergence", eta_s, c, f)
    assert f["e"] < 0.0025 and 3.6 < c["e"] / f["e"] < 5.0
    assert c["vr"] / f["vr"] > (1.7 if eta_s == 0 else 2.4)
    if eta_s > 0:
        assert c["pixx"] / f["pixx"] > 2.9 and c["pinn"] / f["pinn"] > 3.0


# relative L2 errors of an INDEPENDENT numpy restatement of SURVEY 8c (the survey's throw-away
# probe, written before the oracle existed) on configs[1]b, 201x201, dx = 0.05, h = dx/10, at tau = 2, 3, 4.
# Two significant digits, as printed there.  The scheme itself does not reach 1 % on e at tau = 4 (the error sits on the
# ultra-relativistic ring r ~ tau); the numbers are asserted as measured values instead of being left out.
SURVEY_PROBE = {
    (0.0, 1.1): dict(e=(1.1e-2, 2.5e-2, 4.1e-2), vr=(5.5e-3, 3.8e-3, 1.4e-3)),
    (0.0, 2.0): dict(e=(5.2e-3, 1.4e-2, 3.1e-2)),
    (0.2, 1.1): dict(e=(1.2e-2, 2.2e-2, 4.0e-2), vr=(1.2e-3, 1.0e-3, 1.1e-3), pinn=(7.8e-3, 2.0e-2, 4.3e-2),
                     pixx=(4.6e-2, 1.0e-1, 2.6e-1)),
    (0.2, 2.0): dict(e=(5.6e-3, 1.4e-2, 2.9e-2), pinn=(5.0e-3, 1.6e-2, 3.5e-2), pixx=(2.8e-2, 8.5e-2, 1.9e-1)),
}
# this oracle at tau = 1.5 (same runs), measured: asserted to +-10 %
MEASURED_T15 = {
    (0.0, 1.1): dict(e=7.4e-3, vr=3.8e-3), (0.0, 2.0): dict(e=3.0e-3, vr=4.3e-3),
    (0.2, 1.1): dict(e=6.28e-3, vr=1.04e-3, pixx=1.92e-2, pinn=4.73e-3),
    (0.2, 2.0): dict(e=2.72e-3, vr=8.6e-4, pixx=9.2e-3, pinn=2.09e-3),
}


@pytest.mark.parametrize("eta_s,theta", sorted(SURVEY_PROBE))
def test_gubser_configs1b_to_tau4(conformal, eta_s, theta):
    """configs[1]b at the stated resolution, tau = 1 -> 4, production limiter (theta = 1.1) and theta = 2."""
    dx, n = 0.05, 201
    x = (np.arange(n) - (n - 1) / 2) * dx
    Y, X = np.meshgrid(x, x, indexing="ij")
    X, Y = X[None], Y[None]
    g = Gubser(1.0, eta_s)
    h = dx / 10
    T, pi = g.T_tau_mu(1.0, X, Y)
    o = Oracle(n, n, 1, dx, dx, 1.0, h, 1.0, conformal, eta_s, pi_limit_xi=0.0, minmod_theta=theta)
    o.load(T, pi if eta_s > 0 else None)
    o.set_history(g.fields(1.0 - h, X, Y)[1][1:])
    t, got = 1.0, {}
    for t1 in (1.5, 2.0, 3.0, 4.0):
        o.step(int(round((t1 - t) / h))); t = t1
        e, u, p = o.read()
        ea, ua, pa = g.fields(t1, X, Y)
        m = ea > 1e-3 * ea.max()
        l2 = lambda a, b: float(np.sqrt(((a - b)[m] ** 2).sum() / (b[m] ** 2).sum()))
        vr, vra = np.sqrt(u[1] ** 2 + u[2] ** 2) / u[0], np.sqrt(ua[1] ** 2 + ua[2] ** 2) / ua[0]
        got[t1] = dict(e=l2(e, ea), vr=l2(vr, vra))
        if eta_s > 0:
            got[t1].update(pixx=l2(p[4], pa[4]), pinn=l2(p[9], pa[9]))
    print("gubser", eta_s, theta, got)
    for k, v in MEASURED_T15[(eta_s, theta)].items():
        assert abs(got[1.5][k] / v - 1) < 0.10, (k, got[1.5][k], v)
    for k, vals in SURVEY_PROBE[(eta_s, theta)].items():
        for t1, v in zip((2.0, 3.0, 4.0), vals):
            assert abs(got[t1][k] / v - 1) < 0.12, (k, t1, got[t1][k], v)
    # north_star bar (< 1 % L2) where the scheme meets it: v_r at all times; e, pi~^{eta eta} at tau = 1.5
    assert all(got[t1]["vr"] < 0.01 for t1 in got) and got[1.5]["e"] < 0.01
    if eta_s > 0:
        assert got[1.5]["pinn"] < 0.01 and np.all(np.abs(p[[3, 6, 8]]) < 1e-12)


def gubser_lambda1_run(make, dx, t1, L=8.0, lam_on=True):
    """The paper's closed-form test: L = 2 (q = 1/2), eta_v/s = 0.2, lambda1_hat = -10,
    tau_pi from eta_hat lambda1_hat^2 = 3 tau_pi_hat; tau0 = 1.  `make(n, dx, h, lam, c_tau)` builds the solver."""
    from analytic_refs import GubserLambda1
    g = GubserLambda1()
    n = int(round(2 * L / dx)) + 1
    x = (np.arange(n) - (n - 1) / 2) * dx
    Y, X = np.meshgrid(x, x, indexing="ij")
    X, Y = X[None], Y[None]
    h = dx / 10
    T, pi = g.T_tau_mu(1.0, X, Y)
    o = make(n, dx, h, g.lam if lam_on else 0.0, g.c_tau)
    o.load(np.ascontiguousarray(T), np.ascontiguousarray(pi))
    o.set_history(np.ascontiguousarray(g.fields(1.0 - h, X, Y)[1][1:]))
    o.step(int(round((t1 - 1.0) / h)))
    e, u, p = o.read()
    ea, ua, pa = g.fields(t1, X, Y)
    m = ea > 1e-3 * ea.max()
    l2 = lambda a, b: float(np.sqrt(((a - b)[m] ** 2).sum() / (b[m] ** 2).sum()))
    vr, vra = np.sqrt(u[1] ** 2 + u[2] ** 2) / u[0], np.sqrt(ua[1] ** 2 + ua[2] ** 2) / ua[0]
    # "-tau^2 pi^{eta eta} is roughly two times pi^{xx}" at the centre
    c = n // 2
    ratio = -p[9][0, c, c] / p[4][0, c, c]
    return dict(e=l2(e, ea), vr=l2(vr, vra), pixx=l2(p[4], pa[4]), pinn=l2(p[9], pa[9])), ratio, (e, u, p)


def test_gubser_lambda1_closed_form(conformal):
    """the lambda_1 term of Eq.4/33 against the paper's own closed-form solution (Eq.72-76): a pin of the
    viscous sector that needs no ODE solver.  Second order under refinement; and the SAME run without the lambda_1 term
    misses the solution by 4 % in pi^{eta eta} (so the term is really exercised)."""
    def make(n, dx, h, lam, c_tau):
        o = Oracle(n, n, 1, dx, dx, 1.0, h, 1.0, conformal, 0.2, pi_limit_xi=0.0, minmod_theta=2.0)
        o.set_option(Oracle.OPT_LAMBDA1_HAT, lam)
        o.set_option(Oracle.OPT_C_TAU, c_tau)
        return o
    c, rc, _ = gubser_lambda1_run(make, 0.2, 1.5)
    f, rf, _ = gubser_lambda1_run(make, 0.1, 1.5)
    print("gubser lambda1", c, f, rc, rf)
    assert f["e"] < 1.5e-3 and f["pixx"] < 1.5e-3 and f["pinn"] < 1.5e-3 and f["vr"] < 0.01      # measured 1.1e-3, 9.8e-4, 1.2e-3
    assert c["e"] / f["e"] > 3.5 and c["pixx"] / f["pixx"] > 3.0 and c["pinn"] / f["pinn"] > 3.0
    assert abs(rf - 2.0) < 0.05
    off, _, _ = gubser_lambda1_run(make, 0.1, 1.5, lam_on=False)
    assert off["pinn"] > 0.03
