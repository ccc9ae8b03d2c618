"""Pins of the oracle's 8(f)-3 extension: bulk pressure Pi and net-baryon density n (PAPER.md:46-56 Eq.1-3; :153-171
Eq.28, 30, 32, 34; readings A28-A32 in the oracle's header and DESIGN.md).  Each statement is fixed by the mathematics,
not by the oracle's formulas:
  * 0+1 D Bjorken flow with shear, bulk and baryon number: the ODE system that Eq.3 / Eq.4 reduce to, integrated by
    scipy -- fails if zeta theta has the sign printed in Eq.34, if the Milne term u^tau Pi / tau is missing
    (4/3 -> 1/3), if Pi is left out of T^{eta eta}, or if n tau is not conserved;
  * advection of a baryon profile by a uniform flow (exact: n(x - v t));
  * the force of a bulk-pressure gradient on a fluid at rest, d_tau T^{tau x} = -d_x (P + Pi);
  * load -> read round trip of (e, v, Pi) through the root-find with Pi (closed-form T^{tau mu});
  * conservation of sum T^{tau mu} and sum Q_N in a periodic Cartesian box to rounding; the bulk limiter's bound.
CPU only."""
import math

import numpy as np
import pytest
from scipy.integrate import solve_ivp

from analytic_refs import HBARC, T_conformal, bjorken_w_ns
from oracle import Oracle
from paper_1802_04449_b200 import inputs

E0, TAU0 = 30.0, 0.6


def ext_oracle(*a, zeta_s=0.0, **kw):
    o = Oracle(*a, **kw)
    o.set_option(Oracle.OPT_EXT, 1)
    o.set_option(Oracle.OPT_ZETA_S, zeta_s)
    return o


def bjorken_bulk_ode(e0, w0, Pi0, tau0, tau1, eta_s, zeta_s):
    """de/dtau = -(e + P + Pi + w)/tau;  dw/dtau as in analytic_refs.bjorken_is;
    dPi/dtau = -(Pi + zeta/tau)/tau_Pi - (4/3) Pi/tau  (Eq.3 with theta = 1/tau, tau_Pi = tau_pi, zeta = (zeta/s) s)."""
    def f(t, y):
        e, w, Pb = y
        P = e / 3.0
        T = T_conformal(e)
        s_hbarc = (e + P) / T * HBARC
        tpi = 5.0 * eta_s * HBARC / T
        return [-(e + P + Pb + w) / t,
                -(w + 4 * eta_s * s_hbarc / (3 * t)) / tpi - (4.0 / 3.0) * w / t,
                -(Pb + zeta_s * s_hbarc / t) / tpi - (4.0 / 3.0) * Pb / t]
    return solve_ivp(f, (tau0, tau1), [e0, w0, Pi0], rtol=1e-12, atol=1e-14).y[:, -1]


def test_bjorken_with_bulk_and_baryon(conformal):
    eta_s, zeta_s, t1, n0 = 0.2, 0.05, 3.0, 0.7
    w0 = bjorken_w_ns(E0, TAU0, eta_s)
    s0 = (4.0 * E0 / 3.0) / T_conformal(E0) * HBARC
    Pi0 = -zeta_s * s0 / TAU0                                     # Navier-Stokes start, Pi = -zeta theta
    ref = bjorken_bulk_ode(E0, w0, Pi0, TAU0, t1, eta_s, zeta_s)
    errs = []
    for h in (0.02, 0.01, 0.005):
        o = ext_oracle(1, 1, 1, 1.0, 1.0, 1.0, h, TAU0, conformal, eta_s, bc=(1, 1, 1), pi_limit_xi=0.0, zeta_s=zeta_s)
        pi = np.zeros((10, 1, 1, 1)); pi[9] = w0; pi[4] = pi[7] = -w0 / 2
        T = np.zeros((4, 1, 1, 1)); T[0] = E0                     # u = 0: T^{tau tau} = e, whatever Pi is
        o.load_ext(T, pi, np.full((1, 1, 1), Pi0), np.full((1, 1, 1), n0))
        o.step(int(round((t1 - TAU0) / h)))
        e, u, p = o.read()
        Pb, nb = o.read_ext()
        tau = o.diag()["tau"]
        errs.append([abs(e.ravel()[0] / ref[0] - 1), abs(p[9].ravel()[0] / ref[1] - 1), abs(Pb.ravel()[0] / ref[2] - 1)])
        assert abs(nb.ravel()[0] * tau / (n0 * TAU0) - 1) < 1e-12           # Eq.28 with S_N = 0: n tau constant
    errs = np.array(errs)
    print("Bjorken bulk: errors (e, pi^etaeta, Pi) per h", errs, "ref", ref)
    assert errs[-1].max() < 2e-5
    assert np.all(errs[0] / errs[1] > 3.5) and np.all(errs[0] / errs[1] < 4.5)
    assert np.all(errs[1] / errs[2] > 3.5) and np.all(errs[1] / errs[2] < 4.5)
    assert ref[2] < 0 and abs(ref[2]) > 1e-3 * ref[0] / 3        # the bulk pressure is negative and not negligible


def test_baryon_profile_advected_by_uniform_flow(crossover):
    """Uniform e and velocity in a periodic Cartesian box: the flow stays uniform and n obeys d_t(n gamma) + d_x(n gamma v)
    = 0, i.e. n(x, t) = n0(x - v t).  Second order in dx (smooth profile, theta = 2 keeps minmod unclipped away from the
    extrema; the L1 norm is taken)."""
    v, t1 = 0.4, 1.0
    errs = []
    for n in (40, 80):
        dx = 4.0 / n
        h = 0.2 * dx
        x = (np.arange(n) - (n - 1) / 2) * dx
        o = ext_oracle(n, 1, 1, dx, 1.0, 1.0, h, 0.0, crossover, 0.08, bc=(1, 1, 1), geometry=1, minmod_theta=2.0)
        g = 1 / math.sqrt(1 - v * v)
        e = np.full((1, 1, n), 5.0)
        u3 = np.zeros((3, 1, 1, n)); u3[0] = g * v
        o.set_state(e, u3)
        prof = lambda xx: 1.0 + 0.5 * np.sin(2 * math.pi * xx / 4.0)
        o.set_ext(None, prof(x).reshape(1, 1, n))
        o.step(int(round(t1 / h)))
        _, nb = o.read_ext()
        e1, u1, _ = o.read()
        assert np.abs(e1 - 5.0).max() < 1e-12 and np.abs(u1[1] - g * v).max() < 1e-12
        errs.append(np.abs(nb.ravel() - prof(x - v * t1)).mean())
    print("baryon advection L1 errors", errs)
    assert errs[1] < 2e-3 and errs[0] / errs[1] > 3.0


def test_bulk_pressure_gradient_accelerates_the_fluid(crossover):
    """Fluid at rest, uniform e, Pi(x) = A sin(kx), zeta = 0: after one short step T^{tau x} = -h d_x(P + Pi) + O(h^2).
    Fails if Pi is missing from the momentum flux or enters with the wrong sign (A28)."""
    L, A, h = 4.0, 0.02, 1e-3
    k = 2 * math.pi / L
    errs = []
    for n in (64, 128):
        dx = L / n
        x = (np.arange(n) - (n - 1) / 2) * dx
        o = ext_oracle(n, 1, 1, dx, 1.0, 1.0, h, 0.0, crossover, 0.08, bc=(1, 1, 1), geometry=1, minmod_theta=2.0)
        o.set_state(np.full((1, 1, n), 5.0), np.zeros((3, 1, 1, n)))
        o.set_ext((A * np.sin(k * x)).reshape(1, 1, n), None)
        o.step(1)
        Tx = o.read_T()[1].ravel()
        exact = -h * A * k * np.cos(k * x)
        errs.append((np.abs(Tx - exact).mean() / (h * A * k), np.abs(Tx - exact).max() / (h * A * k)))
    print("bulk force relative errors (L1, max) at n = 64, 128:", errs)
    # L1: second order away from the two extrema of Pi, where the limiter clips the slope (first order there, max norm)
    # (plus an O(h / tau_Pi) ~ 0.2 % floor: Pi relaxes during the step)
    assert errs[1][0] < 3e-3 and errs[0][0] / errs[1][0] > 2.0 and errs[1][1] < 0.03


def test_rootfind_with_bulk_round_trip(crossover):
    rng = np.random.default_rng(11)
    n = 6
    e = rng.uniform(0.5, 20.0, (n, n, n))
    v = rng.uniform(-0.4, 0.4, (3, n, n, n))
    o = ext_oracle(n, n, n, 0.2, 0.2, 0.2, 0.02, 1.0, crossover, 0.08, bc=(1, 1, 1), geometry=1)
    P = np.vectorize(lambda q: o.eos(q)[0])(e)
    Pb = rng.uniform(-0.5, 0.5, e.shape) * P
    g2 = 1 / (1 - (v ** 2).sum(0))
    T = np.stack([(e + P + Pb) * g2 - (P + Pb)] + [(e + P + Pb) * g2 * v[a] for a in range(3)])     # Eq.1 with Pi (A28)
    o.load_ext(T, None, Pb, None)
    e1, u1, _ = o.read()
    assert np.abs(e1 / e - 1).max() < 1e-12
    assert np.abs(u1[1:] - np.sqrt(g2) * v).max() < 1e-12
    assert np.abs(o.read_T() - T).max() < 1e-12 * np.abs(T).max()


def test_conservation_and_bulk_limiter(crossover):
    """Periodic Cartesian box, smooth random state with flow, shear, bulk and baryon density: sum T^{tau mu} and
    sum n gamma are conserved to rounding (flux form); with a huge initial Pi the limiter leaves |Pi| <= xi P."""
    e, v, pi = inputs.ic_random_smooth(10, 9, 8, seed=5, vmax=0.3)
    rng = np.random.default_rng(3)
    o = ext_oracle(10, 9, 8, 0.2, 0.2, 0.2, 0.02, 1.0, crossover, 0.1, bc=(1, 1, 1), geometry=1, zeta_s=0.03)
    P = np.vectorize(lambda q: o.eos(q)[0])(e)
    Pb = 0.3 * P * rng.uniform(-1, 1, e.shape)
    nb = 1.0 + 0.5 * rng.uniform(-1, 1, e.shape)
    g2 = 1 / (1 - (v ** 2).sum(0))
    T = np.stack([(e + P + Pb) * g2 - (P + Pb)] + [(e + P + Pb) * g2 * v[a] for a in range(3)]) + pi[:4]
    o.load_ext(T, pi, Pb, nb)
    T0 = o.read_T().reshape(4, -1).sum(1)
    u0 = o.read()[1]
    N0 = (o.read_ext()[1] * u0[0]).sum()
    o.step(5)
    T1 = o.read_T().reshape(4, -1).sum(1)
    N1 = (o.read_ext()[1] * o.read()[1][0]).sum()
    d = o.diag()
    assert d["floored"] == 0 and d["clamped"] == 0
    assert np.abs(T1 - T0).max() < 1e-12 * abs(T0[0]) and abs(N1 / N0 - 1) < 1e-12
    # limiter
    o2 = ext_oracle(10, 9, 8, 0.2, 0.2, 0.2, 0.02, 1.0, crossover, 0.1, bc=(1, 1, 1), geometry=1, pi_limit_xi=0.5)
    o2.set_state(e, np.sqrt(g2) * v)
    o2.set_ext(5.0 * P, None)
    o2.step(1)
    e2 = o2.read()[0]
    P2 = np.vectorize(lambda q: o2.eos(q)[0])(e2)
    assert np.all(np.abs(o2.read_ext()[0]) <= 0.5 * P2 * (1 + 1e-12))
