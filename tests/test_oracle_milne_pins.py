"""Pins of the oracle's Milne terms that only act when u~^eta != 0 (pin 5).

Bjorken and 2+1 D Gubser have u~^eta = 0, the conservation and Riemann pins run in Cartesian mode, so none of them
sees the sign of  S_T^eta = -T_f^{tau eta} (Eq.31),  the Eq.24-26 additions to nabla~_eta u~ (:143-147),
I^{mu nu} (Eq.35-38, :175-183)  or the d_eta/tau flux of a flowing state.  The printed signs of exactly these terms
were re-read (A1).  Three exact statements pin them, none of which repeats the oracle's formulas:

(a) a fluid at rest in Minkowski space, seen in Milne coordinates: u~ = (cosh eta, 0, 0, -sinh eta), e = const.
    T^{mu nu} is constant in (t, z), so T_f^{tau mu}(eta) does not depend on tau and d_tau(tau T_f^{tau mu}) = T_f^{tau mu};
    sigma = theta = Du = 0, so with pi = 0 the pi equation must stay at zero.
(b) the same fluid carrying a shear tensor pi_c that is uniform on the tau-slice: Israel-Stewart reduces to
    d_t pi_c = -pi_c/tau_pi, which in Milne variables reads d_tau(u~^tau pi~^{mu nu}) = -pi~^{mu nu}/tau_pi for all ten
    components (pi~ = Lambda(eta) pi_c Lambda(eta)^T with the (t,z) boost Lambda; derivation in the docstring below).
(c) the Poincare-shifted viscous Gubser solution (3+1 D, every term active): PDE residual of R against finite
    differences in tau of the analytic fields, converging at 2nd order.
"""
import math

import numpy as np
import pytest

from oracle import Oracle
from analytic_refs import Gubser, ShiftedGubser, T_conformal, HBARC

E0 = 3.0


def static_fluid(conformal, deta, eta_s, pi_c=None, tau=1.3, eta_lo=0.3, eta_hi=1.5):
    """RHS of the oracle on a 1 x 1 x nz column holding the Minkowski-static fluid; returns eta, S_T, S_pi, u, pi."""
    nz = int(round((eta_hi - eta_lo) / deta)) + 1
    eta = eta_lo + deta * np.arange(nz)
    e = np.full((nz, 1, 1), E0)
    u3 = np.zeros((3, nz, 1, 1)); u3[2, :, 0, 0] = -np.sinh(eta)
    pi = None
    if pi_c is not None:
        ch, sh = np.cosh(eta), np.sinh(eta)
        pi = np.zeros((10, nz, 1, 1))
        for k in range(nz):
            L = np.eye(4); L[0, 0] = ch[k]; L[0, 3] = -sh[k]; L[3, 0] = -sh[k]; L[3, 3] = ch[k]
            m = L @ pi_c @ L.T
            pi[:, k, 0, 0] = [m[0, 0], m[0, 1], m[0, 2], m[0, 3], m[1, 1], m[1, 2], m[1, 3], m[2, 2], m[2, 3], m[3, 3]]
    # the grid is centred by the oracle on its own origin, which never enters the RHS: only deta does
    o = Oracle(1, 1, nz, 1.0, 1.0, deta, 0.01, tau, conformal, eta_s, pi_limit_xi=0.0, minmod_theta=1.1)
    o.set_state(e, u3, pi)
    ST, SP = o.rhs(np.zeros((4, nz, 1, 1)), tau)
    return eta, ST[:, :, 0, 0], SP[:, :, 0, 0], u3, pi


def test_static_fluid_in_milne_coordinates(conformal):
    """(a) S_T,tot = T_f^{tau mu} = ((e+P) cosh^2 eta - P, 0, 0, -(e+P) cosh eta sinh eta) and S_pi,tot = 0.
    Fails if: S_T^eta has the printed sign of Eq.31 (error 2 T^{tau eta}); S_T^tau has it (2 T^{eta eta}); either
    Eq.25/26 addition is dropped or flipped (sigma != 0 gives S_pi = O(eta_v/tau)); the eta flux lacks its 1/tau."""
    P = E0 / 3
    errs = []
    for deta in (0.02, 0.01):
        eta, ST, SP, _, _ = static_fluid(conformal, deta, 0.2)
        w = slice(4, -4)                                     # outflow ends are not part of the statement
        exact = np.stack([(E0 + P) * np.cosh(eta) ** 2 - P, 0 * eta, 0 * eta, -(E0 + P) * np.cosh(eta) * np.sinh(eta)])
        eT = np.abs(ST - exact)[:, w].max() / np.abs(exact).max()
        eP = np.abs(SP)[:, w].max() / (E0 + P)               # scale: eta_v sigma / tau_pi ~ (e+P)/5 * O(1/tau)
        errs.append((eT, eP))
    print("static fluid", errs)
    assert errs[1][0] < 1.5e-4 and errs[1][1] < 1.5e-4
    assert 3.3 < errs[0][0] / errs[1][0] < 4.7           # 2nd order away from the eta = 0 extremum
    assert errs[0][1] / errs[1][1] > 3.3


def test_slice_uniform_shear_tensor(conformal):
    """(b) With sigma = theta = Du = 0 Eq.4 is u^l d_l pi^{mu nu} = -pi^{mu nu}/tau_pi, i.e. d_t pi_c = -pi_c/tau_pi for the
    Minkowski components.  Slice-uniform means d_eta pi_c = 0 at fixed tau, hence d_z = -tanh(eta) d_t and
    d_tau|_eta = cosh(eta) d_t + sinh(eta) d_z = d_t / cosh(eta): with u~^tau = cosh(eta) constant in tau,
    d_tau(u~^tau pi~) = Lambda (d_t pi_c) Lambda^T = -pi~/tau_pi.  All of pi~^{tau tau}, pi~^{tau eta}, pi~^{eta eta}, pi~^{x eta},
    pi~^{tau x} are non-zero, so every line of Eq.35-38 contributes.  Fails if I^{mu nu} or pi~ u~^tau/tau keep the
    printed sign of Eq.33, if any of Eq.35-38 is mis-indexed, or if the (u pi + u pi) Du term is not orthogonal."""
    a, b = 0.11, 0.07
    pi_c = np.diag([0.0, a, a, -2 * a]); pi_c[1, 3] = pi_c[3, 1] = b        # traceless, transverse to u = (1,0,0,0)
    eta_s = 0.2
    inv_taupi = T_conformal(E0) / (5 * eta_s * HBARC)                     # tau_pi = 5 eta_v/(T s)
    errs = []
    for deta in (0.02, 0.01):
        eta, ST, SP, u3, pi = static_fluid(conformal, deta, eta_s, pi_c)
        w = slice(4, -4)
        exact = -pi[:, :, 0, 0] * inv_taupi
        errs.append(np.abs(SP - exact)[:, w].max() / np.abs(exact).max())
        nz = np.abs(pi[:, :, 0, 0]).max(axis=1)
        assert all(nz[k] > 1e-3 for k in (0, 1, 3, 4, 6, 7, 9))           # tt, tx, tn, xx, xn, yy, nn all present
    print("slice-uniform shear", errs)
    assert errs[1] < 1.5e-3 and 3.0 < errs[0] / errs[1] < 5.0


@pytest.mark.parametrize("eta_s", [0.0, 0.2])
def test_shifted_gubser_pde_residual(conformal, eta_s):
    """(c) R(e, u~, d_tau u~, pi~; tau) on the shifted Gubser fields must equal d_tau(tau T_f^{tau mu}) and
    d_tau(u~^tau pi~^{mu nu}) of the same analytic fields (central differences in tau, step 1e-4), up to the O(dx^2)
    truncation error of the KT divergence and the central velocity gradients."""
    g = Gubser(1.0, eta_s)
    sg = ShiftedGubser(g, 0.7, 0.45)
    tau = 1.2

    def residual(n, d):
        x = 0.6 + d * np.arange(n)                     # a window without extrema of e (minmod stays unclipped)
        y = 0.4 + d * np.arange(n)
        z = -0.9 + d * np.arange(n)
        Z, Y, X = np.meshgrid(z, y, x, indexing="ij")
        dt = 1e-4
        e, u, pi = sg.fields(tau, X, Y, Z)
        ep, up, pip = sg.fields(tau + dt, X, Y, Z)
        em, um, pim = sg.fields(tau - dt, X, Y, Z)

        def QT(t, e_, u_, p_):
            P = e_ / 3
            return t * np.stack([(e_ + P) * u_[0] * u_[m] - (P if m == 0 else 0.0) + p_[m] for m in range(4)])
        dQT = (QT(tau + dt, ep, up, pip) - QT(tau - dt, em, um, pim)) / (2 * dt)
        dQP = (up[0] * pip - um[0] * pim) / (2 * dt)
        dtu = (up - um) / (2 * dt)
        o = Oracle(n, n, n, d, d, d, 0.01, tau, conformal, eta_s, pi_limit_xi=0.0, minmod_theta=2.0)
        o.set_state(e, u[1:], pi if eta_s > 0 else None)
        ST, SP = o.rhs(dtu, tau)
        w = (slice(3, -3),) * 3
        rT = np.abs(ST - dQT)[(slice(None),) + w].max() / np.abs(dQT).max()
        # pi: L1 norm.  Components of u~^a pi~ change sign inside any 3-D window; minmod clips the slope on those
        # surfaces, which is first order there (max norm: ratio 2, measured) and second order in L1.
        rP = np.abs(SP - dQP)[(slice(None),) + w].mean() / max(np.abs(dQP).max(), 1e-300) if eta_s > 0 else 0.0
        assert np.abs(u[3]).max() > 0.05                       # the flow really has u~^eta != 0
        return rT, rP
    c, f = residual(14, 0.04), residual(22, 0.02)
    print("shifted Gubser residual", eta_s, c, f)
    assert f[0] < 1e-4 and 2.9 < c[0] / f[0] < 5.5             # measured 1.8e-4 -> 5.5e-5
    if eta_s > 0:
        assert f[1] < 3e-4 and c[1] / f[1] > 3.3               # measured 9.8e-4 -> 1.6e-4
