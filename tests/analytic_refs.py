"""Analytic / ODE references used to pin the oracle (never imported by the product or the oracle).

Re-derived from PAPER.md:
  * Bjorken: Eq.68 (:386) with the IS equation Eq.4 (:58) reduced to 0+1 D (SURVEY pin 2, A19, A20)
  * Gubser: Weyl map Eq.70-71 (:404-409), back-map Eq.74-76 (:427-433, sign of Eq.75 per A21),
    IS equation with lambda_i = 0 in dS3xR (SURVEY pin 3, 4)
"""
import math

import numpy as np
from scipy.integrate import solve_ivp

HBARC = 0.1973269804
C_SB = 47.5 * math.pi ** 2 / 30.0


def T_conformal(e):
    return HBARC * (e / (C_SB * HBARC)) ** 0.25


def bjorken_is(e0, tau0, tau1, eta_s, w0=None):
    """IS Bjorken: de/dtau = -(e+P+w)/tau, dw/dtau = -(w + 4 eta_v/(3 tau))/tau_pi - (4/3) w/tau,
    w = pi~^{eta eta}; P = e/3.  Returns dense solution callable t -> (e, w)."""
    def f(t, y):
        e, w = y
        P = e / 3.0
        T = T_conformal(e)
        etav = eta_s * (e + P) / T * HBARC
        tpi = 5.0 * eta_s * HBARC / T
        return [-(e + P + w) / t, -(w + 4 * etav / (3 * t)) / tpi - (4.0 / 3.0) * w / t]
    if w0 is None:
        w0 = bjorken_w_ns(e0, tau0, eta_s)
    sol = solve_ivp(f, (tau0, tau1), [e0, w0], rtol=1e-12, atol=1e-14, dense_output=True)
    return sol.sol


def bjorken_w_ns(e0, tau0, eta_s):
    """Navier-Stokes start value pi~^{eta eta} = -4 eta_v/(3 tau) (PAPER.md:384 with A20)."""
    T0 = T_conformal(e0)
    etav = eta_s * (4.0 * e0 / 3.0) / T0 * HBARC
    return -4.0 * etav / (3.0 * tau0)


class Gubser:
    """Gubser flow for conformal IS hydro (lambda_i = 0), q = 1/L."""

    def __init__(self, q=1.0, eta_s=0.2, That0=1.2, rho_range=(-6.0, 3.0)):
        self.q, self.eta_s, self.That0 = q, eta_s, That0
        if eta_s > 0:
            def f(rho, y):
                Th, wb = y
                th = math.tanh(rho)
                return [Th * th * (-2.0 / 3.0 + wb / 3.0),
                        -(4.0 / 3.0) * wb * wb * th - (Th / (5.0 * eta_s)) * (wb - (4.0 / 3.0) * eta_s * th / Th)]
            kw = dict(rtol=1e-12, atol=1e-14, dense_output=True)
            self._neg = solve_ivp(f, (0.0, rho_range[0]), [That0, 0.0], **kw).sol
            self._pos = solve_ivp(f, (0.0, rho_range[1]), [That0, 0.0], **kw).sol

    def hat(self, rho):
        """(T^, pibar) at rho (arrays)."""
        rho = np.asarray(rho, dtype=np.float64)
        if self.eta_s == 0:
            return self.That0 * np.cosh(rho) ** (-2.0 / 3.0), np.zeros_like(rho)
        flat = np.atleast_1d(rho).ravel()
        out = np.empty((2, flat.size))
        neg = flat < 0
        if neg.any():
            out[:, neg] = self._neg(flat[neg])
        if (~neg).any():
            out[:, ~neg] = self._pos(flat[~neg])
        return out[0].reshape(rho.shape), out[1].reshape(rho.shape)

    def fields(self, tau, X, Y):
        """Returns e, u~ (4 comps: tau,x,y,eta), pi~ (10 comps) on arrays X, Y at proper time tau."""
        q = self.q
        r = np.sqrt(X * X + Y * Y)
        sinh_rho = -(1.0 - q * q * tau * tau + q * q * r * r) / (2.0 * q * tau)
        rho = np.arcsinh(sinh_rho)
        Th, wb = self.hat(rho)
        e = C_SB * Th ** 4 * HBARC / tau ** 4
        vr = 2.0 * q * q * tau * r / (1.0 + q * q * tau * tau + q * q * r * r)
        kappa = np.arctanh(vr)
        with np.errstate(invalid="ignore", divide="ignore"):
            nx = np.where(r > 0, X / r, 0.0)
            ny = np.where(r > 0, Y / r, 0.0)
        ch, sh = np.cosh(kappa), np.sinh(kappa)
        u = np.stack([ch, sh * nx, sh * ny, np.zeros_like(r)])
        w = (4.0 / 3.0) * e * wb            # pi~^{eta eta}
        a = -w / 2.0
        pi = np.zeros((10,) + r.shape)
        pi[0] = a * sh * sh
        pi[1] = a * sh * ch * nx
        pi[2] = a * sh * ch * ny
        pi[4] = a * (ch * ch * nx * nx + (1.0 - nx * nx))
        pi[5] = a * (ch * ch * nx * ny - nx * ny)
        pi[7] = a * (ch * ch * ny * ny + (1.0 - ny * ny))
        pi[9] = w
        return e, u, pi

    def T_tau_mu(self, tau, X, Y):
        """Frame tensor T_f^{tau mu} (4 comps) and pi~ for hydro_load / oracle.load."""
        e, u, pi = self.fields(tau, X, Y)
        P = e / 3.0
        T = np.stack([(e + P) * u[0] * u[m] - (P if m == 0 else 0.0) + pi[m] for m in range(4)])
        return T, pi


def boost_tilde(u, pi, delta):
    """Re-express tilde components given in a Milne tetrad at rapidity eta' in the tetrad at eta = eta' - delta:
    a (tau, eta)-block boost by delta on every index (Eq.18-23 define the tetrad).
    u: [4,...] (tau, x, y, eta); pi: [10,...] in the order tt, tx, ty, tn, xx, xy, xn, yy, yn, nn."""
    ch, sh = np.cosh(delta), np.sinh(delta)
    shape = u.shape[1:]
    L = np.zeros((4, 4) + shape)
    L[0, 0] = ch; L[0, 3] = sh; L[3, 0] = sh; L[3, 3] = ch
    L[1, 1] = 1.0; L[2, 2] = 1.0
    un = np.einsum("ab...,b...->a...", L, u)
    idx = [(0, 0), (0, 1), (0, 2), (0, 3), (1, 1), (1, 2), (1, 3), (2, 2), (2, 3), (3, 3)]
    P = np.zeros((4, 4) + shape)
    for k, (a, b) in enumerate(idx):
        P[a, b] = pi[k]; P[b, a] = pi[k]
    Pn = np.einsum("ac...,bd...,cd...->ab...", L, L, P)
    pin = np.stack([Pn[a, b] for (a, b) in idx])
    return un, pin


class GubserLambda1(Gubser):
    """The paper's own closed-form second-order Gubser solution (Eq.72-76): with the lambda_1 term of
    Eq.4 and  eta_hat lambda1_hat^2 = 3 tau_pi_hat,
        e_hat ~ cosh(rho)^-(8/3 - 2/lambda1_hat),   pi_hat^{eta eta} = (2/lambda1_hat) e_hat  (C = -2A = -2B),
    and the velocity of the ideal solution (fixed by the conformal map).  In the notation of Gubser above:
    T_hat = T_hat0 cosh(rho)^-(2/3 - 1/(2 lambda1_hat)),  pibar = pi_hat^{eta eta}/(T_hat s_hat) = 3/(2 lambda1_hat).
    With tau_pi = c_tau eta_v/(T s) the constraint reads c_tau = 4 lambda1_hat^2 / 9  (derivation: DESIGN.md A27)."""

    def __init__(self, q=0.5, lambda1_hat=-10.0, That0=1.2):
        self.q, self.eta_s, self.That0, self.lam = q, 0.2, That0, lambda1_hat
        self.c_tau = 4.0 * lambda1_hat ** 2 / 9.0

    def hat(self, rho):
        rho = np.asarray(rho, dtype=np.float64)
        Th = self.That0 * np.cosh(rho) ** (-(2.0 / 3.0 - 1.0 / (2.0 * self.lam)))
        return Th, np.full_like(rho, 3.0 / (2.0 * self.lam))


class ShiftedGubser:
    """SURVEY 8c pin 5: the Gubser solution translated by (t0, z0) in the (t, z) plane.  Poincare invariance
    makes it an exact solution of the same equations; seen from the unshifted Milne frame it has u~^eta != 0,
    eta-gradients and every component of pi~ non-zero, so all Christoffel-born terms (Eq.24-26, 31, 35-38) act."""

    def __init__(self, gubser, t0, z0):
        self.g, self.t0, self.z0 = gubser, t0, z0

    def fields(self, tau, X, Y, ETA):
        t = tau * np.cosh(ETA) + self.t0
        z = tau * np.sinh(ETA) + self.z0
        taup = np.sqrt(t * t - z * z)
        etap = np.arctanh(z / t)
        e, u, pi = self.g.fields(taup, X, Y)
        u, pi = boost_tilde(u, pi, etap - ETA)
        return e, u, pi
