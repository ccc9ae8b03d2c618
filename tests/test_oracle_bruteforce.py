"""Oracle pin 7: brute-force agreement of the oracle's sweep implementation of the RHS operator
with an independent per-cell evaluation on 4^3 grids (periodic and outflow, Milne and Cartesian).

The per-cell evaluator below gathers its own 13 points and evaluates PAPER.md Eq.27-44 from scratch, with
tensors as 4x4 numpy arrays and index gymnastics done by einsum -- none of the oracle's helper structure
(flat component lists, precomputed point tables, face functions).  A second test checks the oracle's expanded
sigma^{mu nu} against the projector DEFINITION of Eq.5 (they differ only by the discretisation error of
u_b d_a u^b = 0), which catches sign / index mistakes in the expansion."""
import itertools
import math

import numpy as np
import pytest

from oracle import Oracle
from paper_1802_04449_b200 import inputs

G = np.diag([1.0, -1.0, -1.0, -1.0])
PIDX = {(0, 0): 0, (0, 1): 1, (0, 2): 2, (0, 3): 3, (1, 1): 4, (1, 2): 5, (1, 3): 6, (2, 2): 7, (2, 3): 8, (3, 3): 9}
HBARC = 0.1973269804


def pi_matrix(p10):
    m = np.zeros((4, 4))
    for (a, b), k in PIDX.items():
        m[a, b] = m[b, a] = p10[k]
    return m


def minmod3(a, b, c):
    if a > 0 and b > 0 and c > 0:
        return min(a, b, c)
    if a < 0 and b < 0 and c < 0:
        return max(a, b, c)
    return 0.0


class Brute:
    def __init__(self, e, u3, pi10, d, bc, milne, tau, h_theta, eta_s, c_sb):
        self.e, self.u3, self.pi10 = e, u3, pi10
        self.n = e.shape[::-1]            # (nx, ny, nz); arrays are [k][j][i]
        self.d, self.bc, self.milne, self.tau, self.theta, self.eta_s, self.c_sb = d, bc, milne, tau, h_theta, eta_s, c_sb

    def wrap(self, ijk):
        out = []
        for a in range(3):
            n = self.n[a]
            out.append(ijk[a] % n if self.bc[a] == 1 else min(max(ijk[a], 0), n - 1))
        return tuple(out)

    def point(self, ijk):
        """u^mu (4), T_f^{mu nu} (4x4), pi^{mu nu} (4x4), e, P, signal speeds (3) at a (wrapped) point."""
        i, j, k = self.wrap(ijk)
        e = self.e[k, j, i]
        P = e / 3.0                                              # EOSI
        ui = self.u3[:, k, j, i]
        u = np.array([math.sqrt(1.0 + ui @ ui), *ui])
        pi = pi_matrix(self.pi10[:, k, j, i]) if self.eta_s > 0 else np.zeros((4, 4))
        T = (e + P) * np.outer(u, u) - P * G + pi                # Eq.1 in tilde components
        v = ui / u[0]
        cs2 = 1.0 / 3.0
        c = [(abs(v[a]) * (1 - cs2) + math.sqrt(cs2) * math.sqrt(max((1 - v @ v) * (1 - v @ v * cs2 - v[a] ** 2 * (1 - cs2)), 0.0)))
             / (1 - v @ v * cs2) for a in range(3)]
        return u, T, pi, e, P, c

    def kt_face(self, Q, F, c):
        """H_{i+1/2} from four consecutive values (Eq.41-44); Q, F lists of 4, c = face speed."""
        th = self.theta
        sq = [minmod3(th * (Q[k] - Q[k - 1]), 0.5 * (Q[k + 1] - Q[k - 1]), th * (Q[k + 1] - Q[k])) for k in (1, 2)]
        sf = [minmod3(th * (F[k] - F[k - 1]), 0.5 * (F[k + 1] - F[k - 1]), th * (F[k + 1] - F[k])) for k in (1, 2)]
        Ql, Qr = Q[1] + 0.5 * sq[0], Q[2] - 0.5 * sq[1]
        Fl, Fr = F[1] + 0.5 * sf[0], F[2] - 0.5 * sf[1]
        return 0.5 * (Fr + Fl) - 0.5 * c * (Qr - Ql)

    def rhs_cell(self, ijk, dtu):
        tau, tf = self.tau, (self.tau if self.milne else 1.0)
        u0, T0, pi0, e0, P0, _ = self.point(ijk)
        ST, SP = np.zeros(4), np.zeros((4, 4))
        grad = np.zeros((4, 4))
        grad[0] = dtu
        for a in range(3):
            pts = [self.point(tuple(ijk[b] + (s if b == a else 0) for b in range(3))) for s in (-2, -1, 0, 1, 2)]
            scale = 1.0 / self.d[a] / (tau if (a == 2 and self.milne) else 1.0)
            cl, cr = max(pts[1][5][a], pts[2][5][a]), max(pts[2][5][a], pts[3][5][a])
            for mu in range(4):                                   # Eq.27: Q = tau T^{tau mu}, F = tau T^{a mu}
                Q = [tf * p[1][0, mu] for p in pts]
                F = [tf * p[1][a + 1, mu] for p in pts]
                ST[mu] -= (self.kt_face(Q[1:5], F[1:5], cr) - self.kt_face(Q[0:4], F[0:4], cl)) * scale
            if self.eta_s > 0:
                for mu, nu in itertools.combinations_with_replacement(range(4), 2):   # Eq.29
                    Q = [p[0][0] * p[2][mu, nu] for p in pts]
                    F = [p[0][a + 1] * p[2][mu, nu] for p in pts]
                    SP[mu, nu] -= (self.kt_face(Q[1:5], F[1:5], cr) - self.kt_face(Q[0:4], F[0:4], cl)) * scale
            grad[a + 1] = (pts[3][0] - pts[1][0]) * 0.5 * scale   # central difference (A9)
        if self.milne:
            ST[0] -= T0[3, 3]; ST[3] -= T0[0, 3]                  # Eq.31 (sign A1)
            grad[3, 0] += u0[3] / tau; grad[3, 3] += u0[0] / tau  # Eq.25, Eq.26
        if self.eta_s == 0:
            return ST, None
        theta = np.trace(grad)
        Du = u0 @ grad
        up = G @ grad                                              # nabla^mu u^nu
        sigma = up + up.T - np.outer(u0, Du) - np.outer(Du, u0) - (2.0 / 3.0) * (G - np.outer(u0, u0)) * theta
        T_ = HBARC * (e0 / (self.c_sb * HBARC)) ** 0.25
        inv_taupi = T_ / (5.0 * self.eta_s * HBARC)
        Dul = G @ Du                                               # D u_beta
        src = -pi0 * inv_taupi + (e0 + P0) / 5.0 * sigma - pi0 * theta / 3.0
        src -= np.outer(u0, pi0 @ Dul) + np.outer(pi0 @ Dul, u0)
        if self.milne:
            I = np.zeros((4, 4))                                   # Eq.35-38 as printed (A2 corrections)
            un = u0[3]
            I[0, 0] = 2 * un * pi0[0, 3]; I[0, 1] = un * pi0[3, 1]; I[0, 2] = un * pi0[3, 2]
            I[0, 3] = un * (pi0[0, 0] + pi0[3, 3]); I[3, 1] = un * pi0[0, 1]; I[3, 2] = un * pi0[0, 2]
            I[3, 3] = 2 * un * pi0[0, 3]
            I = (I + I.T - np.diag(np.diag(I))) / tau
            src -= pi0 * u0[0] / tau + I
        for mu in range(4):
            for nu in range(mu, 4):
                SP[mu, nu] += src[mu, nu]
        return ST, SP


@pytest.mark.parametrize("bc,geometry,eta_s", [((1, 1, 1), 0, 0.15), ((0, 0, 0), 0, 0.15), ((1, 0, 1), 1, 0.15),
                                               ((0, 1, 0), 0, 0.0)])
def test_rhs_bruteforce_4cubed(conformal, bc, geometry, eta_s):
    n = 4
    e, v, pi = inputs.ic_random_smooth(n, n, n, seed=21, vmax=0.5)
    u3 = v / np.sqrt(1 - (v ** 2).sum(0))
    tau, d = 0.7, (0.2, 0.25, 0.3)
    o = Oracle(n, n, n, *d, 0.02, tau, conformal, eta_s, bc=bc, geometry=geometry, minmod_theta=1.3)
    o.set_state(e, u3, pi)
    rng = np.random.default_rng(5)
    dtu = rng.normal(0, 0.5, (4, n, n, n))
    ST, SP = o.rhs(dtu, tau)
    b = Brute(e, u3, pi, d, bc, geometry == 0, tau, 1.3, eta_s, conformal["c_sb"])
    scale_T, scale_P = np.abs(ST).max(), max(np.abs(SP).max(), 1e-300)
    for k, j, i in itertools.product(range(n), repeat=3):
        bT, bP = b.rhs_cell((i, j, k), dtu[:, k, j, i])
        assert np.abs(bT - ST[:, k, j, i]).max() < 1e-13 * scale_T
        if eta_s > 0:
            for (mu, nu), m in PIDX.items():
                assert abs(bP[mu, nu] - SP[m, k, j, i]) < 1e-13 * scale_P, (mu, nu)


def test_sigma_expansion_matches_projector_definition(conformal):
    """sigma = 2 Delta^{mu nu a b} nabla_a u_b (Eq.5) vs the expansion used in S_pi: on smooth data they differ
    only through u_b d_a u^b (zero in the continuum), so the difference must fall ~4x when the grid is halved."""
    diffs = []
    for n in (8, 16):
        e, v, pi = inputs.ic_random_smooth(n, n, n, seed=3, vmax=0.4)
        u3 = v / np.sqrt(1 - (v ** 2).sum(0))
        d = (1.6 / n,) * 3
        b = Brute(e, u3, np.zeros_like(pi), d, (1, 1, 1), False, 1.0, 1.1, 0.1, conformal["c_sb"])
        worst = 0.0
        for ijk in [tuple(c * n // 8 for c in t) for t in [(1, 2, 3), (5, 0, 7), (7, 6, 4)]]:   # same physical points
            u0 = b.point(ijk)[0]
            grad = np.zeros((4, 4))
            for a in range(3):
                p3 = b.point(tuple(ijk[c] + (1 if c == a else 0) for c in range(3)))[0]
                p1 = b.point(tuple(ijk[c] - (1 if c == a else 0) for c in range(3)))[0]
                grad[a + 1] = (p3 - p1) / (2 * d[a])
            # time row chosen so that u_b d_tau u^b = 0 exactly
            grad[0, 1:] = 0.3 * u0[1:]; grad[0, 0] = (u0[1:] @ grad[0, 1:]) / u0[0]
            theta = np.trace(grad); Du = u0 @ grad; up = G @ grad
            sig_exp = up + up.T - np.outer(u0, Du) - np.outer(Du, u0) - (2 / 3) * (G - np.outer(u0, u0)) * theta
            D2 = G - np.outer(u0, u0)
            D4 = 0.5 * (np.einsum("ma,nb->mnab", D2, D2) + np.einsum("mb,na->mnab", D2, D2)) - np.einsum("mn,ab->mnab", D2, D2) / 3
            sig_def = 2 * np.einsum("mnab,ab->mn", D4, grad @ G)           # nabla_a u_b = nabla_a u^c g_cb
            assert abs(np.einsum("mn,mn->", sig_def, G)) < 1e-12 and np.abs(sig_def @ G @ u0).max() < 1e-12
            worst = max(worst, np.abs(sig_exp - sig_def).max() / np.abs(sig_def).max())
        diffs.append(worst)
    assert diffs[0] < 0.2 and diffs[1] < diffs[0] / 2.5, diffs
