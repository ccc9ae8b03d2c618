"""Pins of the freeze-out surface oracle (oracle/freezeout.py, reading A27) against what the
mathematics fixes: exact crossing positions of linear fronts, closedness of the face set, Gauss's theorem, uniform
Bjorken cooling (Eq.68) and entropy conservation of ideal Gubser flow through the
extracted surface.  CPU only."""
import math

import numpy as np

from analytic_refs import C_SB, HBARC, Gubser, T_conformal
from oracle.freezeout import NWORDS, cell_centres, surface_elements


def static_snap(e):
    u = np.zeros((4,) + e.shape)
    u[0] = 1.0
    return e, u, np.zeros((10,) + e.shape)


def decode(keys, N):
    return keys // (4 * N), (keys // N) % 4, keys % N


def test_linear_fronts_cross_exactly():
    """e linear along one axis: the interpolated crossing must sit on the front to rounding, with the normal
    pointing from hot to cold (+1 when the lower cell is hot), one face per line, and the areas of Eq.22's tilde basis.
    A weight w <-> 1-w, a sign flip or a transposed axis fails here."""
    nx, ny, nz = 9, 7, 5
    dx, dy, de = 0.2, 0.3, 0.25
    xs, ys, zs = cell_centres(nx, dx), cell_centres(ny, dy), cell_centres(nz, de)
    Z, Y, X = np.meshgrid(zs, ys, xs, indexing="ij")
    ef, tau_a, tau_b = 1.0, 2.0, 2.1
    for axis, (coord, c0, n_lines, area) in enumerate([(X, 0.137, ny * nz, tau_b * 0.1 * dy * de),
                                                      (Y, -0.291, nx * nz, tau_b * 0.1 * dx * de),
                                                      (Z, 0.06, nx * ny, 0.1 * dx * dy)]):
        for sign in (+1.0, -1.0):
            e = ef + sign * 0.7 * (c0 - coord)          # hot below c0 when sign = +1
            keys, rows = surface_elements(static_snap(e), static_snap(e), tau_a, tau_b, 3, (dx, dy, de), ef)
            slab, d, cell = decode(keys, nx * ny * nz)
            assert len(keys) == n_lines and np.all(d == 1 + axis) and np.all(slab == 3)
            np.testing.assert_allclose(rows[:, 1 + axis], c0, atol=1e-13)
            np.testing.assert_allclose(rows[:, 0], tau_b)
            np.testing.assert_allclose(rows[:, 4 + 1 + axis], sign * area, rtol=1e-14)
            other = [m for m in range(4) if m != 1 + axis]
            assert np.all(rows[:, [4 + m for m in other]] == 0.0)
    # a front in time: e falls linearly through e_f at tau_c in every cell
    tau_c = 2.0371
    ea = np.full((nz, ny, nx), ef + 0.9 * (tau_c - tau_a))
    eb = np.full((nz, ny, nx), ef + 0.9 * (tau_c - tau_b))
    keys, rows = surface_elements(static_snap(ea), static_snap(eb), tau_a, tau_b, 0, (dx, dy, de), ef)
    assert len(keys) == nx * ny * nz and np.all(decode(keys, nx * ny * nz)[1] == 0)
    np.testing.assert_allclose(rows[:, 0], tau_c, atol=1e-13)
    np.testing.assert_allclose(rows[:, 4], tau_c * dx * dy * de, rtol=1e-13)       # +: hot first, cold later
    keys2, rows2 = surface_elements(static_snap(eb), static_snap(ea), tau_a, tau_b, 0, (dx, dy, de), ef)
    np.testing.assert_allclose(rows2[:, 4], -rows2[:, 0] * dx * dy * de, rtol=1e-13)  # heating up: normal to the past
    # Cartesian geometry drops every tau
    _, rows3 = surface_elements(static_snap(ea), static_snap(eb), tau_a, tau_b, 0, (dx, dy, de), ef, geometry=1)
    np.testing.assert_allclose(rows3[:, 4], dx * dy * de, rtol=1e-13)


def blob(nx, ny, nz, amp, rng):
    xs, ys, zs = cell_centres(nx, 1.0), cell_centres(ny, 1.0), cell_centres(nz, 1.0)
    Z, Y, X = np.meshgrid(zs, ys, xs, indexing="ij")
    e = amp * np.exp(-(X ** 2 + Y ** 2) / 18.0 - Z ** 2 / 8.0)
    for _ in range(4):
        cx, cy, cz = rng.uniform(-3, 3, 3)
        e += 0.4 * amp * np.exp(-((X - cx) ** 2 + (Y - cy) ** 2 + (Z - cz) ** 2) / 3.0)
    return e


def test_face_set_is_closed():
    """The faces bound the hot region: along every grid line the signed face count is 0 (the region does not touch the
    edge), and the signed count of time-like faces is #hot(a) - #hot(b).  Integer identities, exact."""
    rng = np.random.default_rng(7)
    nx, ny, nz = 21, 19, 13
    N = nx * ny * nz
    ea = blob(nx, ny, nz, 3.0, rng)
    eb = 0.8 * blob(nx, ny, nz, 3.0, rng)
    ef = 1.0
    hot_b = eb >= ef
    assert not (hot_b[0].any() or hot_b[-1].any() or hot_b[:, 0].any() or hot_b[:, -1].any()
                or hot_b[:, :, 0].any() or hot_b[:, :, -1].any())
    keys, rows = surface_elements(static_snap(ea), static_snap(eb), 1.0, 1.2, 0, (1.0, 1.0, 1.0), ef, geometry=1)
    assert len(np.unique(keys)) == len(keys)
    _, d, cell = decode(keys, N)
    i, j, k = cell % nx, (cell // nx) % ny, cell // (nx * ny)
    sgn = np.sign(rows[np.arange(len(keys)), 4 + d])
    assert np.all(sgn != 0)
    for axis, line_id in [(1, j + ny * k), (2, i + nx * k), (3, i + nx * j)]:
        m = d == axis
        tot = np.zeros(N)
        np.add.at(tot, line_id[m], sgn[m])
        assert np.all(tot == 0.0)
        assert m.sum() > 50
    assert sgn[d == 0].sum() == int((ea >= ef).sum()) - int(hot_b.sum())
    # periodic wrap: a hot slab touching both x edges is closed through the wrap face
    e = np.full((3, 3, 8), 0.5)
    e[:, :, :2] = 2.0
    e[:, :, -1] = 2.0
    k_o, r_o = surface_elements(static_snap(e), static_snap(e), 1.0, 1.1, 0, (1.0, 1.0, 1.0), ef, bc=(0, 0, 0))
    k_p, r_p = surface_elements(static_snap(e), static_snap(e), 1.0, 1.1, 0, (1.0, 1.0, 1.0), ef, bc=(1, 0, 0))
    assert len(k_o) == 2 * 9 and len(k_p) == 2 * 9      # outflow: faces at 1|2 and 6|7; periodic: the same two
    e[:, :, -1] = 0.5
    k_p2, r_p2 = surface_elements(static_snap(e), static_snap(e), 1.0, 1.1, 0, (1.0, 1.0, 1.0), ef, bc=(1, 0, 0))
    assert len(k_p2) == 2 * 9 and np.isclose(r_p2[:, 5].sum(), 0.0)   # now the wrap face 7|0 closes the slab


def test_gauss_theorem_on_a_ball():
    """Static ball e = e_f (2 - r/R): the faces carry the interpolated crossing positions, so sum_faces x_a dS_a
    = 3 Vol(ball) dtau up to the staircase error, and sum_faces dS_a = 0 exactly.  Halving the spacing halves the error."""
    errs = []
    for n, d in [(25, 0.2), (49, 0.1)]:
        xs = cell_centres(n, d)
        Z, Y, X = np.meshgrid(xs, xs, xs, indexing="ij")
        R = 1.83
        e = 1.0 * (2.0 - np.sqrt(X ** 2 + Y ** 2 + Z ** 2) / R)
        keys, rows = surface_elements(static_snap(e), static_snap(e), 1.0, 1.5, 0, (d, d, d), 1.0, geometry=1)
        assert np.all(decode(keys, n ** 3)[1] > 0)
        for a in (1, 2, 3):
            assert abs(rows[:, 4 + a].sum()) < 1e-12
        flux = (rows[:, 1:4] * rows[:, 5:8]).sum()
        exact = 3.0 * (4.0 / 3.0) * math.pi * R ** 3 * 0.5
        errs.append(abs(flux / exact - 1.0))
    assert errs[0] < 0.03 and errs[1] < 0.015 and errs[1] < 0.7 * errs[0], errs


def test_bjorken_uniform_cooling():
    """Ideal Bjorken flow (Eq.68): every cell crosses e_f in the same slab at tau_f = tau0 (e0/e_f)^{3/4}; the linear
    interpolation is second order in the level spacing: |tau* - tau_f| <= dt^2/8 max|e''/e'| = (7/24) dt^2 / tau_a."""
    e0, tau0, ef = 30.0, 0.6, 2.0
    tau_f = tau0 * (e0 / ef) ** 0.75
    nx, ny, nz = 4, 3, 2
    dx, dy, de = 0.3, 0.3, 0.2
    errs = []
    for dt in (0.2, 0.1, 0.05):
        found = None
        nlev = int((tau_f - tau0) / dt) + 3
        for s in range(nlev):
            ta, tb = tau0 + s * dt, tau0 + (s + 1) * dt
            ea = np.full((nz, ny, nx), e0 * (tau0 / ta) ** (4.0 / 3.0))
            eb = np.full((nz, ny, nx), e0 * (tau0 / tb) ** (4.0 / 3.0))
            keys, rows = surface_elements(static_snap(ea), static_snap(eb), ta, tb, s, (dx, dy, de), ef)
            if len(keys):
                assert found is None and ta <= tau_f <= tb
                found, bound = rows, (7.0 / 24.0) * dt * dt / ta
                assert len(keys) == nx * ny * nz and np.all(decode(keys, nx * ny * nz)[0] == s)
        assert found is not None
        np.testing.assert_allclose(found[:, 4].sum(), found[0, 0] * dx * dy * de * nx * ny * nz, rtol=1e-13)
        np.testing.assert_allclose(found[:, 11], 1.0)
        errs.append(abs(found[0, 0] - tau_f))
        assert 0.0 < errs[-1] <= bound, (dt, errs[-1], bound)
    assert errs[2] < 0.2 * errs[0], errs


def entropy(e):
    return (4.0 / 3.0) * e / T_conformal(e)


def gubser_entropy_balance(n, d, dt, flip=None):
    g = Gubser(q=1.0, eta_s=0.0)
    xs = cell_centres(n, d)
    Y, X = np.meshgrid(xs, xs, indexing="ij")
    deta, ef, tau0 = 0.1, 0.5, 1.0

    def snap(tau):
        e, u, pi = g.fields(tau, X, Y)
        return e[None], u[:, None], pi[:, None]
    a = snap(tau0)
    s_in = (entropy(a[0]) * a[1][0] * tau0 * d * d * deta)[a[0] >= ef].sum()
    s_out, s = 0.0, 0
    while True:
        ta, tb = tau0 + s * dt, tau0 + (s + 1) * dt
        b = snap(tb)
        keys, rows = surface_elements(a, b, ta, tb, s, (d, d, deta), ef)
        if flip == "space":
            rows[:, 5:8] *= -1.0
        if flip == "no_tau":
            rows[:, 5:7] /= tb
        s_out += entropy(ef) * (rows[:, 4] * rows[:, 11] + (rows[:, 5:8] * rows[:, 8:11]).sum(axis=1)).sum()
        a, s = b, s + 1
        if b[0].max() < ef:
            break
        assert s < 400
    return s_in, s_out, s


def test_gubser_entropy_flux_through_the_surface():
    """Ideal Gubser flow conserves entropy: what enters the hot region through the initial slice leaves it through the
    freeze-out surface, sum dSigma~_mu s u~^mu.  Pins the tau factors, the signs of all four face kinds and the fluid
    interpolation together: with the spatial normals flipped, or tau dropped from dSigma_x,y, the balance is off by
    tens of per cent."""
    s_in, s_out, nslab = gubser_entropy_balance(81, 0.1, 0.05)
    assert nslab > 10
    assert abs(s_out / s_in - 1.0) < 0.02, (s_in, s_out)
    s_in2, s_out2, _ = gubser_entropy_balance(41, 0.2, 0.1)
    assert abs(s_out2 / s_in2 - 1.0) < 0.05
    assert abs(gubser_entropy_balance(41, 0.2, 0.1, flip="space")[1] / s_in2 - 1.0) > 0.2
    assert abs(gubser_entropy_balance(41, 0.2, 0.1, flip="no_tau")[1] / s_in2 - 1.0) > 0.1
