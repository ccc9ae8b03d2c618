"""CPU ORACLE -- TEST INFRASTRUCTURE ONLY: freeze-out hypersurface elements between two stored time levels.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may import this module; the product never does.

What it computes.  The paper states WHAT the surface is -- "d Sigma_mu is a freeze-out hyper-surface
element determined by the constant freeze-out temperature T_f or constant freeze-out energy density e_f"
(text under Eq.55) -- and that the finder runs on the GPU next to the e_max reduction that stops the
evolution, but not HOW it is found (it cites its Ref.[64]).  Reading A27: the cuboidal
surface.  Every grid point of every stored time level owns the 4-D cell centred on it; a point is HOT when
e >= e_frz.  The surface is the set of faces between a hot and a cold 4-D cell:

  dir 0 (time-like face)  cell c is hot at level a and cold at level b, or the reverse:
        w = (e_frz - e_a)/(e_b - e_a),  tau* = tau_a + w dtau_out,  position (tau*, x_c, y_c, eta_c)
        dSigma~ = s (tau* dx dy deta, 0, 0, 0),   s = +1 if hot at level a (the normal points to the cold side)
        fluid: u~^i and pi~^{mu nu} interpolated linearly in time with weight w; u~^tau = sqrt(1 + u~.u~)
  dir 1,2,3 (faces normal to x, y, eta_s, taken at level b)  cells c and c + e_a differ at level b:
        w = (e_frz - e_b(c))/(e_b(c+e_a) - e_b(c)),  position = cell centre + w * spacing along the axis, time tau_b
        dSigma~_x = s tau_b dtau_out dy deta,  dSigma~_y = s tau_b dtau_out dx deta,  dSigma~_eta = s dtau_out dx dy
        (tilde components, Eq.22: d~_eta = d_eta / tau, so the eta component carries no tau),
        s = +1 if c is hot;  fluid interpolated linearly between the two cells with weight w.
  Cartesian geometry: tau -> 1 in every area.  Outflow axes have no face across the domain edge; periodic axes wrap.

Each element carries the integer key  ((slab * 4 + dir) * N + cell)  (cell = linear index of c, x fastest), which
is unique, so two implementations can be compared after sorting by key.  Element row (22 words):
  tau, x, y, eta, dS_tau, dS_x, dS_y, dS_eta, u~^x, u~^y, u~^eta, u~^tau is NOT stored (derived), pi~[10], e_frz-side
  flag is not stored: [0:4] position, [4:8] dSigma~_mu (covariant), [8:11] u~^i, [11] u~^tau, [12:22] pi~.

Pins (tests/test_oracle_freezeout.py): uniform Bjorken cooling (count, tau*, total volume), closedness of the
face set (integer sums), Gauss's theorem on a static ball with interpolated positions, entropy flux through the
surface of analytic ideal Gubser flow against the initial entropy of the hot region.
"""
from __future__ import annotations

import numpy as np

NWORDS = 22


def cell_centres(n, d):
    """Cell-centre coordinates of an axis with n cells of size d, centred on 0 (inputs.py uses the same rule)."""
    return (np.arange(n) - 0.5 * (n - 1)) * d


def surface_elements(snap_a, snap_b, tau_a, tau_b, slab, spacing, e_frz, bc=(0, 0, 0), geometry=0):
    """snap_x = (e [nz,ny,nx], u [4,nz,ny,nx], pi [10,nz,ny,nx]) at the two levels.  Returns (keys int64 [M],
    rows float64 [M, 22]) sorted by key."""
    ea, ua, pa = [np.asarray(x, dtype=np.float64) for x in snap_a]
    eb, ub, pb = [np.asarray(x, dtype=np.float64) for x in snap_b]
    nz, ny, nx = ea.shape
    N = nx * ny * nz
    dx, dy, de = spacing
    dt = tau_b - tau_a
    xs, ys, zs = cell_centres(nx, dx), cell_centres(ny, dy), cell_centres(nz, de)
    hot_a, hot_b = ea >= e_frz, eb >= e_frz
    keys, rows = [], []

    def emit(direction, k, j, i, pos, dS, ui, pi):
        row = np.zeros(NWORDS)
        row[0:4] = pos
        row[4:8] = dS
        row[8:11] = ui
        row[11] = np.sqrt(1.0 + ui[0] ** 2 + ui[1] ** 2 + ui[2] ** 2)
        row[12:22] = pi
        keys.append((slab * 4 + direction) * N + (k * ny + j) * nx + i)
        rows.append(row)

    for k in range(nz):
        for j in range(ny):
            for i in range(nx):
                # time-like face of cell (i,j,k)
                if hot_a[k, j, i] != hot_b[k, j, i]:
                    w = (e_frz - ea[k, j, i]) / (eb[k, j, i] - ea[k, j, i])
                    ts = tau_a + w * dt
                    s = 1.0 if hot_a[k, j, i] else -1.0
                    tf = ts if geometry == 0 else 1.0
                    ui = (1.0 - w) * ua[1:, k, j, i] + w * ub[1:, k, j, i]
                    pi = (1.0 - w) * pa[:, k, j, i] + w * pb[:, k, j, i]
                    emit(0, k, j, i, (ts, xs[i], ys[j], zs[k]), (s * tf * dx * dy * de, 0.0, 0.0, 0.0), ui, pi)
                # faces normal to x, y, eta_s at level b, between this cell and its upper neighbour
                for axis in range(3):
                    n_ax = (nx, ny, nz)[axis]
                    c_ax = (i, j, k)[axis]
                    up = c_ax + 1
                    if up >= n_ax:
                        if not bc[axis] or n_ax < 2:
                            continue
                        up = 0
                    i2, j2, k2 = (up, j, k) if axis == 0 else ((i, up, k) if axis == 1 else (i, j, up))
                    if hot_b[k, j, i] == hot_b[k2, j2, i2]:
                        continue
                    w = (e_frz - eb[k, j, i]) / (eb[k2, j2, i2] - eb[k, j, i])
                    s = 1.0 if hot_b[k, j, i] else -1.0
                    tf = tau_b if geometry == 0 else 1.0
                    pos = [tau_b, xs[i], ys[j], zs[k]]
                    pos[1 + axis] += w * spacing[axis]
                    dS = [0.0, 0.0, 0.0, 0.0]
                    if axis == 0:
                        dS[1] = s * tf * dt * dy * de
                    elif axis == 1:
                        dS[2] = s * tf * dt * dx * de
                    else:
                        dS[3] = s * dt * dx * dy
                    ui = (1.0 - w) * ub[1:, k, j, i] + w * ub[1:, k2, j2, i2]
                    pi = (1.0 - w) * pb[:, k, j, i] + w * pb[:, k2, j2, i2]
                    emit(1 + axis, k, j, i, pos, dS, ui, pi)
    if not keys:
        return np.zeros(0, dtype=np.int64), np.zeros((0, NWORDS))
    keys = np.asarray(keys, dtype=np.int64)
    rows = np.asarray(rows)
    order = np.argsort(keys, kind="stable")
    return keys[order], rows[order]
