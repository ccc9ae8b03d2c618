"""Seeded synthetic inputs shared by the tests, bench.py and smoke().

This module holds NO hydrodynamics arithmetic: it only draws random numbers and
lays out initial-condition arrays (T_f^{tau mu}, pi~^{mu nu}) and the EoS table that
are then handed, as plain arrays, to the CUDA library and (in tests) to the oracle.
It stands in for the paper's Glauber/Trento/AMPT events and
lattice EoS tables, none of which exist offline; the recipes
are BASELINE.json configs[0..4] / SURVEY.md section 8(d), restated in DESIGN.md.

Arrays are numpy float64, component-major SoA [comp][nz][ny][nx], x fastest.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

HBARC = 0.1973269804          # GeV fm
C_SB = 47.5 * math.pi ** 2 / 30.0   # e = C_SB T^4 / hbarc^3, 3-flavour QGP
BASE_SEED = 18020444


@dataclass
class Config:
    name: str
    nx: int
    ny: int
    nz: int
    dx: float
    dy: float
    deta: float
    tau0: float
    dtau: float
    steps: int
    eta_over_s: float
    eos: str                      # "conformal" | "crossover"
    bc: tuple = (0, 0, 0)         # 0 outflow, 1 periodic
    geometry: int = 0             # 0 Milne, 1 Cartesian
    extra: dict = field(default_factory=dict)

    @property
    def cells(self) -> int:
        return self.nx * self.ny * self.nz


def axes(cfg: Config):
    """Cell-centre coordinates, grid centred on 0."""
    x = (np.arange(cfg.nx) - (cfg.nx - 1) / 2.0) * cfg.dx
    y = (np.arange(cfg.ny) - (cfg.ny - 1) / 2.0) * cfg.dy
    z = (np.arange(cfg.nz) - (cfg.nz - 1) / 2.0) * cfg.deta
    return x, y, z


def config0(scale: int = 1) -> Config:
    return Config("cfg0", 33, 33, 17, 0.3, 0.3, 0.3, 0.6, 0.03, 40, 0.0, "conformal")


def config2(nx=201, ny=201, nz=105, steps=400, eta_over_s=0.08) -> Config:
    return Config("cfg2", nx, ny, nz, 0.16, 0.16, 0.16, 0.4, 0.016, steps, eta_over_s,
                  "crossover", extra={"partons": 3000, "moving": False})


def config3(nx=201, ny=201, nz=105, steps=400, eta_over_s=0.08) -> Config:
    return Config("cfg3", nx, ny, nz, 0.16, 0.16, 0.16, 0.4, 0.016, steps, eta_over_s,
                  "crossover", extra={"partons": 3000, "moving": True})


def config4(nx=301, ny=301, nz=201, steps=200, eta_over_s=0.16) -> Config:
    return Config("cfg4", nx, ny, nz, 0.1, 0.1, 0.08, 0.4, 0.01, steps, eta_over_s,
                  "crossover", extra={"partons": 8000, "moving": True})


def ic_config0(cfg: Config, seed: int = BASE_SEED) -> tuple[np.ndarray, None]:
    """BASELINE.json configs[0]: smooth Gaussian + 3 seeded hotspots, static, pi = 0."""
    rng = np.random.default_rng(seed)
    x, y, z = axes(cfg)
    Z, Y, X = np.meshgrid(z, y, x, indexing="ij")
    e = 30.0 * np.exp(-(X ** 2 + Y ** 2) / (2 * 1.5 ** 2) - Z ** 2 / (2 * 1.0 ** 2))
    for _ in range(3):
        A = rng.uniform(5.0, 15.0)
        x0 = rng.uniform(-3.0, 3.0)
        y0 = rng.uniform(-3.0, 3.0)
        z0 = rng.uniform(-1.0, 1.0)
        e += A * np.exp(-((X - x0) ** 2 + (Y - y0) ** 2) / (2 * 0.5 ** 2)
                        - (Z - z0) ** 2 / (2 * 0.5 ** 2))
    e = np.maximum(e, 1e-6)
    T = np.zeros((4,) + e.shape)
    T[0] = e
    return T, None


def _gauss_window(centre, sigma, coords, d, nsig=6.0):
    """Unit-integral 1D Gaussian sampled at cell centres inside +-nsig*sigma."""
    n = coords.shape[0]
    lo = int(np.searchsorted(coords, centre - nsig * sigma, side="left"))
    hi = int(np.searchsorted(coords, centre + nsig * sigma, side="right"))
    lo, hi = max(lo, 0), min(hi, n)
    if hi <= lo:
        return lo, lo, np.zeros(0)
    g = np.exp(-(coords[lo:hi] - centre) ** 2 / (2 * sigma ** 2)) / (math.sqrt(2 * math.pi) * sigma)
    return lo, hi, g


def ic_partons(cfg: Config, seed: int = BASE_SEED + 20) -> tuple[np.ndarray, None]:
    """BASELINE.json configs[2]/[3]/[4]: seeded parton deposits (stand-in for AMPT).

    Draw order per run: all x, all y, all eta, all E, then (moving only) all pT, all phi.
    Each parton deposits K = Gx*Gy*Geta/tau0 (unit-integral Gaussians, sigma 0.6, cut at 6 sigma):
      T^{tau tau} += p^tau K, with p^tau = E (static) or sqrt(E^2 + pT^2) (moving),
      T^{tau x} += pT cos(phi) K, T^{tau y} += pT sin(phi) K, T^{tau eta} = 0.
    Floor on T^{tau tau}: 1e-6.  pi = 0.
    """
    n = int(cfg.extra["partons"])
    moving = bool(cfg.extra["moving"])
    rng = np.random.default_rng(seed)
    px = rng.normal(0.0, 3.0, n)
    py = rng.normal(0.0, 3.0 * 0.7, n)
    pz = rng.uniform(-5.0, 5.0, n)
    E = rng.exponential(1.0, n)
    if moving:
        pT = rng.exponential(0.5, n)
        phi = rng.uniform(0.0, 2 * math.pi, n)
    else:
        pT = np.zeros(n)
        phi = np.zeros(n)
    x, y, z = axes(cfg)
    T = np.zeros((4, cfg.nz, cfg.ny, cfg.nx))
    sr, sz = 0.6, 0.6
    # windowed 1D profiles of every parton, then one (ny x n_sel) @ (n_sel x nx) product per eta plane
    Gx = np.zeros((n, cfg.nx)); Gy = np.zeros((n, cfg.ny)); Gz = np.zeros((n, cfg.nz))
    for p in range(n):
        x0, x1, gx = _gauss_window(px[p], sr, x, cfg.dx)
        y0, y1, gy = _gauss_window(py[p], sr, y, cfg.dy)
        z0, z1, gz = _gauss_window(pz[p], sz, z, cfg.deta)
        Gx[p, x0:x1] = gx; Gy[p, y0:y1] = gy; Gz[p, z0:z1] = gz / cfg.tau0
    ptau = np.sqrt(E ** 2 + pT ** 2)
    wts = [ptau, pT * np.cos(phi), pT * np.sin(phi)] if moving else [ptau]
    for k in range(cfg.nz):
        sel = np.nonzero(Gz[:, k])[0]
        if sel.size == 0:
            continue
        gxs, gys, gzs = Gx[sel], Gy[sel], Gz[sel, k]
        for m, w in enumerate(wts):
            T[m, k] = (gys * (w[sel] * gzs)[:, None]).T @ gxs
    np.maximum(T[0], 1e-6, out=T[0])
    return T, None


def ic_random_smooth(nx, ny, nz, seed, vmax=0.3, with_pi=True):
    """Random smooth periodic fields for conservation / brute-force tests:
    a few low Fourier modes for e>0, v_i, and (optionally) small pi components.
    Returns primitives e, v[3] and raw pi[10] (NOT projected; the scheme evolves all ten
    components independently)."""
    rng = np.random.default_rng(seed)
    k = np.arange(nz)[:, None, None] * 2 * math.pi / nz
    j = np.arange(ny)[None, :, None] * 2 * math.pi / ny
    i = np.arange(nx)[None, None, :] * 2 * math.pi / nx

    def mode():
        a = rng.uniform(-1, 1, 4)
        ph = rng.uniform(0, 2 * math.pi, 3)
        return (a[0] * np.sin(i + ph[0]) + a[1] * np.sin(j + ph[1]) + a[2] * np.sin(k + ph[2])
                + a[3] * np.sin(i + j + k)) / 4.0 + np.zeros((nz, ny, nx))

    e = 5.0 * (1.5 + mode())
    v = np.stack([vmax * mode() for _ in range(3)])
    pi = np.stack([(0.05 * mode() * e if with_pi else np.zeros_like(e)) for _ in range(10)])
    return e, v, pi


# ----------------------------------------------------------------------------------------
# Synthetic crossover EoS table (BASELINE.json configs[2]; stands in for lattice tables).
# c_s^2(e) = 1/3 - 0.2 exp(-ln^2(e/a)), a = 0.6 GeV/fm^3; P = int_0^e c_s^2 de' (closed form);
# T from dT/T = c_s^2 de/(e+P), normalised to Stefan-Boltzmann at e = 1e3.
# This is input generation (a table handed to hydro_create / the oracle), not method arithmetic.
# ----------------------------------------------------------------------------------------
EOS_A = 0.6


def crossover_cs2(e):
    e = np.asarray(e, dtype=np.float64)
    return 1.0 / 3.0 - 0.2 * np.exp(-np.log(e / EOS_A) ** 2)


def crossover_pressure(e):
    from scipy.special import erf
    e = np.asarray(e, dtype=np.float64)
    return e / 3.0 - 0.2 * EOS_A * math.exp(0.25) * (math.sqrt(math.pi) / 2.0) * (
        erf(np.log(e / EOS_A) - 0.5) + 1.0)


def crossover_table(n: int = 2000, e_min: float = 1e-4, e_max: float = 1e3):
    """Returns dict(kind=1, n, e_min, e_max, P[n], T[n], c_sb) with log-spaced nodes
    e_k = e_min (e_max/e_min)^{k/(n-1)}."""
    k = np.arange(n)
    e = e_min * (e_max / e_min) ** (k / (n - 1.0))
    P = crossover_pressure(e)
    # ln T(e) = ln T(e_max) - int_e^{e_max} c_s^2/(e'+P) de', composite Simpson in ln e on a
    # 16x refined grid (smooth integrand; error << 1e-12).
    sub = 16
    m = (n - 1) * sub + 1
    le = np.linspace(math.log(e_min), math.log(e_max), m)
    ef = np.exp(le)
    f = crossover_cs2(ef) * ef / (ef + crossover_pressure(ef))     # d ln T / d ln e
    h = le[1] - le[0]
    # cumulative Simpson over pairs of sub-intervals
    seg = (f[0:-2:2] + 4 * f[1:-1:2] + f[2::2]) * h / 3.0
    cum = np.concatenate([[0.0], np.cumsum(seg)])                  # at even fine nodes
    lnT_rel = cum[:: sub // 2]                                      # at table nodes
    T_max = HBARC * (e_max / (C_SB * HBARC)) ** 0.25
    lnT = math.log(T_max) + (lnT_rel - lnT_rel[-1])
    return dict(kind=1, n=n, e_min=e_min, e_max=e_max, P=P.copy(), T=np.exp(lnT), c_sb=C_SB)


def conformal_eos():
    return dict(kind=0, n=0, e_min=0.0, e_max=0.0, P=None, T=None, c_sb=C_SB)


def eos_for(cfg: Config):
    return conformal_eos() if cfg.eos == "conformal" else crossover_table()


def seed_for(cfg_index: int, variant: int = 0) -> int:
    return BASE_SEED + 10 * cfg_index + variant
