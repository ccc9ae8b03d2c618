"""Helpers of the GPU-vs-oracle parity tests (comparison only; no method arithmetic is shared with
either side: the frame tensor below is the definition PAPER.md:50 (Eq.1) applied to BOTH outputs)."""
import numpy as np

from oracle import Oracle
from paper_1802_04449_b200 import inputs


def pressure(eos, e):
    """P(e) by the table rule of DESIGN.md A16, vectorised (used only to form T^{tau mu} for comparison)."""
    if eos["kind"] == 0:
        return e / 3.0
    n = eos["n"]
    nodes = eos["e_min"] * (eos["e_max"] / eos["e_min"]) ** (np.arange(n) / (n - 1.0))
    P = np.interp(e, nodes, eos["P"])
    P = np.where(e <= eos["e_min"], eos["P"][0] * e / eos["e_min"], P)
    P = np.where(e >= eos["e_max"], eos["P"][-1] + (e - eos["e_max"]) / 3.0, P)
    return P


def T_tau_mu(eos, e, u, pi):
    """T_f^{tau mu} = (e+P) u^tau u^mu - P g^{tau mu} + pi^{tau mu}."""
    P = pressure(eos, e)
    T = np.stack([(e + P) * u[0] * u[0] - P, (e + P) * u[0] * u[1], (e + P) * u[0] * u[2], (e + P) * u[0] * u[3]])
    return T + pi[:4]


def make_oracle(cfg, eos, **kw):
    return Oracle(cfg.nx, cfg.ny, cfg.nz, cfg.dx, cfg.dy, cfg.deta, cfg.dtau, cfg.tau0, eos, cfg.eta_over_s,
                  bc=cfg.bc, geometry=cfg.geometry, **kw)


def errors(eos, ref, got):
    """ref, got: (e, u, pi) triples of float64 arrays.  Returns the parity figures used in the tests:
    rel_e   max_c |de| / e_ref                         (pointwise)
    rel_T   max_c,mu |dT^{tau mu}| / T^{tau tau}_ref   (pointwise, normalised by the local energy density)
    abs_u   max |du~^i| / u~^tau_ref
    rel_pi  max_c,m |dpi_m| / (e+P)_ref                (pointwise, enthalpy-normalised)
    l2_e    relative L2 of e over cells with e > 1e-3 max e (the fp32 figure of north_star)
    """
    e0, u0, p0 = [np.asarray(a, dtype=np.float64) for a in ref]
    e1, u1, p1 = [np.asarray(a, dtype=np.float64) for a in got]
    T0, T1 = T_tau_mu(eos, e0, u0, p0), T_tau_mu(eos, e1, u1, p1)
    m = e0 > 1e-3 * e0.max()
    return dict(
        rel_e=float(np.max(np.abs(e1 - e0) / e0)),
        rel_T=float(np.max(np.abs(T1 - T0) / T0[0])),
        abs_u=float(np.max(np.abs(u1[1:] - u0[1:]) / u0[0])),
        rel_pi=float(np.max(np.abs(p1 - p0) / (e0 + pressure(eos, e0)))),
        l2_e=float(np.sqrt(((e1 - e0)[m] ** 2).sum() / (e0[m] ** 2).sum())),
        l2_T=float(np.sqrt((((T1 - T0)[:, m]) ** 2).sum() / ((T0[:, m]) ** 2).sum())),
    )


def small_parton_config(nx=40, ny=36, nz=24, eta_over_s=0.08, moving=True, partons=60, steps=5):
    """A cut-down configs[2]/[3] event: same sampler, EoS and spacings, fewer cells and partons.
    Spans several 32x8 thread tiles plus a ragged tail in x and y."""
    cfg = inputs.Config("small", nx, ny, nz, 0.16, 0.16, 0.16, 0.4, 0.016, steps, eta_over_s, "crossover",
                        extra={"partons": partons, "moving": moving})
    return cfg


def squeeze_partons(cfg, seed):
    """ic_partons with the sampler's widths scaled to the small box (positions only; the draw order and
    the deposit rule are inputs.ic_partons')."""
    T, _ = inputs.ic_partons(cfg, seed)
    return T
