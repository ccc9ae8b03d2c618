"""GPU parity of SURVEY 8(f)-3: bulk pressure Pi and net-baryon density n (Eq.28, 30, 32, 34; readings
A28-A32) -- hydro_opts.bulk_baryon through hydro_load_ext / hydro_step / hydro_read_ext against the oracle's extension
(pinned in tests/test_oracle_bulk_baryon.py) on identical seeded inputs."""
import numpy as np
import pytest

from oracle import Oracle
from paper_1802_04449_b200 import inputs
from parity_util import errors, make_oracle, pressure, small_parton_config

pytestmark = pytest.mark.gpu

ZETA_S = 0.03


def gpu(cfg, eos, **kw):
    from paper_1802_04449_b200 import from_config
    return from_config(cfg, eos, bulk_baryon=1, zeta_over_s=ZETA_S, **kw)


def ext_oracle(cfg, eos, **kw):
    o = make_oracle(cfg, eos, **kw)
    o.set_option(Oracle.OPT_EXT, 1)
    o.set_option(Oracle.OPT_ZETA_S, ZETA_S)
    return o


def ext_errors(eos, oref, gref, e_ref):
    (Po, no), (Pg, ng) = oref, gref
    w = e_ref + pressure(eos, e_ref)
    return dict(rel_Pi=float(np.max(np.abs(Pg - Po) / w)), rel_n=float(np.max(np.abs(ng - no) / np.maximum(np.abs(no), 1e-300))))


@pytest.mark.parametrize("kernel", [2, 4])
@pytest.mark.parametrize("precision", [64, 32])
def test_small_event_with_bulk_and_baryon(crossover, precision, kernel):
    """Small moving viscous event (eta/s = 0.16, zeta/s = 0.03), initial Pi = -0.2 P(T^{tau tau}) (|Pi| < P also on the
    fast dilute rim, where T^{tau tau} >> e) and n = 0.3 T^{tau tau}: one step at the 1e-10 bar, 12 steps at 1e-7 (fp64);
    fp32 relative L2 of e <= 2e-4."""
    cfg = small_parton_config(eta_over_s=0.16, moving=True)
    T, _ = inputs.ic_partons(cfg, inputs.seed_for(3))
    o = ext_oracle(cfg, crossover)
    o.load(T)
    Pi0, nb0 = -0.2 * pressure(crossover, o.read()[0]), 0.3 * T[0]      # P of the Pi-free root-find: an input recipe
    o.load_ext(T, None, Pi0, nb0)
    g = gpu(cfg, crossover, precision=precision, kernel=kernel)
    assert g.kernel() == kernel
    dt = g.np_dtype
    g.load_ext(T.astype(dt), None, Pi0.astype(dt), nb0.astype(dt))
    # the load itself: root-find with Pi
    er = errors(crossover, o.read(), g.read())
    print("load_ext", precision, er)
    if precision == 64:
        assert er["rel_e"] < 1e-10 and er["abs_u"] < 1e-10
    else:
        assert er["l2_e"] < 2e-4          # pointwise the rim cells (gamma ~ 22) amplify fp32 rounding by gamma^2
    for steps, bar in ((1, 1e-10), (11, 1e-7)):
        o.step(steps); g.step(steps)
        ref = o.read()
        er = errors(crossover, ref, g.read())
        ex = ext_errors(crossover, o.read_ext(), g.read_ext(), ref[0])
        print("bulk/baryon", precision, "steps", o.diag()["step"], er, ex)
        if precision == 64:
            assert er["rel_e"] < bar and er["rel_T"] < bar and er["rel_pi"] < 10 * bar
            assert ex["rel_Pi"] < 10 * bar and ex["rel_n"] < 10 * bar
        else:
            assert er["l2_e"] < 2e-4
    Pg, ng = g.read_ext()
    assert np.abs(Pg).max() > 1e-3 and g.diag()["nan"] == 0 and g.diag()["root_unconverged"] == 0
    # the extension is not a no-op on e: the same event without it differs
    if precision == 64:
        from paper_1802_04449_b200 import from_config
        d = from_config(cfg, crossover)
        d.load(T); d.step(12)
        assert errors(crossover, d.read(), g.read())["l2_e"] > 1e-4


def test_bjorken_cell_with_bulk(conformal):
    """0+1 D: 1x1x1 periodic cell, 150 steps, against the oracle (which is pinned by the ODE)."""
    from paper_1802_04449_b200 import Hydro
    h, n = 0.01, 150
    T = np.zeros((4, 1, 1, 1)); T[0] = 30.0
    pi = np.zeros((10, 1, 1, 1)); pi[9] = -0.9; pi[4] = pi[7] = 0.45
    Pi0, nb0 = np.full((1, 1, 1), -0.3), np.full((1, 1, 1), 0.7)
    o = Oracle(1, 1, 1, 1.0, 1.0, 1.0, h, 0.6, conformal, 0.2, bc=(1, 1, 1), pi_limit_xi=0.0)
    o.set_option(Oracle.OPT_EXT, 1); o.set_option(Oracle.OPT_ZETA_S, 0.05)
    o.load_ext(T, pi, Pi0, nb0)
    g = Hydro(1, 1, 1, 1.0, 1.0, 1.0, h, 0.6, conformal, 0.2, bc=(1, 1, 1), pi_limit_xi=0.0, bulk_baryon=1, zeta_over_s=0.05)
    g.load_ext(T, pi, Pi0, nb0)
    o.step(n); g.step(n)
    eo, _, po = o.read(); eg, _, pg = g.read()
    (Po, no), (Pg, ng) = o.read_ext(), g.read_ext()
    print("Bjorken cell with bulk", eo.ravel(), Po.ravel(), no.ravel())
    assert abs(eg.ravel()[0] / eo.ravel()[0] - 1) < 1e-11 and abs(pg[9].ravel()[0] / po[9].ravel()[0] - 1) < 1e-10
    assert abs(Pg.ravel()[0] / Po.ravel()[0] - 1) < 1e-10 and abs(ng.ravel()[0] / no.ravel()[0] - 1) < 1e-12
    assert abs(ng.ravel()[0] * g.diag()["tau"] / (0.7 * 0.6) - 1) < 1e-12          # n tau is conserved (Eq.28, S_N = 0)


def test_cartesian_box_conserves_baryon_number(crossover):
    """Periodic Cartesian box with flow, shear, bulk and baryon density: sum of n u^tau conserved to rounding on the GPU
    (flux form of Eq.28), and parity with the oracle after 4 steps."""
    e, v, pi = inputs.ic_random_smooth(37, 11, 9, seed=7, vmax=0.3)
    rng = np.random.default_rng(2)
    cfg = inputs.Config("box", 37, 11, 9, 0.2, 0.2, 0.2, 1.0, 0.02, 4, 0.1, "crossover", bc=(1, 1, 1), geometry=1)
    P = pressure(crossover, e)
    Pb = 0.3 * P * rng.uniform(-1, 1, e.shape)
    nb = 1.0 + 0.5 * rng.uniform(-1, 1, e.shape)
    g2 = 1 / (1 - (v ** 2).sum(0))
    T = np.stack([(e + P + Pb) * g2 - (P + Pb)] + [(e + P + Pb) * g2 * v[a] for a in range(3)]) + pi[:4]
    o = ext_oracle(cfg, crossover)
    o.load_ext(T, pi, Pb, nb)
    g = gpu(cfg, crossover, kernel=4)
    g.load_ext(T, pi, Pb, nb)
    N0 = (g.read_ext()[1] * g.read()[1][0]).sum()
    o.step(4); g.step(4)
    N1 = (g.read_ext()[1] * g.read()[1][0]).sum()
    assert abs(N1 / N0 - 1) < 1e-12
    ref = o.read()
    er = errors(crossover, ref, g.read())
    ex = ext_errors(crossover, o.read_ext(), g.read_ext(), ref[0])
    print("box", er, ex)
    assert er["rel_e"] < 1e-10 and er["rel_T"] < 1e-10 and ex["rel_Pi"] < 1e-10 and ex["rel_n"] < 1e-10


def test_extension_is_refused_where_it_does_not_exist(crossover):
    from paper_1802_04449_b200 import from_config
    from paper_1802_04449_b200.hydro import HydroError
    cfg = small_parton_config(eta_over_s=0.08)
    with pytest.raises(HydroError):
        from_config(cfg, crossover, bulk_baryon=1, kernel=3)
    with pytest.raises(HydroError):
        from_config(small_parton_config(eta_over_s=0.0), crossover, bulk_baryon=1)
    with pytest.raises(HydroError):
        from_config(cfg, crossover).read_ext()


def test_freezeout_finder_on_an_extended_context(crossover):
    """The freeze-out finder (8(f)-1) reads e, u~, pi~ of a 16-word context through the same read path: keys bit-exact and
    rows to 1e-8 against oracle/freezeout.py fed with the extended oracle's evolution."""
    from oracle.freezeout import surface_elements
    cfg = small_parton_config(eta_over_s=0.08, moving=True)
    T, _ = inputs.ic_partons(cfg, inputs.seed_for(3))
    nb0 = 0.3 * T[0]
    o = ext_oracle(cfg, crossover)
    o.load_ext(T, None, None, nb0)
    e_frz = 0.35 * float(o.read()[0].max())
    g = gpu(cfg, crossover)
    g.load_ext(T, None, None, nb0)
    g.freezeout_begin(e_frz, capacity=20000)
    snap = o.read()
    o.step(4); g.step(4)
    nxt = o.read()
    ok, orows = surface_elements(snap, nxt, cfg.tau0, cfg.tau0 + 4 * cfg.dtau, 0, (cfg.dx, cfg.dy, cfg.deta), e_frz)
    n, hot = g.freezeout_slab()
    keys, rows = g.freezeout_elements()
    keys, rows = keys.cpu().numpy(), rows.cpu().numpy()
    order = np.argsort(keys)
    assert n == len(ok) and np.array_equal(keys[order], ok)
    scale = np.maximum(np.abs(orows).max(axis=0), 1e-300)
    assert (np.abs(rows[order] - orows).max(axis=0) / scale).max() < 1e-8
