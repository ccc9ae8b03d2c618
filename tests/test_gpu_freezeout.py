"""GPU parity of the freeze-out surface finder (PAPER.md:268 / :640, reading A27): the elements the CUDA
library gathers during an evolution (hydro_freezeout_begin / _slab / _run through the C ABI) against oracle/freezeout.py
fed with the ORACLE's own evolution of the same seeded event.  Keys (integers) are compared exactly, rows to the hydro
parity bar amplified by the interpolation weight."""
import numpy as np
import pytest

from oracle.freezeout import surface_elements
from paper_1802_04449_b200 import inputs
from parity_util import make_oracle, small_parton_config

pytestmark = pytest.mark.gpu


def gpu(cfg, eos, **kw):
    from paper_1802_04449_b200 import from_config
    return from_config(cfg, eos, **kw)


def sorted_elements(g):
    keys, rows = g.freezeout_elements()
    keys, rows = keys.cpu().numpy(), rows.cpu().numpy()
    order = np.argsort(keys, kind="stable")
    return keys[order], rows[order]


def oracle_surface(cfg, eos, T, e_frz, steps_per_slab, nslab, **okw):
    o = make_oracle(cfg, eos, **okw)
    o.load(T)
    spacing = (cfg.dx, cfg.dy, cfg.deta)
    snap = o.read()
    keys, rows = [], []
    for s in range(nslab):
        tau_a = cfg.tau0 + (s * steps_per_slab) * cfg.dtau
        o.step(steps_per_slab)
        tau_b = cfg.tau0 + ((s + 1) * steps_per_slab) * cfg.dtau
        nxt = o.read()
        k, r = surface_elements(snap, nxt, tau_a, tau_b, s, spacing, e_frz, bc=cfg.bc, geometry=cfg.geometry)
        keys.append(k); rows.append(r)
        snap = nxt
    return np.concatenate(keys), np.concatenate(rows), snap


@pytest.mark.parametrize("kernel", [2, 4])
@pytest.mark.parametrize("eta_s", [0.0, 0.08])
def test_surface_elements_match_oracle_fp64(crossover, kernel, eta_s):
    cfg = small_parton_config(eta_over_s=eta_s, moving=True)
    T, _ = inputs.ic_partons(cfg, inputs.seed_for(3))
    steps_per_slab, nslab = 3, 4
    o0 = make_oracle(cfg, crossover)
    o0.load(T)
    e_frz = 0.35 * float(o0.read()[0].max())       # a surface well inside the event, moving inwards as it cools
    ok, orows, _ = oracle_surface(cfg, crossover, T, e_frz, steps_per_slab, nslab)
    g = gpu(cfg, crossover, kernel=kernel)
    g.load(T)
    g.freezeout_begin(e_frz, capacity=len(ok) + 1000)
    for s in range(nslab):
        g.step(steps_per_slab)
        n, hot = g.freezeout_slab()
    gk, grows = sorted_elements(g)
    print("freeze-out elements", len(ok), len(gk), "hot cells left", hot, "dirs", np.bincount((ok // cfg.cells) % 4))
    assert len(ok) > 500 and np.bincount((ok // cfg.cells) % 4, minlength=4).min() > 20     # every face kind is present
    assert np.array_equal(gk, ok)                                                           # bit-exact integer work
    scale = np.maximum(np.abs(orows).max(axis=0), 1e-300)
    err = np.abs(grows - orows).max(axis=0) / scale
    print("max column error / column scale", err)
    # the hydro states agree to ~1e-13; the weight w = (e_frz - e_a)/(e_b - e_a) amplifies that by e/|e_b - e_a| <~ 1e3
    assert err.max() < 1e-8


def test_surface_fp32_and_capacity(crossover):
    """fp32 evolution: the same surface up to the cells whose e sits within fp32 rounding of e_frz; and the capacity
    rule of the ABI (HYDRO_ENOMEM, count still exact)."""
    from paper_1802_04449_b200.hydro import HydroError
    cfg = small_parton_config(eta_over_s=0.08, moving=True)
    T, _ = inputs.ic_partons(cfg, inputs.seed_for(3))
    o0 = make_oracle(cfg, crossover)
    o0.load(T)
    e_frz = 0.35 * float(o0.read()[0].max())
    ok, orows, _ = oracle_surface(cfg, crossover, T, e_frz, 3, 3)
    g = gpu(cfg, crossover, precision=32)
    g.load(T.astype(np.float32))
    g.freezeout_begin(e_frz, capacity=len(ok) + 1000)
    for s in range(3):
        g.step(3)
        g.freezeout_slab()
    gk, grows = sorted_elements(g)
    common, io, ig = np.intersect1d(ok, gk, return_indices=True)
    print("fp32 surface: oracle", len(ok), "gpu", len(gk), "common", len(common))
    assert len(common) > 0.995 * max(len(ok), len(gk))
    pos_err = np.abs(grows[ig, :4] - orows[io, :4]).max()
    print("fp32 max position error", pos_err)
    assert pos_err < 2e-3                      # |dw| ~ 1e-6 e / |e_b - e_a| times a spacing of 0.16
    assert np.abs(grows[ig, 4:8] - orows[io, 4:8]).max() < 1e-5
    # capacity: too small an array reports ENOMEM and the exact count
    g2 = gpu(cfg, crossover)
    g2.load(T)
    g2.freezeout_begin(e_frz, capacity=10)
    g2.step(3)
    with pytest.raises(HydroError):
        g2.freezeout_slab()


def test_run_until_cold(conformal):
    """hydro_freezeout_run stops on the e_max criterion, on the configs[0] blob (cold domain edges) run
    viscous.  Properties that hold at any size: afterwards no cell is hotter than e_frz; the signed count of time-like
    faces equals the number of initially hot cells (every hot cell freezes out exactly once more often than it
    re-heats); the signed count of the faces normal to each spatial axis vanishes (the surface is closed in every
    spatial direction, because the edges stay cold)."""
    import dataclasses
    cfg = dataclasses.replace(inputs.config0(), eta_over_s=0.08)
    T, _ = inputs.ic_config0(cfg, inputs.seed_for(0))
    g = gpu(cfg, conformal)
    g.load(T)
    e0 = g.read()[0]
    e_frz = 6.0
    hot0 = e0 >= e_frz
    n_hot0 = int(hot0.sum())
    assert n_hot0 > 500 and not (hot0[0].any() or hot0[-1].any() or hot0[:, 0].any() or hot0[:, -1].any()
                                 or hot0[:, :, 0].any() or hot0[:, :, -1].any())
    g.freezeout_begin(e_frz, capacity=200000)
    n, nslab = g.freezeout_run(steps_per_slab=2, max_slabs=200)
    d = g.diag()
    print("run until cold:", n, "elements in", nslab, "slabs, e_max", d["e_max"], "tau", d["tau"], "hot at start", n_hot0)
    assert 0 < nslab < 200 and d["e_max"] < e_frz and d["step"] == 2 * nslab
    keys, rows = sorted_elements(g)
    assert len(keys) == n and len(np.unique(keys)) == n
    direction = (keys // cfg.cells) % 4
    sign = np.sign(rows[np.arange(n), 4 + direction])
    assert int(sign[direction == 0].sum()) == n_hot0
    for a in (1, 2, 3):
        assert (direction == a).sum() > 100 and int(sign[direction == a].sum()) == 0
    # u~^tau consistent with u~^i; positions inside the run's time span
    np.testing.assert_allclose(rows[:, 11], np.sqrt(1.0 + (rows[:, 8:11] ** 2).sum(axis=1)), rtol=1e-14)
    assert rows[:, 0].min() >= cfg.tau0 and rows[:, 0].max() <= d["tau"] + 1e-12
