"""Long-run evidence on the GPU: full-length stability of BASELINE.json configs[2], [3], [4],
oracle-vs-CUDA drift over 100 steps on a 96x96x64 sub-box, and configs[1]a (Bjorken) on the GPU to tau = 10.

The drift figures asserted for the moving-parton event are MEASURED values with a stated margin: on the clamped rim
(gamma at the v_max limit) two correct roundings of the same algorithm diverge, which the test shows by building the
oracle a second time with FMA contraction (-ffp-contract=fast) and comparing oracle with oracle."""
import os
import tempfile

import numpy as np
import pytest

from paper_1802_04449_b200 import from_config, inputs
from parity_util import errors, make_oracle

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("kernel", [2, 3, 4])
@pytest.mark.parametrize("which,precision", [("cfg2", 64), ("cfg2", 32), ("cfg3", 64), ("cfg3", 32), ("cfg4", 64),
                                             ("cfg4", 32)])
def test_full_length_stability(crossover, which, precision, kernel):
    """configs[2], [3]: 400 steps; configs[4]: 200 steps; no NaN, converged root-find, falling e_max, CFL sum < 1."""
    cfg = {"cfg2": inputs.config2, "cfg3": inputs.config3, "cfg4": inputs.config4}[which]()
    idx = {"cfg2": 2, "cfg3": 3, "cfg4": 4}[which]
    T, _ = inputs.ic_partons(cfg, inputs.seed_for(idx))
    g = from_config(cfg, crossover, precision=precision, kernel=kernel)
    g.load(T.astype(g.np_dtype))
    emax, chunk = [g.diag()["e_max"]], 25
    for s in range(0, cfg.steps, chunk):
        g.step(chunk)
        d = g.diag()
        emax.append(d["e_max"])
        assert d["nan"] == 0 and d["root_unconverged"] == 0, (s, d)
        assert sum(d["cfl"]) < 1.0, d
        assert np.isfinite(d["e_max"])
    print(which, precision, "e_max", ["%.4g" % v for v in emax], d)
    assert d["step"] == cfg.steps
    # Bjorken-like dilution: e_max falls monotonically once the first chunk is over -- down to the scale of the isolated
    # rim spikes.  On the clamped rim single dilute cells jump to e ~ 0.3-0.6 GeV/fm^3 for a few steps in EVERY
    # implementation, the oracle included (measured on the 96x96x64 sub-box: at step 125 the oracle holds a cell at 0.51
    # where its own FMA-contracted build and both CUDA kernels hold 0.03-0.06; test_moving_event_drift_is_rounding_chaos),
    # so once the core has diluted below ~1 GeV/fm^3 the maximum may sit on such a cell.
    assert all(b <= max(a * (1 + 1e-6), 1.0) for a, b in zip(emax[1:], emax[2:])), emax
    assert emax[-1] < 0.5 * emax[0] and max(emax[2:]) <= emax[1]
    e, u, p = g.read()
    assert np.isfinite(e).all() and np.isfinite(u).all() and np.isfinite(p).all()
    assert e.min() >= 1e-7 * (1 - 1e-6) and u[0].max() <= 22.4 * (1 + 1e-3)       # floor (A8) and v_max clamp (A7)


def sub_box(moving, eta_s=0.08):
    cfg = (inputs.config3 if moving else inputs.config2)(nx=96, ny=96, nz=64, steps=100, eta_over_s=eta_s)
    cfg.extra = {"partons": 600, "moving": moving}
    return cfg


def test_static_event_100_steps(crossover):
    """96x96x64 sub-box of configs[2] (static partons, eta/s = 0.08): the v_max clamp never fires, and the CUDA path
    stays within the north_star bars of the oracle for 100 steps (fp64 1e-7 pointwise; fp32 L2 2e-4)."""
    cfg = sub_box(False)
    T, _ = inputs.ic_partons(cfg, inputs.seed_for(2))
    o = make_oracle(cfg, crossover); o.load(T)
    gs = {(k, pr): from_config(cfg, crossover, precision=pr, kernel=k) for k in (2, 3, 4) for pr in (64, 32)}
    for g in gs.values():
        g.load(T.astype(g.np_dtype))
    for s in (25, 50, 100):
        n = s - o.diag()["step"]
        o.step(n)
        ref = o.read()
        for (k, pr), g in gs.items():
            g.step(n)
            er = errors(crossover, ref, g.read())
            print("static", s, "kernel", k, "fp", pr, er)
            if pr == 64:
                assert er["rel_e"] <= 1e-7 and er["rel_T"] <= 1e-7 and er["l2_e"] <= 1e-12
            else:
                assert er["l2_e"] <= 2e-4 and er["l2_T"] <= 2e-4
    assert o.diag()["clamped"] == 0 and all(g.diag()["clamped"] == 0 for g in gs.values())


@pytest.mark.parametrize("kernel", [2, 3, 4])
def test_moving_event_drift_is_rounding_chaos(crossover, kernel):
    """96x96x64 sub-box of configs[3] (moving partons, eta/s = 0.08).  The rim is clamped to gamma = 22.4 within 25
    steps; from then on ANY two roundings of the algorithm drift apart.  Measured (B200, round 2), L2(e) over
    e > 1e-3 max e:   steps   CUDA fp64 vs oracle   oracle(FMA) vs oracle   CUDA fp32 vs oracle   clamp events
                         5         6.8e-16               2.3e-16              2.6e-07              811
                        25         7.6e-07               2.1e-05              8.4e-05            9 279
                        50         3.1e-04               7.9e-04              1.2e-03           16 578
                       100         2.8e-03               3.1e-03              6.8e-03           19 605
    Asserted: the CUDA drift stays within 10x of the oracle-vs-oracle drift at every checkpoint (and below 2e-2),
    and the two are equal to rounding (1e-12) up to the first clamp."""
    cfg = sub_box(True)
    T, _ = inputs.ic_partons(cfg, inputs.seed_for(3))
    import oracle as oracle_mod
    with tempfile.TemporaryDirectory() as tmp:
        fma = oracle_mod.build_variant(os.path.join(tmp, "liboracle_fma.so"), ["-ffp-contract=fast", "-march=native"])
        o = make_oracle(cfg, crossover); o.load(T)
        of = make_oracle(cfg, crossover, lib=fma); of.load(T)
        g = from_config(cfg, crossover, kernel=kernel); g.load(T)
        g32 = from_config(cfg, crossover, precision=32, kernel=kernel); g32.load(T.astype(np.float32))
        rows = []
        for s in (5, 25, 50, 100):
            n = s - o.diag()["step"]
            o.step(n); of.step(n); g.step(n); g32.step(n)
            ref = o.read()
            a, b, c = errors(crossover, ref, g.read()), errors(crossover, ref, of.read()), errors(crossover, ref, g32.read())
            rows.append((s, a["l2_e"], b["l2_e"], c["l2_e"], o.diag()["clamped"], g.diag()["clamped"]))
            print("moving step %d: L2(e) cuda64 %.2e  oracle_fma %.2e  cuda32 %.2e  clamped oracle %d cuda %d" % rows[-1])
        del of
    s5 = rows[0]
    assert s5[1] < 1e-12                                           # before the rim is clamped: rounding level
    for s, cuda, fma_drift, cuda32, nco, ncg in rows[1:]:
        assert nco > 0
        assert cuda < 2e-2 and cuda < 10 * max(fma_drift, 1e-9), rows
        assert cuda32 < 2e-2
        assert abs(ncg - nco) <= 0.05 * nco + 10


@pytest.mark.parametrize("kernel", [2, 3, 4])
@pytest.mark.parametrize("eta_s", [0.0, 0.08, 0.2])
def test_bjorken_on_gpu_to_tau10(conformal, eta_s, kernel):
    """configs[1]a on the GPU: 1x1x1 periodic cell, e(0.6) = 30, tau 0.6 -> 10 with h = 0.01 (940 steps), against the
    oracle (same steps) and the closed form / IS ODE (Eq.68)."""
    from analytic_refs import bjorken_is, bjorken_w_ns
    from oracle import Oracle
    from paper_1802_04449_b200 import Hydro
    h, n = 0.01, 940
    T = np.zeros((4, 1, 1, 1)); T[0] = 30.0
    pi = None
    if eta_s > 0:
        w0 = bjorken_w_ns(30.0, 0.6, eta_s)
        pi = np.zeros((10, 1, 1, 1)); pi[9] = w0; pi[4] = pi[7] = -w0 / 2
    o = Oracle(1, 1, 1, 1.0, 1.0, 1.0, h, 0.6, conformal, eta_s, bc=(1, 1, 1), pi_limit_xi=0.0)
    g = Hydro(1, 1, 1, 1.0, 1.0, 1.0, h, 0.6, conformal, eta_s, bc=(1, 1, 1), pi_limit_xi=0.0, kernel=kernel)
    o.load(T, pi); g.load(T, pi)
    o.step(n); g.step(n)
    er = errors(conformal, o.read(), g.read())
    e = g.read()[0].item()
    tau = g.diag()["tau"]
    assert abs(tau - 10.0) < 1e-9
    print("bjorken to tau=10", eta_s, er, e)
    assert er["rel_e"] <= 1e-10 and er["rel_pi"] <= 1e-10
    if eta_s == 0:
        assert abs(e * tau ** (4 / 3) / (30.0 * 0.6 ** (4 / 3)) - 1) < 1e-5      # Heun drift at h = 0.01: 6.9e-6
    else:
        ref = bjorken_is(30.0, 0.6, 10.0, eta_s)(10.0)
        assert abs(e / ref[0] - 1) < 1e-5 and abs(g.read()[2][9].item() / ref[1] - 1) < 1e-4
