"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times (default kernel), and the
analytic validation of configs[1]b run on the GPU.  The oracle runs whole steps here: a configs[4] step is
~35 s on 16 host cores, which is why only the first step(s) are compared (error growth over many steps is covered
by the sub-box cases of test_gpu_parity.py and by the analytic tests)."""
import numpy as np
import pytest

from paper_1802_04449_b200 import from_config, inputs
from parity_util import errors, make_oracle

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("which,steps", [("cfg2", 2), ("cfg3", 2), ("cfg4", 1)])
def test_full_size_first_steps(crossover, which, steps):
    cfg = {"cfg2": inputs.config2, "cfg3": inputs.config3, "cfg4": inputs.config4}[which]()
    idx = {"cfg2": 2, "cfg3": 3, "cfg4": 4}[which]
    T, _ = inputs.ic_partons(cfg, inputs.seed_for(idx))
    o = make_oracle(cfg, crossover)
    o.load(T)
    o.step(steps)
    ref = o.read()
    do = o.diag()
    for kernel in (2, 3, 4):                       # both production kernels, fp64
        g = from_config(cfg, crossover, kernel=kernel)
        g.load(T)
        g.step(steps)
        er = errors(crossover, ref, g.read())
        print(which, "fp64 kernel", kernel, er, g.diag())
        assert er["rel_e"] <= 1e-10 * (1 if steps == 1 else 10) and er["rel_T"] <= 1e-10 * (1 if steps == 1 else 10)
        assert er["rel_pi"] <= 1e-9 and er["l2_e"] <= 1e-13 and er["l2_T"] <= 1e-12
        dg = g.diag()
        assert np.allclose(dg["cfl"], do["cfl"], rtol=1e-9) and abs(dg["e_max"] / do["e_max"] - 1) < 1e-10
        assert dg["nan"] == 0 and dg["root_unconverged"] == 0
        del g
    for kernel in (2, 3, 4):
        g32 = from_config(cfg, crossover, precision=32, kernel=kernel)
        g32.load(T.astype(np.float32))
        g32.step(steps)
        er = errors(crossover, ref, g32.read())
        print(which, "fp32 kernel", kernel, er)
        assert er["l2_e"] <= 2e-4 and er["l2_T"] <= 2e-4 and g32.diag()["nan"] == 0
        del g32


@pytest.mark.parametrize("kernel", [2, 3, 4])
@pytest.mark.parametrize("eta_s", [0.0, 0.2])
def test_gubser_on_gpu(conformal, eta_s, kernel):
    """configs[1]b at the stated resolution (201x201x1, dx = 0.05) from tau = 1 to 1.5 on the GPU, against the
    Gubser solution (closed form for eta/s = 0, IS ODE for 0.2)."""
    from analytic_refs import Gubser
    from paper_1802_04449_b200 import Hydro
    dx, n, t1 = 0.05, 201, 1.5
    x = (np.arange(n) - (n - 1) / 2) * dx
    Y, X = np.meshgrid(x, x, indexing="ij")
    X, Y = X[None], Y[None]
    gub = Gubser(1.0, eta_s)
    h = dx / 10
    T, pi = gub.T_tau_mu(1.0, X, Y)
    g = Hydro(n, n, 1, dx, dx, 1.0, h, 1.0, conformal, eta_s, pi_limit_xi=0.0, minmod_theta=2.0, kernel=kernel)
    g.load(np.ascontiguousarray(T), np.ascontiguousarray(pi) if eta_s > 0 else None)
    g.set_history(np.ascontiguousarray(gub.fields(1.0 - h, X, Y)[1][1:]))
    g.step(int(round((t1 - 1.0) / h)))
    e, u, p = g.read()
    ea, ua, pa = gub.fields(t1, X, Y)
    m = ea > 1e-3 * ea.max()
    l2 = lambda a, b: float(np.sqrt(((a - b)[m] ** 2).sum() / (b[m] ** 2).sum()))
    vr = np.sqrt(u[1] ** 2 + u[2] ** 2) / u[0]
    vra = np.sqrt(ua[1] ** 2 + ua[2] ** 2) / ua[0]
    out = dict(e=l2(e, ea), vr=l2(vr, vra))
    if eta_s > 0:
        out.update(pixx=l2(p[4], pa[4]), pinn=l2(p[9], pa[9]))
    print("gubser on GPU", eta_s, out)
    assert out["e"] < 0.01 and out["vr"] < 0.01
    if eta_s > 0:
        assert out["pixx"] < 0.012 and out["pinn"] < 0.01
        assert np.all(np.abs(p[[3, 6, 8]]) < 1e-12) and np.all(np.abs(u[3]) < 1e-12)


@pytest.mark.parametrize("kernel", [1, 2, 3, 4])
def test_gubser_lambda1_on_gpu(conformal, kernel):
    """SURVEY 8(f)-2 on the GPU: the lambda_1 term and the free tau_pi coefficient against the paper's closed-form
    Gubser solution and against the oracle on the same grid."""
    from oracle import Oracle
    from paper_1802_04449_b200 import Hydro
    from test_oracle_gubser import gubser_lambda1_run

    def make_gpu(n, dx, h, lam, c_tau):
        return Hydro(n, n, 1, dx, dx, 1.0, h, 1.0, conformal, 0.2, pi_limit_xi=0.0, minmod_theta=2.0, kernel=kernel,
                     lambda1_hat=lam, tau_pi_coeff=c_tau)

    def make_cpu(n, dx, h, lam, c_tau):
        o = Oracle(n, n, 1, dx, dx, 1.0, h, 1.0, conformal, 0.2, pi_limit_xi=0.0, minmod_theta=2.0)
        o.set_option(Oracle.OPT_LAMBDA1_HAT, lam); o.set_option(Oracle.OPT_C_TAU, c_tau)
        return o
    f, ratio, got = gubser_lambda1_run(make_gpu, 0.1, 1.5)
    print("gubser lambda1 on GPU, kernel", kernel, f, ratio)
    assert f["e"] < 1.5e-3 and f["pixx"] < 1.5e-3 and f["pinn"] < 1.5e-3 and abs(ratio - 2.0) < 0.05
    _, _, ref = gubser_lambda1_run(make_cpu, 0.1, 1.5)
    er = errors(conformal, ref, got)
    print("   vs oracle", er)
    assert er["rel_e"] <= 1e-9 and er["rel_pi"] <= 1e-9 and er["l2_e"] <= 1e-12
