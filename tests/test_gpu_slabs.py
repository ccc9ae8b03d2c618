"""eta_s-slab decomposition on the GPU: one event split into slabs with two ghost planes per
interior side, stepped stage by stage with a ghost-plane exchange after each stage (hydro_stage / hydro_planes through
the C ABI), against the undivided grid.  The slabs run one after the other in ONE process on one GPU (no kernel waits
on another); the arithmetic of an interior cell is the same in both runs, so the results must be IDENTICAL, not close."""
import numpy as np
import pytest

from paper_1802_04449_b200 import inputs, slabs
from parity_util import small_parton_config

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("kernel", [2, 4])
@pytest.mark.parametrize("nslab,periodic", [(3, False), (2, True), (4, True)])
def test_slabs_reproduce_the_undivided_grid_bit_for_bit(crossover, kernel, nslab, periodic):
    import dataclasses
    from paper_1802_04449_b200 import from_config
    cfg = small_parton_config(eta_over_s=0.16, moving=True)
    if periodic:
        cfg = dataclasses.replace(cfg, bc=(0, 0, 1))
    T, _ = inputs.ic_partons(cfg, inputs.seed_for(3))
    steps = 6
    whole = from_config(cfg, crossover, kernel=kernel)
    whole.load(T)
    whole.step(steps)
    e0, u0, p0 = whole.read()
    parts = [slabs.Slab(cfg, crossover, r, nslab, kernel=kernel) for r in range(nslab)]
    for s in parts:
        s.load(T)
    slabs.step_local(parts, steps)
    pieces = [s.read_interior() for s in parts]
    e1 = np.concatenate([p[0] for p in pieces], axis=0)
    u1 = np.concatenate([p[1] for p in pieces], axis=1)
    p1 = np.concatenate([p[2] for p in pieces], axis=1)
    assert e1.shape == e0.shape
    print("slabs", nslab, "periodic", periodic, "kernel", kernel, "max |de|", np.abs(e1 - e0).max(), "max |dpi|",
          np.abs(p1 - p0).max())
    assert np.array_equal(e1, e0) and np.array_equal(u1, u0) and np.array_equal(p1, p0)
    for s in parts:
        d = s.h.diag()
        assert d["step"] == steps and d["nan"] == 0


def test_stage_order_is_enforced(crossover):
    from paper_1802_04449_b200 import from_config
    from paper_1802_04449_b200.hydro import HydroError
    cfg = small_parton_config(eta_over_s=0.08)
    T, _ = inputs.ic_partons(cfg, inputs.seed_for(3))
    g = from_config(cfg, crossover)
    g.load(T)
    with pytest.raises(HydroError):
        g.stage(2)                     # stage 2 before stage 1
    g.stage(1)
    with pytest.raises(HydroError):
        g.step(1)                      # a whole step in the middle of one
    g.stage(2)
    assert g.diag()["step"] == 1
    ref = from_config(cfg, crossover)
    ref.load(T); ref.step(1)
    assert np.array_equal(g.read()[0], ref.read()[0])          # stage(1); stage(2) is step(1)
    with pytest.raises(HydroError):
        from_config(cfg, crossover, kernel=3).stage(1)         # the ghosted store of kernel 3 has no plane interface
