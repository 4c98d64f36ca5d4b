"""-m gpu: the HOST-buffer entry point of the whole block step (nbody_step_host, what bench.py's e2e leg times)
gives bit-identical results to the device-pointer calls driven by the scheduler, and matches the oracle's step."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_1312_1789_b200 import workloads as W
import gpu_util as U


@pytest.mark.parametrize("order", [4, 6, 8])
def test_step_host_equals_device_path_and_oracle(order):
    import torch
    from oracle import integrate as OI
    from paper_1312_1789_b200 import nbody
    from paper_1312_1789_b200.scheduler import Integrator
    c = W.cluster(5, 777)
    eps2 = 1e-6
    crit = 4 if order >= 6 else 0
    so = OI.bootstrap(c["m"], c["x"], c["v"], order, eps2)
    # a few oracle blocks first so that t, dt are a genuine mix of levels
    for _ in range(5):
        OI.block_step(so, eps2, 0.1, 2.0**-30, 2.0**-4, crit_order=crit)
    g = Integrator(c["m"], c["x"], c["v"], order, eps2, dt_criterion_order=crit)
    for k in range(8):
        g.D[k].copy_(U.dev(so.D[k]))
    for dst, src in ((g.t, so.t), (g.dt, so.dt), (g.x, so.x), (g.v, so.v), (g.pot, so.pot)):
        dst.copy_(U.dev(src))
    # host-side copy of the same state
    h = dict(t=so.t.copy(), dt=so.dt.copy(), x=so.x.copy(), v=so.v.copy(), D=[d.copy() for d in so.D], pot=so.pot.copy())
    ctx = nbody.Context(so.n)
    ctx.set_option("dt_criterion_order", crit)
    for blk in range(3):
        tn_h, na_h, up, down = ctx.step_host(so.n, order, eps2, 0.1, 2.0**-30, 2.0**-4, h["t"], h["dt"], so.m, h["x"],
                                             h["v"], h["D"], h["pot"])
        tn_g, na_g = g.block_step()
        h_old = so.dt.copy()
        tn_o, idx_o = OI.block_step(so, eps2, 0.1, 2.0**-30, 2.0**-4, crit_order=crit)
        torch.cuda.synchronize()
        assert (tn_h, na_h) == (tn_g, na_g)
        assert up == 8 * so.n * (4 + 6 + 3 * order) and down == 8 * so.n * (3 + 6 + 3 * order)
        for a, b in ((h["t"], g.t), (h["dt"], g.dt), (h["x"], g.x), (h["v"], g.v), (h["pot"], g.pot)):
            assert np.array_equal(a, b.cpu().numpy())
        for k in range(order):
            assert np.array_equal(h["D"][k], g.D[k].cpu().numpy())
        if blk == 0:  # identical inputs on the first block: same membership as the oracle, state within tolerance
            assert tn_h == tn_o and na_h == idx_o.shape[0]
            U.check_corrected(order, idx_o, h_old[idx_o], h["x"], h["v"], so.x, so.v, so.D)
    ctx.close()
