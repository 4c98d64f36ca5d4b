"""-m gpu: the multi-GPU step on the hardware that is here (ONE GPU; no scaling curve is measured, DESIGN.md
section 8): (i) the i-shards of world = 2 and 3, run one after another through the real nbody.Context with the
block's geometry pinned ("geometry_n_act"), reproduce the unsharded step bit for bit -- including slices that start
at lo > 0; (ii) parallel.sharded_block_step through a single-rank NCCL group (pack kernel -> ncclAllGather -> unpack
kernel) equals Integrator.block_step bit for bit; (iii) the row pack / unpack kernels round-trip."""
import os

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_1312_1789_b200 import workloads as W
from paper_1312_1789_b200 import parallel as P


def _integ(config, n, order):
    from paper_1312_1789_b200.scheduler import Integrator
    import torch
    c = W.cluster(config, n)
    g = Integrator(c["m"], c["x"], c["v"], order, c["eps2"], dt_max=2.0**-5)
    g.bootstrap()
    torch.cuda.synchronize()
    return g


def _snapshot(g, order):
    return [a.clone() for a in (g.t, g.dt, g.x, g.v, g.pot, *g.D[:order])]


def _restore(g, snap, order):
    for dst, src in zip((g.t, g.dt, g.x, g.v, g.pot, *g.D[:order]), snap):
        dst.copy_(src)


@pytest.mark.parametrize("order,world", [(6, 2), (8, 3), (4, 3)])
def test_shards_reproduce_unsharded_step_bitwise(order, world):
    import torch
    g = _integ(4, 6151, order)
    c, n, p = g.ctx, g.n, order
    snap_, crk_ = (g.snap if p >= 6 else None), (g.crk if p >= 8 else None)
    checked = 0
    for blk in range(30):
        before = _snapshot(g, order)
        # unsharded reference step
        t_next, n_act = g.block_step()
        ref_state = _snapshot(g, order)
        ref_force = [a[:n_act].clone() for a in (g.acc, g.jerk, g.snap, g.crk, g.fpot)]
        ref_geo = c.last_force_geometry()
        if n_act < world:
            continue
        # the same block, shard by shard (what ranks 0..world-1 would do), from the same initial state
        _restore(g, before, order)
        tn2, na2 = c.next_block(n, g.t, g.dt, g.active)
        assert tn2 == t_next and na2 == n_act
        c.predict(n, t_next, p, g.t, g.m, g.x, g.v, g.D)
        c.set_option("geometry_n_act", n_act)
        for a in (g.acc, g.jerk, g.snap, g.crk, g.fpot):
            a.fill_(float("nan"))
        for r in range(world):
            lo, hi = P.shard_bounds(n_act, r, world)
            if hi == lo:
                continue
            act = g.active[lo:hi]
            sl3 = lambda a: None if a is None else a[lo:hi]
            c.force(act, hi - lo, p, g.eps2, g.acc[lo:hi], g.jerk[lo:hi], sl3(snap_), sl3(crk_), g.fpot[lo:hi])
            geo = c.last_force_geometry()
            assert geo["j_lanes"] == ref_geo["j_lanes"] and geo["j_splits"] == ref_geo["j_splits"]
            c.correct(act, hi - lo, p, t_next, g.eta, g.dt_min, g.dt_max, g.t, g.dt, g.x, g.v, g.D, g.pot,
                      g.acc[lo:hi], g.jerk[lo:hi], sl3(snap_), sl3(crk_), g.fpot[lo:hi])
        c.set_option("geometry_n_act", 0)
        torch.cuda.synchronize()
        for k, (a, b) in enumerate(zip((g.acc, g.jerk, g.snap, g.crk, g.fpot), ref_force)):
            if k < p // 2 or k == 4:
                assert torch.equal(a[:n_act], b), ("force component", k, n_act)
        for a, b in zip(_snapshot(g, order), ref_state):
            assert torch.equal(a, b)
        checked += 1
    assert checked >= 10


def test_sharded_block_step_single_rank_nccl_matches_block_step():
    import torch
    import torch.distributed as dist
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    os.environ.setdefault("MASTER_PORT", "29533")
    dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", 0))
    try:
        order = 6
        a = _integ(5, 4099, order)
        b = _integ(5, 4099, order)
        sent = 0
        for _ in range(20):
            ta, na = a.block_step()
            tb, nb_, s = P.sharded_block_step(b, 0, 1, force_exchange=True)  # pack -> ncclAllGather -> unpack
            assert (ta, na) == (tb, nb_)
            sent += s
        torch.cuda.synchronize()
        assert sent > 0
        for x, y in zip(_snapshot(a, order), _snapshot(b, order)):
            assert torch.equal(x, y)
        # sharded_run: device-driven runs of small blocks + sharded large blocks; same end state as integrate()
        T = 2.0**-5
        a.integrate(T)
        blocks, _ = P.sharded_run(b, T, 0, 1)
        torch.cuda.synchronize()
        assert a.blocks == b.blocks
        for x, y in zip(_snapshot(a, order), _snapshot(b, order)):
            assert torch.equal(x, y)
    finally:
        dist.destroy_process_group()


def test_pack_unpack_rows_roundtrip():
    import torch
    order = 8
    g = _integ(5, 1031, order)
    idx = torch.from_numpy(np.sort(W.rng_for(5, 3).choice(g.n, 300, replace=False)).astype(np.int32)).cuda()
    rec = torch.zeros(300, P.state_columns(order), dtype=torch.float64, device="cuda")
    g.ctx.pack_rows(idx, 300, order, g.t, g.dt, g.pot, g.x, g.v, g.D, rec)
    torch.cuda.synchronize()
    i64 = idx.to(torch.int64)
    assert torch.equal(rec[:, 0], g.t[i64]) and torch.equal(rec[:, 1], g.dt[i64]) and torch.equal(rec[:, 2], g.pot[i64])
    assert torch.equal(rec[:, 3:6], g.x[i64]) and torch.equal(rec[:, 6:9], g.v[i64])
    for k in range(order):
        assert torch.equal(rec[:, 9 + 3 * k: 12 + 3 * k], g.D[k][i64])
    snap = _snapshot(g, order)
    rec2 = rec * 2.0 + 1.0
    g.ctx.unpack_rows(idx, 300, order, g.t, g.dt, g.pot, g.x, g.v, g.D, rec2)
    torch.cuda.synchronize()
    mask = torch.zeros(g.n, dtype=torch.bool, device="cuda")
    mask[i64] = True
    for a, b in zip(_snapshot(g, order), snap):
        assert torch.equal(a[~mask], b[~mask])
        assert torch.equal(a[mask], b[mask] * 2.0 + 1.0)
