"""-m "not gpu": the N>1 host logic (i-sharding bounds, packing, the one all-gather per block) on CPU with the gloo
backend, world_size 2 and 3.  After the exchange every replica must hold the identical full state."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1312_1789_b200 import parallel as P


def test_shard_bounds_partition():
    for n_act in (0, 1, 2, 5, 7, 1024, 1048576, 1048577):
        for world in (1, 2, 3, 4, 8):
            cover = []
            for r in range(world):
                lo, hi = P.shard_bounds(n_act, r, world)
                assert 0 <= lo <= hi <= n_act
                cover.append((lo, hi))
            assert cover[0][0] == 0 and cover[-1][1] == n_act
            assert all(cover[i][1] == cover[i + 1][0] for i in range(world - 1))
            sizes = [hi - lo for lo, hi in cover]
            chunk = (n_act + world - 1) // world
            # fixed chunks, the last non-empty one shorter: the gathered buffer is the record array in list order
            assert max(sizes) == chunk
            assert all(lo == min(r * chunk, n_act) for r, (lo, hi) in enumerate(cover))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, order, n, n_act, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    g = torch.Generator().manual_seed(1234)  # same initial replica on every rank
    mk = lambda *s: torch.randn(*s, dtype=torch.float64, generator=g)
    t, dt, pot, x, v = mk(n), mk(n), mk(n), mk(n, 3), mk(n, 3)
    D = [mk(n, 3) for _ in range(8)]
    active = torch.sort(torch.randperm(n, generator=g)[:n_act]).values.to(torch.int32)
    # "correct" my slice: a rank-independent function of the row, applied only to the rows this rank owns
    lo, hi = P.shard_bounds(n_act, rank, world)
    mine = active[lo:hi].to(torch.int64)
    for a in (t, dt, pot, x, v, *D[:order]):
        a[mine] = a[mine] * 2.0 + 1.0
    sent = P.exchange_corrected(active, n_act, rank, world, t, dt, pot, x, v, D, order)
    assert sent == (hi - lo) * P.state_columns(order) * 8
    np.savez(os.path.join(out_dir, "r%d.npz" % rank), t=t.numpy(), dt=dt.numpy(), pot=pot.numpy(), x=x.numpy(),
             v=v.numpy(), **{"D%d" % k: D[k].numpy() for k in range(8)})
    dist.destroy_process_group()


@pytest.mark.parametrize("world,order,n,n_act", [(2, 6, 101, 37), (3, 8, 64, 64), (2, 4, 50, 1)])
def test_exchange_corrected_replicas_identical(tmp_path, world, order, n, n_act):
    port = _free_port()
    mp.spawn(_worker, args=(world, port, order, n, n_act, str(tmp_path)), nprocs=world, join=True)
    # expected: the same update applied to ALL active rows of the common initial replica
    g = torch.Generator().manual_seed(1234)
    mk = lambda *s: torch.randn(*s, dtype=torch.float64, generator=g)
    t, dt, pot, x, v = mk(n), mk(n), mk(n), mk(n, 3), mk(n, 3)
    D = [mk(n, 3) for _ in range(8)]
    active = torch.sort(torch.randperm(n, generator=g)[:n_act]).values.to(torch.int64)
    want = dict(t=t, dt=dt, pot=pot, x=x, v=v, **{"D%d" % k: D[k] for k in range(8)})
    for name, a in want.items():
        if name.startswith("D") and int(name[1:]) >= order:
            continue
        a[active] = a[active] * 2.0 + 1.0
    for r in range(world):
        got = np.load(os.path.join(str(tmp_path), "r%d.npz" % r))
        for name, a in want.items():
            assert np.array_equal(got[name], a.numpy()), (r, name)


# ------------------------------------------------------------------------------------------------------------
# sharded_block_step end to end on CPU: the ctx is a stand-in that runs the ORACLE on numpy views of CPU tensors
# (tests may use the oracle), so the whole i-sharded step -- selection, replicated predict, force + correct on the
# rank's slice, one all-gather -- is exercised with gloo and must reproduce the single-process oracle step exactly.
# ------------------------------------------------------------------------------------------------------------
class _OracleCtx:
    def __init__(self, m):
        from oracle import oracle as O
        self.O, self.m = O, m
        self.pred = None

    def set_option(self, key, value):
        assert key == "geometry_n_act"  # the oracle's summation order does not depend on the partition

    def next_block(self, n, t, dt, active):
        tn, idx = self.O.next_block(t.numpy(), dt.numpy())
        active[: idx.shape[0]] = torch.from_numpy(idx)
        return tn, idx.shape[0]

    def predict(self, n, t_now, order, t, m, x, v, D):
        self.pred = self.O.predict(t_now, order, t.numpy(), x.numpy(), v.numpy(), [d.numpy() for d in D])

    def force(self, act, n_act, order, eps2, acc, jerk, snap, crk, pot):
        xp, vp, ap, jp = self.pred
        out = self.O.force(self.m.numpy(), xp, vp, ap, jp, act[:n_act].numpy(), order, eps2)
        for dst, src in zip((acc, jerk, snap, crk, pot), out):
            if dst is not None and src is not None:
                dst[:n_act] = torch.from_numpy(src)

    def correct(self, act, n_act, order, t_now, eta, dt_min, dt_max, t, dt, x, v, D, pot_state, acc, jerk, snap, crk, pot):
        f = lambda a: None if a is None else a[:n_act].numpy()
        self.O.correct(act[:n_act].numpy(), order, t_now, eta, dt_min, dt_max, t.numpy(), dt.numpy(), x.numpy(),
                       v.numpy(), [d.numpy() for d in D], pot_state.numpy(), f(acc), f(jerk), f(snap), f(crk), f(pot),
                       crit_order=4 if order >= 6 else 0)


class _State:
    pass


def _make_state(order, n):
    from paper_1312_1789_b200 import workloads as W
    from oracle import integrate as OI
    c = W.cluster(5, n)
    so = OI.bootstrap(c["m"], c["x"], c["v"], order, 1e-6)
    s = _State()
    T = lambda a: torch.from_numpy(np.ascontiguousarray(a).copy())
    s.n, s.order, s.eps2, s.eta, s.dt_min, s.dt_max = n, order, 1e-6, 0.1, 2.0**-30, 2.0**-4
    s.m, s.x, s.v, s.t, s.dt, s.pot = T(so.m), T(so.x), T(so.v), T(so.t), T(so.dt), T(so.pot)
    s.D = [T(d) for d in so.D]
    z = lambda *sh: torch.zeros(*sh, dtype=torch.float64)
    s.acc, s.jerk, s.snap, s.crk, s.fpot = z(n, 3), z(n, 3), z(n, 3), z(n, 3), z(n)
    s.active = torch.zeros(n, dtype=torch.int32)
    s.time, s.blocks, s.pairs = 0.0, 0, 0
    s.ctx = _OracleCtx(s.m)
    return s, so


def _step_worker(rank, world, port, order, n, nblk, out_dir, force_exchange):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    s, _ = _make_state(order, n)
    sent = 0
    for _ in range(nblk):
        sent += P.sharded_block_step(s, rank, world, force_exchange=force_exchange)[2]
    assert sent > 0 or not force_exchange
    np.savez(os.path.join(out_dir, "s%d.npz" % rank), t=s.t.numpy(), dt=s.dt.numpy(), x=s.x.numpy(), v=s.v.numpy(),
             pot=s.pot.numpy(), **{"D%d" % k: s.D[k].numpy() for k in range(order)})
    dist.destroy_process_group()


@pytest.mark.parametrize("world,order,force_exchange", [(2, 6, True), (3, 4, True), (2, 8, False)])
def test_sharded_block_step_matches_single_process(tmp_path, world, order, force_exchange):
    """force_exchange: every block is sharded and exchanged; otherwise blocks below REDUNDANT_BELOW are computed by
    every rank with no collective and only larger blocks are sharded."""
    from oracle import integrate as OI
    n, nblk = 193, 12
    mp.spawn(_step_worker, args=(world, _free_port(), order, n, nblk, str(tmp_path), force_exchange), nprocs=world,
             join=True)
    _, so = _make_state(order, n)
    for _ in range(nblk):
        OI.block_step(so, 1e-6, 0.1, 2.0**-30, 2.0**-4, crit_order=4 if order >= 6 else 0)
    for r in range(world):
        got = np.load(os.path.join(str(tmp_path), "s%d.npz" % r))
        assert np.array_equal(got["t"], so.t) and np.array_equal(got["dt"], so.dt), r
        assert np.array_equal(got["x"], so.x) and np.array_equal(got["v"], so.v), r
        assert np.array_equal(got["pot"], so.pot), r
        for k in range(order):
            assert np.array_equal(got["D%d" % k], so.D[k]), (r, k)
