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
            assert max(sizes) - min(sizes) <= 1


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
