"""-m gpu: nbody_nearest (SURVEY 8(f) N4 neighbour output, reading R16) against the oracle's c-17, bit for bit: the index
is integer work and the distance that decides it is taken in the same precision on both sides (fp64-formed differences
rounded to fp32, fp32 fma sum in a stated order).  Both sides see the same predicted positions: the j-store's own, read
back through the nbody_get_predicted test hook (the predictor's parity is tested in test_gpu_parity.py)."""
import json
import os

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_1312_1789_b200 import workloads as W
import gpu_util as U


def _predicted(ctx, c, order, n):
    import torch
    D = W.smooth_field_derivs(c, order - 2)
    t, _ = W.predictor_times(c["x"])
    ctx.predict(n, 2.0**-10, order, U.dev(t), U.dev(c["m"]), U.dev(c["x"]), U.dev(c["v"]), [U.dev(d) for d in D])
    xp = U.zeros(n, 3)
    vp = torch.zeros(n, 3, dtype=torch.float32, device="cuda")
    m32 = torch.zeros(n, dtype=torch.float32, device="cuda")
    ctx.get_predicted(xp, vp, None, None, m32)
    torch.cuda.synchronize()
    return xp.cpu().numpy()


def _check(ctx, O, xp, idx):
    import torch
    na = idx.shape[0]
    who = torch.full((na,), -7, dtype=torch.int32, device="cuda")
    r2 = U.zeros(na)
    r2.fill_(float("nan"))
    ctx.nearest(U.dev(idx), na, who, r2)
    torch.cuda.synchronize()
    owho, or2 = O.nearest(xp, idx)
    assert np.array_equal(who.cpu().numpy(), owho)
    assert np.array_equal(r2.cpu().numpy(), or2)


@pytest.mark.parametrize("n", [2, 257, 20011])
def test_nearest_bit_exact(n):
    from paper_1312_1789_b200 import nbody as nb
    from oracle import oracle as O
    c = W.cluster(2, n)
    ctx = nb.Context(n)
    xp = _predicted(ctx, c, 6, n)
    rng = W.rng_for(2, 60)
    _check(ctx, O, xp, np.arange(n, dtype=np.int32))  # all active: several i-tiles and j-splits at n = 20011
    for na in (1, min(n, 37), min(n, 1000)):
        _check(ctx, O, xp, W.active_list(n, na, rng))
    _check(ctx, O, xp, np.arange(n - 1, -1, -1, dtype=np.int32)[: min(n, 300)].copy())  # outputs follow the list's order
    ctx.close()


def test_nearest_ties_coincident_and_single():
    import torch
    from paper_1312_1789_b200 import nbody as nb
    from oracle import oracle as O
    # six particles: four at distance 1 of the first (ties -> lowest index), two coincident far away
    x = np.array([[0.0, 0.0, 0.0], [1.0, 0.0, 0.0], [-1.0, 0.0, 0.0], [0.0, 1.0, 0.0], [9.0, 9.0, 9.0], [9.0, 9.0, 9.0]])
    n = x.shape[0]
    z3, z1 = np.zeros((n, 3)), np.zeros(n)
    ctx = nb.Context(n)
    ctx.predict(n, 0.0, 4, U.dev(z1), U.dev(z1 + 1.0), U.dev(x), U.dev(z3), [U.dev(z3), U.dev(z3)])
    idx = np.arange(n, dtype=np.int32)
    _check(ctx, O, x, idx)
    who = torch.zeros(n, dtype=torch.int32, device="cuda")
    r2 = U.zeros(n)
    ctx.nearest(U.dev(idx), n, who, r2)
    assert who.cpu().tolist() == [1, 0, 0, 0, 5, 4] and r2.cpu().tolist() == [1.0, 1.0, 1.0, 1.0, 0.0, 0.0]
    ctx.close()
    # a single particle has no neighbour
    ctx = nb.Context(1)
    ctx.predict(1, 0.0, 4, U.dev(z1[:1]), U.dev(z1[:1] + 1.0), U.dev(x[:1]), U.dev(z3[:1]), [U.dev(z3[:1]), U.dev(z3[:1])])
    who = torch.zeros(1, dtype=torch.int32, device="cuda")
    r2 = U.zeros(1)
    ctx.nearest(U.dev(idx[:1]), 1, who, r2)
    assert who.cpu().tolist() == [-1] and np.isinf(r2.cpu().numpy()[0])
    # errors: before any predict, more active particles than the j-store holds
    ctx2 = nb.Context(4)
    with pytest.raises(nb.NBodyError) as e:
        ctx2.nearest(U.dev(idx[:1]), 1, who, r2)
    assert e.value.code == nb.ESTATE
    with pytest.raises(nb.NBodyError) as e:
        ctx.nearest(U.dev(idx[:2]), 2, who, r2)
    assert e.value.code == nb.EINVAL
    ctx.close()
    ctx2.close()


def test_nearest_full_size_sampled():
    """Config 5's full size (N = 2 097 152): the oracle sample (black holes, innermost, outermost, nearest to the BHs, a
    seeded draw) bit for bit, and the rate of an all-particles-vs-65 536 call for the record."""
    import torch
    from paper_1312_1789_b200 import nbody as nb
    from oracle import oracle as O
    c = W.cluster(5)
    n = c["n"]
    ctx = nb.Context(n)
    xp = _predicted(ctx, c, 8, n)
    _check(ctx, O, xp, np.sort(W.oracle_sample(c, size=2048)).astype(np.int32))
    na = 65536
    idx = U.dev(W.active_list(n, na, W.rng_for(5, 61)))
    who = torch.zeros(na, dtype=torch.int32, device="cuda")
    r2 = U.zeros(na)
    ctx.nearest(idx, na, who, r2)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(3):
        ctx.nearest(idx, na, who, r2)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / 3
    line = dict(test="nearest_full_size", config=5, n=n, n_act=na, ms=ms, pairs_per_s=na * n / (ms * 1e-3))
    print(json.dumps(line))
    os.makedirs("gpurun_out", exist_ok=True)
    with open(os.path.join("gpurun_out", "nearest_fullsize.json"), "w") as f:
        json.dump(line, f)
    ctx.close()
