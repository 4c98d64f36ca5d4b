"""-m gpu: the boundary's error behaviour and edge cases (include/nbody.h): alignment, eps2 that would flush to zero,
the "validate" debug option, the exponent range of the power-of-two step rule, forced splits beyond the scratch,
pads masked by index, coincident particles at eps2 = 0, j-split independence at the fp64 level."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_1312_1789_b200 import workloads as W
import gpu_util as U


class _Off:
    """A device pointer displaced by `off` bytes (argument marshalling test only)."""

    def __init__(self, t, off):
        self.t, self.off = t, off

    def data_ptr(self):
        return self.t.data_ptr() + self.off

    def is_contiguous(self):
        return True


def test_alignment_and_eps2_flush_are_rejected():
    import torch
    from paper_1312_1789_b200 import nbody as nb
    ctx = nb.Context(100)
    z, z1 = U.zeros(101, 3), U.zeros(101)
    idx = torch.arange(100, dtype=torch.int32, device="cuda")
    with pytest.raises(nb.NBodyError) as e:
        ctx.predict(100, 0.0, 4, z1, z1, _Off(z, 4), z, [z, z])
    assert e.value.code == nb.EINVAL
    ctx.predict(100, 0.0, 4, z1, z1, z, z, [z, z])
    with pytest.raises(nb.NBodyError) as e:
        ctx.force(idx, 10, 4, 1e-4, z, _Off(z, 4), None, None, z1)
    assert e.value.code == nb.EINVAL
    with pytest.raises(nb.NBodyError) as e:
        ctx.force(_Off(idx, 2), 10, 4, 1e-4, z, z, None, None, z1)
    assert e.value.code == nb.EINVAL
    ctx.force(_Off(idx, 4), 10, 4, 1e-4, z, z, None, None, z1)  # an offset active list (a shard) is fine
    with pytest.raises(nb.NBodyError) as e:
        ctx.force(idx, 10, 4, 1e-40, z, z, None, None, z1)  # 0 < eps2 < FLT_MIN: would silently become 0
    assert e.value.code == nb.EINVAL
    ctx.force(idx, 10, 4, 0.0, z, z, None, None, z1)
    with pytest.raises(nb.NBodyError) as e:
        ctx.correct(idx, 10, 4, 0.1, 0.1, 2.0**-10, 2.0**-4, z1, z1, z, z, [z] * 4, _Off(z1, 4), z, z, None, None, z1)
    assert e.value.code == nb.EINVAL
    with pytest.raises(nb.NBodyError):
        ctx.set_option("geometry_n_act", 101)
    for bad in (3, 512, -1):  # the j-lane variants are the powers of two up to 256
        with pytest.raises(nb.NBodyError) as e:
            ctx.set_option("force_lanes", bad)
        assert e.value.code == nb.EINVAL
    for ok in (256, 16, 0):
        ctx.set_option("force_lanes", ok)
    with pytest.raises(nb.NBodyError) as e:
        ctx.set_option("no_such_option", 1)
    assert e.value.code == nb.EINVAL
    ctx.set_option("geometry_n_act", 5)
    with pytest.raises(nb.NBodyError) as e:
        ctx.force(idx, 10, 4, 1e-4, z, z, None, None, z1)  # n_act above the declared block size
    assert e.value.code == nb.EINVAL
    ctx.close()


def test_validate_option_checks_indices_and_due_times():
    import torch
    from paper_1312_1789_b200 import nbody as nb
    n = 500
    c = W.cluster(1, n)
    ctx = nb.Context(n)
    ctx.set_option("validate", 1)
    D = [U.dev(np.zeros((n, 3))) for _ in range(4)]
    t, dt = U.dev(np.zeros(n)), U.dev(np.full(n, 2.0**-6))
    m, x, v = U.dev(c["m"]), U.dev(c["x"]), U.dev(c["v"])
    ctx.predict(n, 2.0**-6, 4, t, m, x, v, D)
    acc, jerk, pot = U.zeros(n, 3), U.zeros(n, 3), U.zeros(n)
    good = torch.tensor([3, 17, 18, 499], dtype=torch.int32, device="cuda")
    ctx.force(good, 4, 4, 1e-4, acc, jerk, None, None, pot)
    for bad in ([3, 17, 17, 499], [3, 18, 17, 499], [3, 17, 18, 500], [-1, 17, 18, 499]):
        b = torch.tensor(bad, dtype=torch.int32, device="cuda")
        acc.fill_(7.0)
        with pytest.raises(nb.NBodyError) as e:
            ctx.force(b, 4, 4, 1e-4, acc, jerk, None, None, pot)
        assert e.value.code == nb.EINVAL
        assert bool((acc == 7.0).all())  # rejected before any arithmetic
    pstate = U.zeros(n)
    ctx.correct(good, 4, 4, 2.0**-6, 0.1, 2.0**-20, 2.0**-4, t, dt, x, v, D, pstate, acc, jerk, None, None, pot)
    # the four particles now sit at t = 2^-6: they are no longer due at 2^-6
    with pytest.raises(nb.NBodyError) as e:
        ctx.correct(good, 4, 4, 2.0**-6, 0.1, 2.0**-20, 2.0**-4, t, dt, x, v, D, pstate, acc, jerk, None, None, pot)
    assert e.value.code == nb.EINVAL
    ctx.close()


def test_dt_exponent_range():
    """R9's exact power-of-two comparison needs (|k| + 1) q <= 1022: dt_min = 2^-300 is fine (and bit-exact against
    the oracle) with the 4-derivative criterion, rejected with the order-8 criterion (q = 5)."""
    import torch
    from oracle import oracle as O
    from paper_1312_1789_b200 import nbody as nb
    n, order = 300, 8
    c = W.cluster(5, n)
    D = U.oracle_bootstrap_derivs(c, 8)
    t, dt = W.predictor_times(c["x"])
    t_now = 2.0**-10
    idx = np.arange(n, dtype=np.int32)
    xp, vp, ap, jp = O.predict(t_now, order, t, c["x"], c["v"], D)
    f = O.force(c["m"], xp, vp, ap, jp, idx, order, c["eps2"])
    ctx = nb.Context(n)
    args = lambda: (U.dev(t), U.dev(dt), U.dev(c["x"]), U.dev(c["v"]), [U.dev(d) for d in D], U.zeros(n))
    gt, gdt, gx, gv, gD, gp = args()
    ctx.set_option("dt_criterion_order", 4)
    ctx.correct(U.dev(idx), n, order, t_now, 0.1, 2.0**-300, 2.0**-4, gt, gdt, gx, gv, gD, gp, *[U.dev(a) for a in f])
    ot, odt, ox, ov, oD = t.copy(), dt.copy(), c["x"].copy(), c["v"].copy(), [d.copy() for d in D]
    O.correct(idx, order, t_now, 0.1, 2.0**-300, 2.0**-4, ot, odt, ox, ov, oD, np.zeros(n), *f, crit_order=4)
    torch.cuda.synchronize()
    assert np.array_equal(gdt.cpu().numpy(), odt) and np.array_equal(gx.cpu().numpy(), ox)
    ctx.set_option("dt_criterion_order", 8)
    with pytest.raises(nb.NBodyError) as e:
        ctx.correct(U.dev(idx), n, order, t_now, 0.1, 2.0**-300, 2.0**-4, gt, gdt, gx, gv, gD, gp, *[U.dev(a) for a in f])
    assert e.value.code == nb.EINVAL
    ctx.correct(U.dev(idx), n, order, t_now, 0.1, 2.0**-200, 2.0**-4, gt, gdt, gx, gv, gD, gp, *[U.dev(a) for a in f])
    with pytest.raises(nb.NBodyError) as e:
        ctx.initial_dt(n, U.dev(f[0]), U.dev(f[1]), 0.01, 5e-324, 2.0**-4, U.zeros(n))  # subnormal dt_min
    assert e.value.code == nb.EINVAL
    ctx.close()


def test_forced_split_beyond_scratch_is_rejected():
    from paper_1312_1789_b200 import nbody as nb
    n = 4099
    c = W.cluster(2, n)
    ctx = nb.Context(n)
    D = [np.zeros((n, 3)) for _ in range(2)]
    idx = np.arange(n, dtype=np.int32)
    ctx.set_option("force_split", 17)  # 17 tiles: S = 17 is legal, 17 x 4099 rows fit
    U.gpu_force(ctx, n, 4, c["eps2"], 0.0, np.zeros(n), c["m"], c["x"], c["v"], D, idx)
    assert ctx.last_force_geometry()["j_splits"] == 17
    ctx.set_option("force_split", 60000)  # clamped to the tile count: still inside the scratch
    U.gpu_force(ctx, n, 4, c["eps2"], 0.0, np.zeros(n), c["m"], c["x"], c["v"], D, idx)
    assert ctx.last_force_geometry()["j_splits"] == 17
    ctx.close()
    # capacity 70 000: 274 tiles, scratch = max(4 x 148 x 1024, 4 x 70 000) = 606 208 rows; S = 9 x 70 000 rows exceeds it
    n = 70000
    c = W.cluster(2, n)
    ctx = nb.Context(n)
    ctx.set_option("force_split", 9)
    with pytest.raises(nb.NBodyError) as e:
        U.gpu_force(ctx, n, 4, c["eps2"], 0.0, np.zeros(n), c["m"], c["x"], c["v"], [np.zeros((n, 3))] * 2,
                    np.arange(n, dtype=np.int32))
    assert e.value.code == nb.EINVAL
    ctx.set_option("force_split", 8)
    U.gpu_force(ctx, n, 4, c["eps2"], 0.0, np.zeros(n), c["m"], c["x"], c["v"], [np.zeros((n, 3))] * 2,
                np.arange(n, dtype=np.int32))
    ctx.close()


def test_pads_are_masked_by_index_and_coincident_pairs():
    """A real particle sitting exactly where the zero-mass pads are parked (1e6, 1e6, 1e6) gets finite results even
    with eps2 = 0 (the pads of the last j-tile are excluded by index); two DISTINCT coincident particles at
    eps2 = 0 are the documented undefined case: NaN in their own outputs, finite for everybody else."""
    from oracle import oracle as O
    from paper_1312_1789_b200 import nbody as nb
    m = np.array([0.5, 0.25, 0.25])
    x = np.array([[1e6, 1e6, 1e6], [0.3, 0.1, -0.2], [-0.4, 0.2, 0.1]])
    v = np.array([[0.0, 0.1, 0.0], [0.2, 0.0, 0.0], [0.0, -0.3, 0.1]])
    D = [np.zeros((3, 3)) for _ in range(6)]
    idx = np.arange(3, dtype=np.int32)
    ctx = nb.Context(16)
    for order in (4, 6, 8):
        got = U.gpu_force(ctx, 3, order, 0.0, 0.0, np.zeros(3), m, x, v, D, idx)
        for a in got:
            if a is not None:
                assert np.all(np.isfinite(a))
        ref = O.force(m, x, v, D[0], D[1], idx, order, 0.0)
        acc_err = np.linalg.norm(got[0] - ref[0], axis=1) / np.linalg.norm(ref[0], axis=1)
        assert np.all(acc_err < 1e-5)
    x2 = np.array([[0.1, 0.2, 0.3], [0.1, 0.2, 0.3], [-1.0, 0.5, 0.25]])
    got = U.gpu_force(ctx, 3, 4, 0.0, 0.0, np.zeros(3), m, x2, v, D, idx)
    assert not np.all(np.isfinite(got[0][0])) and not np.all(np.isfinite(got[0][1]))
    assert np.all(np.isfinite(got[0][2])) and np.isfinite(got[4][2])
    ctx.close()


def test_split_independence_at_fp64_level_for_one_lane():
    """At JL = 1 a j-split moves no fp32 chunk boundary (chunks are 64 consecutive j of a 256-particle tile): it only
    regroups the fp64 sum of the chunk partials, so results agree to ~1e-15 times the conditioning of the sum
    (SURVEY.md 7.3 item 3); checked per particle with kappa from the oracle's c-16 diagnostic."""
    from oracle import oracle as O
    from paper_1312_1789_b200 import nbody as nb
    c = W.cluster(3, 5003)
    n, order = c["n"], 6
    D = U.oracle_bootstrap_derivs(c, 6)
    t = np.zeros(n)
    idx = W.active_list(n, 1500, W.rng_for(3, 9))
    xp, vp, ap, jp = O.predict(0.0, order, t, c["x"], c["v"], D)
    ref = O.force(c["m"], xp, vp, ap, jp, idx, order, c["eps2"])
    absn = O.force_abs(c["m"], xp, vp, ap, jp, idx, order, c["eps2"])
    ctx = nb.Context(n)
    ctx.set_option("force_lanes", 1)
    ctx.set_option("force_split", 1)
    base = U.gpu_force(ctx, n, order, c["eps2"], 0.0, t, c["m"], c["x"], c["v"], D, idx)
    worst = 0.0
    for split in (2, 3, 7, 20):
        ctx.set_option("force_split", split)
        got = U.gpu_force(ctx, n, order, c["eps2"], 0.0, t, c["m"], c["x"], c["v"], D, idx)
        assert ctx.last_force_geometry() == dict(i_per_thread=2, j_lanes=1, j_splits=split, ctas=2 * split)
        for k in range(3):
            kap = absn[k] / np.linalg.norm(ref[k], axis=1)
            rel = np.linalg.norm(got[k] - base[k], axis=1) / np.linalg.norm(base[k], axis=1)
            assert np.all(rel <= 1e-15 * np.maximum(kap, 1.0)), (split, k, float(np.max(rel / kap)))
            worst = max(worst, float(np.max(rel)))
        assert np.all(np.abs(got[4] - base[4]) <= 1e-15 * np.abs(base[4]))
    print("JL=1 split independence: worst relative difference %.2e" % worst)
    ctx.close()
