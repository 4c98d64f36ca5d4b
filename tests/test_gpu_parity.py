"""-m gpu parity tests: the CUDA path (through the C ABI, include/nbody.h) against the CPU oracle, element by
element on the same seeded inputs.  Integer / index / fp64-exact work must match bit for bit (predictor, corrector,
time step, block membership); the mixed-precision force within BASELINE.json's tolerances (tests/gpu_util.TOL)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_1312_1789_b200 import workloads as W
import gpu_util as U


@pytest.fixture(scope="module")
def nb():
    from paper_1312_1789_b200 import nbody
    return nbody


@pytest.fixture(scope="module")
def O():
    from oracle import oracle
    return oracle


def _cluster_small(config, n):
    c = W.cluster(config, n)
    return c


# ------------------------------------------------------------------------------------------------------------
# predictor: bit-exact (R5, R12)
# ------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("order", [4, 6, 8])
@pytest.mark.parametrize("n", [1, 255, 4099])
def test_predict_bit_exact(nb, O, order, n):
    import torch
    c = _cluster_small(3, max(n, 2))
    m, x, v = c["m"][:n], c["x"][:n], c["v"][:n]
    c = dict(c, m=m, x=np.ascontiguousarray(x), v=np.ascontiguousarray(v), n=n, bh=c["bh"][c["bh"] < n])
    D = W.smooth_field_derivs(c, 6)
    t, dt = W.predictor_times(c["x"])
    t_now = 2.0**-10
    xp, vp, ap, jp = O.predict(t_now, order, t, c["x"], c["v"], D)
    ctx = nb.Context(n)
    ctx.predict(n, t_now, order, U.dev(t), U.dev(m), U.dev(c["x"]), U.dev(c["v"]), [U.dev(d) for d in D[: order - 2]])
    gx = U.zeros(n, 3)
    gv = U.zeros(n, 3, dtype=torch.float32)
    ga = U.zeros(n, 3, dtype=torch.float32) if order >= 6 else None
    gj = U.zeros(n, 3, dtype=torch.float32) if order >= 8 else None
    gm = U.zeros(n, dtype=torch.float32)
    ctx.get_predicted(gx, gv, ga, gj, gm)
    torch.cuda.synchronize()
    assert np.array_equal(gx.cpu().numpy(), xp)
    assert np.array_equal(gv.cpu().numpy(), vp.astype(np.float32))
    assert np.array_equal(gm.cpu().numpy(), m.astype(np.float32))
    if order >= 6:
        assert np.array_equal(ga.cpu().numpy(), ap.astype(np.float32))
    if order >= 8:
        assert np.array_equal(gj.cpu().numpy(), jp.astype(np.float32))
    ctx.close()


# ------------------------------------------------------------------------------------------------------------
# force: config 1 in full, all orders; odd N spanning many tiles with a ragged tail; N_act sweep
# ------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("order", [4, 6, 8])
def test_force_config1_all_active(nb, O, order):
    c = W.cluster(1)
    n = c["n"]
    D = U.oracle_bootstrap_derivs(c, 6)
    t = np.zeros(n)
    idx = np.arange(n, dtype=np.int32)
    xp, vp, ap, jp = O.predict(0.0, order, t, c["x"], c["v"], D)
    ref = O.force(c["m"], xp, vp, ap, jp, idx, order, c["eps2"])
    ctx = nb.Context(n)
    got = U.gpu_force(ctx, n, order, c["eps2"], 0.0, t, c["m"], c["x"], c["v"], D, idx)
    U.check_force(got, ref, order, "cfg1 order %d" % order)
    ctx.close()


@pytest.mark.parametrize("config,order,n", [(2, 4, 4099), (3, 6, 4099), (4, 6, 6151), (5, 8, 4099)])
def test_force_nact_sweep(nb, O, config, order, n):
    """Scaled twins of configs 2..5 (same generators), odd N (16+ tiles and a ragged tail), predicted to
    t = 1/1024 from per-particle times, N_act from 1 to N through every kernel variant."""
    c = W.cluster(config, n)
    D = U.oracle_bootstrap_derivs(c, 6)
    t, dt = W.predictor_times(c["x"])
    t_now = 2.0**-10
    xp, vp, ap, jp = O.predict(t_now, order, t, c["x"], c["v"], D)
    ctx = nb.Context(n)
    rng = W.rng_for(config, 7)
    for n_act in (1, 2, 3, 5, 16, 17, 64, 100, 256, 257, 1000, n):
        idx = W.active_list(n, n_act, rng)
        if n_act < n and c["bh"].size:  # keep the black holes in the small lists: hardest particles
            idx = np.unique(np.concatenate([idx[: max(1, n_act - c["bh"].size)], c["bh"]])).astype(np.int32)
        ref = O.force(c["m"], xp, vp, ap, jp, idx, order, c["eps2"])
        got = U.gpu_force(ctx, n, order, c["eps2"], t_now, t, c["m"], c["x"], c["v"], D, idx)
        U.check_force(got, ref, order, "cfg%d n_act %d geom %s" % (config, n_act, ctx.last_force_geometry()))
    ctx.close()


def test_force_split_and_lane_independence(nb, O):
    """Results do not depend on the j-split factor or the lane variant beyond fp64 summation order
    (<= 1e-12 relative), and are bit-reproducible run to run."""
    c = W.cluster(3, 3001)
    n, order = c["n"], 6
    D = U.oracle_bootstrap_derivs(c, 6)
    t = np.zeros(n)
    idx = W.active_list(n, 37, W.rng_for(3, 9))
    ctx = nb.Context(n)
    base = U.gpu_force(ctx, n, order, c["eps2"], 0.0, t, c["m"], c["x"], c["v"], D, idx)
    again = U.gpu_force(ctx, n, order, c["eps2"], 0.0, t, c["m"], c["x"], c["v"], D, idx)
    for a, b in zip(base, again):
        if a is not None:
            assert np.array_equal(a, b)
    for split, lanes in ((1, 0), (2, 0), (7, 0), (12, 0), (0, 1), (0, 2), (0, 4), (0, 8), (0, 16), (0, 32), (0, 64), (0, 128), (0, 256), (3, 128), (5, 16), (2, 64), (4, 256)):
        ctx.set_option("force_split", split)
        ctx.set_option("force_lanes", lanes)
        got = U.gpu_force(ctx, n, order, c["eps2"], 0.0, t, c["m"], c["x"], c["v"], D, idx)
        g = ctx.last_force_geometry()
        if split:
            assert g["j_splits"] == split
        if lanes:
            assert g["j_lanes"] == lanes
        # different fp32 tile boundaries per lane layout: compare at the fp32-partial level
        assert U.rel_vec(got[0], base[0]) < 2e-6 and U.rel_vec(got[1], base[1]) < 2e-5
        assert U.rel_scal(got[4], base[4]) < 5e-7
    ctx.close()


def test_force_two_body_eps0_and_single(nb, O):
    """eps2 = 0 closed form (R2: self term excluded by index, so no 0 * inf) and N = 1 (all outputs exactly 0)."""
    m = np.array([0.6, 0.4])
    d = 0.8
    x = np.array([[-0.4 * d, 0.0, 0.0], [0.6 * d, 0.0, 0.0]])
    w = np.sqrt(1.0 / d**3)
    v = np.array([[0.0, -0.4 * d * w, 0.0], [0.0, 0.6 * d * w, 0.0]])
    t = np.zeros(2)
    idx = np.arange(2, dtype=np.int32)
    D = [np.zeros((2, 3)) for _ in range(6)]
    ctx = nb.Context(16)
    acc, jerk, _, _, pot = U.gpu_force(ctx, 2, 4, 0.0, 0.0, t, m, x, v, D, idx)
    r = x[1] - x[0]
    dv = v[1] - v[0]
    assert np.allclose(acc[0], m[1] * r / d**3, rtol=1e-6, atol=0)
    assert np.allclose(acc[1], -m[0] * r / d**3, rtol=1e-6, atol=0)
    assert np.allclose(jerk[0][1], m[1] * dv[1] / d**3, rtol=1e-5)
    assert np.allclose(pot, [-m[1] / d, -m[0] / d], rtol=1e-6)
    ref = O.force(m, x, v, None, None, idx, 4, 0.0)
    U.check_force((acc, jerk, None, None, pot), ref, 4, "two-body")
    got = U.gpu_force(ctx, 1, 8, 1e-4, 0.0, t[:1], m[:1], x[:1], v[:1], [d_[:1] for d_ in D], idx[:1])
    for a in got:
        assert np.all(a == 0.0)
    ctx.close()


def test_force_double_single_mode(nb, O):
    """diff_mode 1 (double-single positions) stays inside the same tolerances."""
    c = W.cluster(4, 4099)
    n, order = c["n"], 6
    D = U.oracle_bootstrap_derivs(c, 6)
    t = np.zeros(n)
    idx = np.arange(n, dtype=np.int32)
    xp, vp, ap, jp = O.predict(0.0, order, t, c["x"], c["v"], D)
    ref = O.force(c["m"], xp, vp, ap, jp, idx, order, c["eps2"])
    ctx = nb.Context(n)
    ctx.set_option("diff_mode", 1)
    got = U.gpu_force(ctx, n, order, c["eps2"], 0.0, t, c["m"], c["x"], c["v"], D, idx)
    U.check_force(got, ref, order, "double-single")
    ctx.close()


def test_force_degenerate_inputs(nb, O):
    """Empty inputs are no-ops; a DIFFERENT particle at the identical position is included (R2): with eps2 > 0 it
    adds exactly 0 to acc/jerk/snap and -m/eps to pot; zero-mass particles contribute exactly nothing."""
    import torch
    ctx = nb.Context(64)
    z3, z1 = U.zeros(8, 3), U.zeros(8)
    ctx.predict(0, 0.0, 4, None, None, None, None, [None, None])  # n == 0
    ctx.force(None, 0, 4, 1e-4, None, None, None, None, None)     # n_act == 0
    eps2 = 1e-4
    m = np.array([0.3, 0.2, 0.0, 0.5])
    x = np.array([[0.1, 0.2, 0.3], [0.1, 0.2, 0.3], [0.4, -0.1, 0.0], [-1.0, 0.5, 0.25]])  # 0 and 1 coincide
    v = np.array([[0.0, 0.1, 0.0], [0.0, 0.1, 0.0], [3.0, 2.0, 1.0], [0.2, 0.0, -0.1]])
    D = [np.zeros((4, 3)) for _ in range(6)]
    t = np.zeros(4)
    idx = np.arange(4, dtype=np.int32)
    got = U.gpu_force(ctx, 4, 6, eps2, 0.0, t, m, x, v, D, idx)
    ref = O.force(m, x, v, D[0], D[1], idx, 6, eps2)
    U.check_force(got, ref, 6, "coincident pair")
    # particle 0 sees particle 1 only through the potential: acc equals the pull of particle 3 alone
    only3 = O.force(m[[0, 3]], x[[0, 3]], v[[0, 3]], D[0][[0, 3]], D[1][[0, 3]], np.array([0], dtype=np.int32), 6, eps2)
    assert np.allclose(got[0][0], only3[0][0], rtol=1e-6)
    assert np.isclose(got[4][0], only3[4][0] - m[1] / np.sqrt(eps2), rtol=1e-6)
    # the zero-mass particle 2 changes nobody's result
    wo = U.gpu_force(ctx, 3, 6, eps2, 0.0, t[:3], m[[0, 1, 3]], x[[0, 1, 3]], v[[0, 1, 3]], [d[:3] for d in D], idx[:3])
    for a, b in zip(got, wo):
        if a is not None:
            assert np.array_equal(a[[0, 1, 3]], b)
    ctx.close()
