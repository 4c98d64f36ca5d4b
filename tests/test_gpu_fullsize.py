"""-m gpu: parity at BASELINE.json's FULL sizes, in the launch configurations bench.py times, on sampled outputs the
oracle computes one by one (forced members: every BH, innermost / outermost particles, nearest to each BH, plus a
seeded draw -- where mixed-precision errors are largest).

  config 4: N = 1 048 576, 6th order, ALL active (the bench.py launch: 1024 CTAs of 512 threads, no j-split)
  config 3: N =   262 144, 6th order, N_act sweep 4^0 .. 4^9 (every lane variant and j-split at full N)
  config 2: N =    65 536, 4th order, N_act = 1, 16, 256, 4096, 65 536
  config 5: N = 2 097 152, 8th order, ALL active, and N_act = 3 .. 1.5 M (j-split partials at the largest N)
"""
import json
import os

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_1312_1789_b200 import workloads as W
import gpu_util as U


def _setup(config, order):
    import torch
    from paper_1312_1789_b200 import nbody
    c = W.cluster(config)
    n = c["n"]
    D = W.smooth_field_derivs(c, 6)
    t, dt = W.predictor_times(c["x"])
    t_now = 2.0**-10
    ctx = nbody.Context(n)
    ctx.predict(n, t_now, order, U.dev(t), U.dev(c["m"]), U.dev(c["x"]), U.dev(c["v"]), [U.dev(d) for d in D[: order - 2]])
    from oracle import oracle as O
    xp, vp, ap, jp = O.predict(t_now, order, t, c["x"], c["v"], D)
    return c, n, ctx, O, (xp, vp, ap, jp)


def _force(ctx, idx_dev, n_act, order, eps2):
    import torch
    acc, jerk, pot = U.zeros(n_act, 3), U.zeros(n_act, 3), U.zeros(n_act)
    snap = U.zeros(n_act, 3) if order >= 6 else None
    crk = U.zeros(n_act, 3) if order >= 8 else None
    ctx.force(idx_dev, n_act, order, eps2, acc, jerk, snap, crk, pot)
    torch.cuda.synchronize()
    return acc, jerk, snap, crk, pot


@pytest.mark.parametrize("config,order,sample", [(4, 6, 1024), (5, 8, 512)])
def test_all_active_full_size_sampled(config, order, sample):
    import torch
    c, n, ctx, O, (xp, vp, ap, jp) = _setup(config, order)
    idx_all = torch.arange(n, dtype=torch.int32, device="cuda")
    out = _force(ctx, idx_all, n, order, c["eps2"])
    g = ctx.last_force_geometry()
    assert g["j_lanes"] == 1 and g["j_splits"] == 1 and g["ctas"] == (n + 1023) // 1024  # the configuration bench.py times
    s = W.oracle_sample(c, size=sample)
    ref = O.force(c["m"], xp, vp, ap, jp, s, order, c["eps2"])
    ii = torch.from_numpy(s.astype(np.int64)).cuda()
    got = tuple(None if a is None else a[ii].cpu().numpy() for a in out)
    errs = U.check_force(got, ref, order, "cfg%d all-active N=%d" % (config, n))
    print("cfg%d N=%d order %d sampled max rel errors: %s" % (config, n, order, errs))
    ctx.close()


@pytest.mark.parametrize("config,order,nacts", [(3, 6, [4**k for k in range(10)]), (2, 4, [1, 16, 256, 4096, 65536]),
                                                 (5, 8, [3, 1000, 300000, 1500000])])
def test_nact_sweep_full_size_sampled(config, order, nacts):
    import torch
    c, n, ctx, O, (xp, vp, ap, jp) = _setup(config, order)
    rng = W.rng_for(config, 31)
    forced = W.oracle_sample(c, size=160)  # forced members only (+ a few): always part of every active list
    for n_act in nacts:
        n_act = min(n_act, n)
        idx = W.active_list(n, n_act, rng)
        if n_act < n:
            k = min(forced.shape[0], n_act)
            idx = np.unique(np.concatenate([idx[: n_act - k], forced[:k]])).astype(np.int32)
        na = idx.shape[0]
        out = _force(ctx, U.dev(idx), na, order, c["eps2"])
        # oracle on <= 1024 of the active particles (positions inside the active list)
        pick = np.arange(na) if na <= 1024 else np.unique(np.concatenate(
            [np.nonzero(np.isin(idx, forced))[0], rng.choice(na, 1024 - forced.shape[0], replace=False)]))
        ref = O.force(c["m"], xp, vp, ap, jp, idx[pick], order, c["eps2"])
        pp = torch.from_numpy(pick.astype(np.int64)).cuda()
        got = tuple(None if a is None else a[pp].cpu().numpy() for a in out)
        U.check_force(got, ref, order, "cfg%d N=%d n_act=%d geom %s" % (config, n, na, ctx.last_force_geometry()))
    ctx.close()


@pytest.mark.parametrize("config,order", [(3, 6), (4, 6), (5, 8)])
def test_full_size_physically_consistent_derivatives(config, order):
    """The hard inputs (SURVEY.md 8(d) "primary", Appendix A): the Taylor coefficients D_0..D_3 are the cluster's OWN
    acceleration, jerk, snap and crackle (GPU bootstrap R9b, handed unchanged to the oracle), so Sum m_j a_j =
    Sum m_j j_j = 0 and the far-halo snap / crackle sums are near-total cancellations.  All-active call at the full
    size (the launch bench.py times), predicted to t = 2^-10; oracle on the forced-member sample: every BH, the 32
    innermost, the 4096 OUTERMOST, the 32 nearest to each BH and a seeded draw.  Prints, per quantity, max / 99.9th
    percentile / worst particle's radius and kappa and asserts BASELINE.json's tolerances."""
    import torch
    from paper_1312_1789_b200.scheduler import Integrator
    from oracle import oracle as O
    c = W.cluster(config)
    n, eps2 = c["n"], c["eps2"]
    H = 2.0**-10
    g = Integrator(c["m"], c["x"], c["v"], order, eps2)
    g.bootstrap(fixed_dt=H)
    torch.cuda.synchronize()
    D = [d.cpu().numpy().copy() for d in g.D[:6]]  # D_4, D_5 are zero after the bootstrap (R9b)
    t = np.zeros(n)
    s = W.oracle_sample(c, size=6144, n_outer=4096)
    xp, vp, ap, jp = O.predict(H, order, t, c["x"], c["v"], D)
    ref = O.force(c["m"], xp, vp, ap, jp, s, order, eps2)
    absn = O.force_abs(c["m"], xp, vp, ap, jp, s, order, eps2)
    g.ctx.predict(n, H, order, g.t, g.m, g.x, g.v, g.D)
    out = _force(g.ctx, g.all_idx, n, order, eps2)
    geo = g.ctx.last_force_geometry()
    assert geo["j_lanes"] == 1 and (geo["j_splits"] == 1 or config == 3)  # configs 4 and 5: the unsplit launch bench.py times
    ii = torch.from_numpy(s.astype(np.int64)).cuda()
    got = tuple(None if a is None else a[ii].cpu().numpy() for a in out)
    radius = np.linalg.norm(c["x"][s], axis=1)
    rep = U.conditioning_report(got, ref, absn, radius, order)
    line = dict(test="full_size_physically_consistent", config=config, n=n, order=order, sample=int(s.shape[0]),
                geometry=geo, report=rep)
    print(json.dumps(line))
    os.makedirs("gpurun_out", exist_ok=True)
    with open(os.path.join("gpurun_out", "parity_fullsize_cfg%d.json" % config), "w") as f:
        json.dump(line, f, indent=1)
    U.check_force(got, ref, order, "cfg%d full size, bootstrap derivatives" % config)
    g.ctx.close()


def test_double_single_mode_order4_full_size():
    """diff_mode 1 (double-single positions, |dd|/|d| <= 1.2e-7 instead of 6e-8; R10 note) at config 2's full size,
    4th order, ALL 65 536 particles against the oracle, with the conditioning report; the literal mode beside it.  The
    option stays off by default (BASELINE.json words the contract as "differences formed in fp64"): this is the evidence
    for what it would cost in accuracy."""
    import torch
    from paper_1312_1789_b200 import nbody
    from oracle import oracle as O
    c = W.cluster(2)
    n, order, eps2 = c["n"], 4, c["eps2"]
    idx = np.arange(n, dtype=np.int32)
    D = [np.zeros((n, 3)), np.zeros((n, 3))]
    t = np.zeros(n)
    ref = O.force(c["m"], c["x"], c["v"], None, None, idx, order, eps2)
    absn = O.force_abs(c["m"], c["x"], c["v"], None, None, idx, order, eps2)
    radius = np.linalg.norm(c["x"], axis=1)
    out = {}
    for mode in (0, 1):
        ctx = nbody.Context(n)
        ctx.set_option("diff_mode", mode)
        got = U.gpu_force(ctx, n, order, eps2, 0.0, t, c["m"], c["x"], c["v"], D, idx)
        out[mode] = U.conditioning_report(got, ref, absn, radius, order)
        U.check_force(got, ref, order, "cfg2 full size diff_mode %d" % mode)
        ctx.close()
    line = dict(test="double_single_order4_full_size", config=2, n=n, order=order, literal=out[0], double_single=out[1])
    print(json.dumps(line))
    os.makedirs("gpurun_out", exist_ok=True)
    with open(os.path.join("gpurun_out", "parity_fullsize_cfg2_diffmodes.json"), "w") as f:
        json.dump(line, f, indent=1)


def test_device_driven_run_full_size_bit_identical():
    """nbody_run_blocks at config 3's full size (N = 262 144, 6th order): the first 40 blocks after the bootstrap --
    the all-active first block (S = 4 j-split, 1024 work items on the persistent grid) down to single-particle blocks --
    leave the same bits as the host-driven path."""
    import torch
    from paper_1312_1789_b200.scheduler import Integrator
    c = W.cluster(3)
    a = Integrator(c["m"], c["x"], c["v"], 6, c["eps2"])
    b = Integrator(c["m"], c["x"], c["v"], 6, c["eps2"])
    a.bootstrap(fixed_dt=2.0**-10)  # everybody due at 2^-10: the first block is all-active, the criterion then spreads the steps
    b.bootstrap(fixed_dt=2.0**-10)
    sizes = [a.block_step()[1] for _ in range(40)]
    r = b.run(1.0, max_blocks=40)
    torch.cuda.synchronize()
    assert r["blocks"] == 40 and r["pairs"] == sum(sizes) * a.n and max(sizes) == a.n
    for x, y in ((a.t, b.t), (a.dt, b.dt), (a.x, b.x), (a.v, b.v), (a.pot, b.pot), *zip(a.D[:6], b.D[:6])):
        assert torch.equal(x, y)
