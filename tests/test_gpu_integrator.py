"""-m gpu tests of corrector / time step / block selection (bit-exact vs the oracle), the host scheduler
(end-to-end block-step integration vs the oracle's own driver), error codes and the host-buffer path."""
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


def _state(config, n, order, seed_stream=11):
    """A mid-run looking state: positions/velocities of the cluster, D_k from the oracle bootstrap, per-particle
    dyadic t, dt with every particle of the active list due at t_now."""
    c = W.cluster(config, n)
    D = U.oracle_bootstrap_derivs(c, 8)
    t, dt = W.predictor_times(c["x"])
    return c, D, t, dt


@pytest.mark.parametrize("order,crit", [(4, 0), (6, 0), (8, 0), (4, 4), (6, 6), (8, 8), (6, 4), (8, 4), (8, 6)])
def test_correct_bit_exact(nb, O, order, crit):
    import torch
    n = 3001
    c, D, t, dt = _state(3, n, order)
    t_now = 2.0**-10
    rng = W.rng_for(3, 21)
    idx = W.active_list(n, 1203, rng)
    # force inputs at t1: the oracle's force on the oracle's prediction (any fp64 arrays would do: the corrector
    # is compared on identical inputs)
    xp, vp, ap, jp = O.predict(t_now, order, t, c["x"], c["v"], D)
    acc, jerk, snap, crk, pot = O.force(c["m"], xp, vp, ap, jp, idx, order, c["eps2"])
    for eta in (0.1, 0.02, 0.75):
        # oracle
        ot, odt, ox, ov = t.copy(), dt.copy(), c["x"].copy(), c["v"].copy()
        oD = [d.copy() for d in D]
        opot = np.zeros(n)
        O.correct(idx, order, t_now, eta, 2.0**-30, 2.0**-4, ot, odt, ox, ov, oD, opot, acc, jerk, snap, crk, pot,
                  crit_order=crit)
        # GPU
        gt, gdt, gx, gv = U.dev(t), U.dev(dt), U.dev(c["x"]), U.dev(c["v"])
        gD = [U.dev(d) for d in D]
        gpot = U.zeros(n)
        ctx = nb.Context(n)
        ctx.set_option("dt_criterion_order", crit)  # same value, same meaning on both sides (0 = automatic, R8b)
        ctx.correct(U.dev(idx), idx.shape[0], order, t_now, eta, 2.0**-30, 2.0**-4, gt, gdt, gx, gv, gD, gpot,
                    U.dev(acc), U.dev(jerk), None if snap is None else U.dev(snap),
                    None if crk is None else U.dev(crk), U.dev(pot))
        torch.cuda.synchronize()
        assert np.array_equal(gt.cpu().numpy(), ot)
        assert np.array_equal(gdt.cpu().numpy(), odt), "block time steps differ"
        assert np.array_equal(gx.cpu().numpy(), ox)
        assert np.array_equal(gv.cpu().numpy(), ov)
        assert np.array_equal(gpot.cpu().numpy(), opot)
        for k in range(order):
            assert np.array_equal(gD[k].cpu().numpy(), oD[k]), "a^(%d) differs" % k
        for k in range(order, 8):
            assert np.array_equal(gD[k].cpu().numpy(), D[k])  # untouched
        assert len(np.unique(odt[idx])) > 1  # the test exercises several step levels
        ctx.close()


def test_initial_dt_and_next_block_bit_exact(nb, O):
    import torch
    n = 70001  # several selection chunks (2048 per CTA) and a ragged tail
    c = W.cluster(2, n)
    idx = np.arange(n, dtype=np.int32)
    rng = W.rng_for(2, 5)
    acc = rng.normal(size=(n, 3)) * np.exp(rng.uniform(-3, 3, (n, 1)))
    jerk = rng.normal(size=(n, 3)) * np.exp(rng.uniform(-3, 8, (n, 1)))
    jerk[17] = 0.0
    ref = O.initial_dt(acc, jerk, 0.01, 2.0**-30, 2.0**-4)
    ctx = nb.Context(n)
    gdt = U.zeros(n)
    ctx.initial_dt(n, U.dev(acc), U.dev(jerk), 0.01, 2.0**-30, 2.0**-4, gdt)
    torch.cuda.synchronize()
    assert np.array_equal(gdt.cpu().numpy(), ref)
    assert ref[17] == 2.0**-4
    # block selection at several stages of a synthetic schedule
    t = np.zeros(n)
    dt = ref.copy()
    act = torch.zeros(n, dtype=torch.int32, device="cuda")
    for step in range(6):
        tn, oidx = O.next_block(t, dt)
        gtn, gna = ctx.next_block(n, U.dev(t), U.dev(dt), act)
        assert gtn == tn and gna == oidx.shape[0]
        assert np.array_equal(act[:gna].cpu().numpy(), oidx)
        t[oidx] = tn  # advance the block (keep dt): next selection differs
        if step == 3:
            dt[oidx] *= 0.5
    # all due at once
    t[:] = 0.25
    dt[:] = 0.125
    gtn, gna = ctx.next_block(n, U.dev(t), U.dev(dt), act)
    assert gtn == 0.375 and gna == n and np.array_equal(act.cpu().numpy(), idx)
    ctx.close()


@pytest.mark.parametrize("n", [1, 31, 1025, 300007, 2600003])
def test_next_block_chunk_shapes(nb, O, n):
    """The one-pass selection kernel over its chunk shapes: a single particle, less than a warp, one row per CTA, several
    rows, and more rows than the shared-memory key cache holds (n > 16 x 1024 x 148).  Blocks: a few scattered particles
    including the first and the last one, every other particle, a dense stretch inside one chunk, everybody; t_next, n_act
    and the ascending index list against the oracle, bit for bit."""
    import torch
    rng = W.rng_for(3, 77)
    ctx = nb.Context(n)
    act = torch.zeros(n, dtype=torch.int32, device="cuda")
    t = rng.integers(0, 8, n).astype(np.float64) * 2.0**-6
    dt = 2.0 ** -rng.integers(3, 9, n).astype(np.float64)
    cases = []
    few = np.unique(np.concatenate([[0, n - 1], rng.integers(0, n, 13)]))
    cases.append(few)
    cases.append(np.arange(0, n, 2))
    lo = n // 3
    cases.append(np.arange(lo, min(n, lo + 5000)))
    cases.append(np.arange(n))
    for k, due in enumerate(cases):
        tt, dd = t.copy(), dt.copy()
        tt += 1.0  # nobody else is due before the chosen block
        tt[due] = 0.5
        dd[due] = 2.0**-7
        tn, oidx = O.next_block(tt, dd)
        assert tn == 0.5 + 2.0**-7 and np.array_equal(oidx, due.astype(np.int32))
        act.fill_(-1)
        gtn, gna = ctx.next_block(n, U.dev(tt), U.dev(dd), act)
        assert gtn == tn and gna == oidx.shape[0], (n, k, gtn, gna)
        assert np.array_equal(act[:gna].cpu().numpy(), oidx), (n, k)
    ctx.close()


@pytest.mark.parametrize("order", [4, 6, 8])
def test_block_integration_vs_oracle(nb, O, order):
    """Scheduler end to end on a small cluster with a central BH: same block sequence (bit-exact membership while
    the trajectories agree) and x, v close to the oracle's own integration after a few dozen blocks."""
    import torch
    from oracle import integrate as OI
    from paper_1312_1789_b200.scheduler import Integrator
    c = W.cluster(5, 513)
    eps2 = 1e-6
    DTMAX = 2.0**-6  # every particle is synchronised at t = 1/64
    so = OI.bootstrap(c["m"], c["x"], c["v"], order, eps2, dt_max=DTMAX)
    CRIT = 4 if order >= 6 else 0  # R8b on both sides
    g = Integrator(c["m"], c["x"], c["v"], order, eps2, dt_max=DTMAX, dt_criterion_order=CRIT)
    g.bootstrap()
    torch.cuda.synchronize()
    # bootstrap forces within tolerance; the first time steps may differ only where dt_crit sits on a power of two
    assert U.rel_vec(g.D[0].cpu().numpy(), so.D[0]) < 1e-5
    assert U.rel_vec(g.D[1].cpu().numpy(), so.D[1]) < 1e-4
    same = np.mean(g.dt.cpu().numpy() == so.dt)
    assert same > 0.98
    # lock-step: before every block the GPU state is re-synchronised to the oracle's, so the selection (indices,
    # block membership, t_next) must agree bit for bit and the corrected rows to mixed-precision accuracy
    def sync():
        for k in range(8):
            g.D[k].copy_(U.dev(so.D[k]))
        for dst, src in ((g.t, so.t), (g.dt, so.dt), (g.x, so.x), (g.v, so.v), (g.pot, so.pot)):
            dst.copy_(U.dev(src))
    agree = []
    for b in range(40):
        if float(np.min(so.t + so.dt)) > DTMAX:
            break
        sync()
        h_old = so.dt.copy()
        tn_o, idx_o = OI.block_step(so, eps2, 0.1, 2.0**-30, DTMAX, crit_order=CRIT)
        tn_g, na_g = g.block_step()
        assert tn_g == tn_o and na_g == idx_o.shape[0], "block %d differs" % b
        assert np.array_equal(g.active[:na_g].cpu().numpy(), idx_o)
        assert np.array_equal(g.t.cpu().numpy(), so.t)
        # one corrector step from identical states: the derived per-particle bound (gpu_util.corrector_bounds: BJ's
        # force tolerances carried through the corrector's coefficients with each particle's own h and derivatives)
        gx, gv = g.x.cpu().numpy(), g.v.cpu().numpy()
        U.check_corrected(order, idx_o, h_old[idx_o], gx, gv, so.x, so.v, so.D)
        rest = np.setdiff1d(np.arange(so.n), idx_o)
        assert np.array_equal(gx[rest], so.x[rest]) and np.array_equal(gv[rest], so.v[rest])  # inactive rows untouched
        agree.append(np.mean(g.dt.cpu().numpy()[idx_o] == so.dt[idx_o]))
        gdt = g.dt.cpu().numpy()[idx_o]
        # every GPU step is a valid block step: power of two, in range, commensurate with the block time
        assert np.all(np.frexp(gdt)[0] == 0.5) and np.all(gdt >= 2.0**-30) and np.all(gdt <= DTMAX)
        assert np.all(np.fmod(tn_o, gdt) == 0.0)
    # The step is a DECISION taken from a^(K..2K-1), which the corrector interpolates from differences of forces
    # divided by h^k: identical inputs give identical steps (test_correct_bit_exact); against the fp64 oracle the
    # mixed-precision forces move a decision only where dt_crit sits next to a power of two (R8b criterion).
    assert len(agree) >= 10 and np.mean(agree) > 0.9, (len(agree), np.mean(agree))
    # free-running: both integrate on their own to t = 1/64; trajectories stay close
    sync()
    OI.integrate(so, DTMAX, eps2, 0.1, 2.0**-30, DTMAX, crit_order=CRIT)
    g.integrate(DTMAX)
    torch.cuda.synchronize()
    assert np.all(so.t == DTMAX) and bool((g.t == DTMAX).all())
    assert np.max(np.abs(g.x.cpu().numpy() - so.x)) < 1e-7
    assert np.max(np.abs(g.v.cpu().numpy() - so.v)) < 1e-5


def test_energy_conservation_gpu(nb):
    """Short 6th-order block integration of a 1024-body Plummer sphere: |dE/E| small (invariant, no oracle)."""
    from paper_1312_1789_b200.scheduler import Integrator
    c = W.cluster(1)
    g = Integrator(c["m"], c["x"], c["v"], 6, 1e-4, dt_max=2.0**-5, dt_min=2.0**-20)
    assert g.dt_criterion_order == 4  # R8b default for p >= 6
    g.bootstrap()
    e0 = g.energy()
    g.integrate(2.0**-3)
    assert g.time == 2.0**-3 and bool((g.t == 2.0**-3).all())
    e1 = g.energy()
    assert abs(e0 + 0.25) < 0.03
    assert abs((e1 - e0) / e0) < 1e-6


def test_error_codes(nb):
    import torch
    ctx = nb.Context(100)
    z = U.zeros(100, 3)
    z1 = U.zeros(100)
    idx = torch.arange(100, dtype=torch.int32, device="cuda")
    with pytest.raises(nb.NBodyError) as e:
        ctx.force(idx, 10, 4, 1e-4, z, z, None, None, z1)
    assert e.value.code == nb.ESTATE  # force before predict
    with pytest.raises(nb.NBodyError) as e:
        ctx.predict(101, 0.0, 4, z1, z1, z, z, [z, z])
    assert e.value.code == nb.EINVAL  # n > capacity
    with pytest.raises(nb.NBodyError) as e:
        ctx.predict(100, 0.0, 5, z1, z1, z, z, [z, z])
    assert e.value.code == nb.EINVAL  # order
    with pytest.raises(nb.NBodyError) as e:
        ctx.predict(100, 0.0, 6, z1, z1, z, z, [z, z])
    assert e.value.code == nb.EINVAL  # missing D_2, D_3
    ctx.predict(100, 0.0, 4, z1, z1, z, z, [z, z])
    with pytest.raises(nb.NBodyError) as e:
        ctx.force(idx, 10, 6, 1e-4, z, z, z, None, z1)
    assert e.value.code == nb.ESTATE  # order above the predict's
    with pytest.raises(nb.NBodyError) as e:
        ctx.force(idx, 10, 4, -1.0, z, z, None, None, z1)
    assert e.value.code == nb.EINVAL
    with pytest.raises(nb.NBodyError) as e:
        ctx.force(idx, 101, 4, 1e-4, z, z, None, None, z1)
    assert e.value.code == nb.EINVAL
    ctx.force(idx, 0, 4, 1e-4, None, None, None, None, None)  # n_act == 0: no-op
    with pytest.raises(nb.NBodyError) as e:
        ctx.correct(idx, 10, 4, 0.1, 0.1, 0.3, 0.5, z1, z1, z, z, [z] * 4, z1, z, z, None, None, z1)
    assert e.value.code == nb.EINVAL  # dt_min not a power of two
    with pytest.raises(nb.NBodyError):
        ctx.set_option("no_such_option", 1)
    assert nb.strerror(nb.EINVAL) == "invalid argument" and nb.strerror(12345).startswith("unknown")
    ctx.close()


def test_force_host_matches_device_path(nb, O):
    """Host-buffer entry point = same kernels: bit-identical to the device-pointer calls, and within tolerance
    of the oracle."""
    c = W.cluster(3, 2500)
    n, order = c["n"], 6
    D = U.oracle_bootstrap_derivs(c, 6)
    t, dt = W.predictor_times(c["x"])
    t_now = 2.0**-10
    idx = W.active_list(n, 700, W.rng_for(3, 4))
    ctx = nb.Context(n)
    dev_out = U.gpu_force(ctx, n, order, c["eps2"], t_now, t, c["m"], c["x"], c["v"], D, idx)
    na = idx.shape[0]
    acc, jerk, snap, pot = np.zeros((na, 3)), np.zeros((na, 3)), np.zeros((na, 3)), np.zeros(na)
    up, down = ctx.force_host(n, t_now, order, t, c["m"], c["x"], c["v"], D[:4], idx, na, c["eps2"], acc, jerk, snap,
                              None, pot)
    assert up == 8 * n * (2 + 6 + 12) + 4 * na and down == 8 * na * 10
    assert np.array_equal(acc, dev_out[0]) and np.array_equal(jerk, dev_out[1])
    assert np.array_equal(snap, dev_out[2]) and np.array_equal(pot, dev_out[4])
    xp, vp, ap, jp = O.predict(t_now, order, t, c["x"], c["v"], D)
    ref = O.force(c["m"], xp, vp, ap, jp, idx, order, c["eps2"])
    U.check_force((acc, jerk, snap, None, pot), ref, order, "force_host")
    ctx.close()


def test_correct_step_rejection_bit_exact(nb, O):
    """R14 (oracle c-9b): with a small eta many end-point criteria ask for dt <= h/4; those particles must keep their
    whole state except dt = h/4, bit for bit as in the oracle, and the device counter equals the oracle's count."""
    import torch
    n, order = 3001, 8
    c, D, t, dt = _state(3, n, order)
    t_now = 2.0**-10
    idx = W.active_list(n, 1500, W.rng_for(3, 22))
    xp, vp, ap, jp = O.predict(t_now, order, t, c["x"], c["v"], D)
    f = O.force(c["m"], xp, vp, ap, jp, idx, order, c["eps2"])
    for R, eta in ((4, 0.004), (2, 0.02), (16, 0.001)):
        ot, odt, ox, ov, oD, op = t.copy(), dt.copy(), c["x"].copy(), c["v"].copy(), [d.copy() for d in D], np.zeros(n)
        nrej = O.correct(idx, order, t_now, eta, 2.0**-30, 2.0**-4, ot, odt, ox, ov, oD, op, *f, reject_ratio=R)
        assert 0 < nrej < idx.shape[0]
        ctx = nb.Context(n)
        ctx.set_option("step_reject_ratio", R)
        gt, gdt, gx, gv, gD, gp = U.dev(t), U.dev(dt), U.dev(c["x"]), U.dev(c["v"]), [U.dev(d) for d in D], U.zeros(n)
        ctx.correct(U.dev(idx), idx.shape[0], order, t_now, eta, 2.0**-30, 2.0**-4, gt, gdt, gx, gv, gD, gp,
                    *[U.dev(a) for a in f])
        assert ctx.rejected_steps(reset=True) == nrej and ctx.rejected_steps() == 0
        for a, b in ((gt, ot), (gdt, odt), (gx, ox), (gv, ov), (gp, op)):
            assert np.array_equal(a.cpu().numpy(), b)
        for k in range(8):
            assert np.array_equal(gD[k].cpu().numpy(), oD[k])
        rej = idx[ot[idx] != t_now]
        assert rej.shape[0] == nrej and np.all(odt[rej] == dt[rej] / R)
        ctx.close()
    with pytest.raises(nb.NBodyError):
        nb.Context(4).set_option("step_reject_ratio", 3)


@pytest.mark.parametrize("order", [6, 8])
def test_flyby_step_rejection_gpu(nb, order):
    """The oracle's fly-by pin on the CUDA path (closest approach on the end point of a long first step): without R14
    the energy error is astronomic, with step_reject_ratio = 4 the step is refused and redone on shorter steps --
    through block times that run BACKWARDS for the refused particles -- and the device-driven run reproduces the
    host-driven one bit for bit."""
    import torch
    from paper_1312_1789_b200.scheduler import Integrator
    h0 = 2.0**-4
    m = np.array([5e-4, 5e-4])
    x = np.array([[-h0 / 2, 5e-4, 0.0], [h0 / 2, -5e-4, 0.0]])
    v = np.array([[0.5, 0.0, 0.0], [-0.5, 0.0, 0.0]])

    def energy(g):
        xx, vv = g.x.cpu().numpy(), g.v.cpu().numpy()
        return 0.5 * np.sum(m * np.sum(vv * vv, axis=1)) - m[0] * m[1] / np.linalg.norm(xx[0] - xx[1])

    out = {}
    for R, driver in ((0, "host"), (4, "host"), (4, "device")):
        g = Integrator(m, x, v, order, 0.0, dt_min=2.0**-40, dt_max=h0, step_reject_ratio=R)
        g.bootstrap(fixed_dt=h0)
        e0 = energy(g)
        if driver == "host":
            g.integrate(2 * h0)
            rej = g.ctx.rejected_steps()
        else:
            r = g.run(2 * h0)
            rej = r["rejected"]
        torch.cuda.synchronize()
        assert bool((g.t == 2 * h0).all())
        out[(R, driver)] = (abs((energy(g) - e0) / e0), rej, g.blocks, g.x.cpu().numpy(), g.v.cpu().numpy())
    assert out[(0, "host")][0] > 1e3 and out[(0, "host")][1] == 0
    assert out[(4, "host")][0] < 1e-5 and out[(4, "host")][1] >= 1
    a, b = out[(4, "host")], out[(4, "device")]
    assert a[1] == b[1] and a[2] == b[2] and np.array_equal(a[3], b[3]) and np.array_equal(a[4], b[4])
    ang = np.degrees(np.arctan2(a[4][0][1], a[4][0][0]))
    assert abs(abs(ang) - 90.0) < 2.5


@pytest.mark.parametrize("order", [4, 6, 8])
def test_pec2_block_step_vs_oracle(nb, order):
    """N4 P(EC)^2 on the CUDA path against the oracle's P(EC)^2, lock-step from identical states: same membership, same
    times, corrected rows within the derived corrector bound; the step uses only C-ABI calls (predict, force, correct,
    pack_rows, unpack_rows)."""
    import torch
    from oracle import integrate as OI
    from paper_1312_1789_b200.scheduler import Integrator
    c = W.cluster(5, 513)
    eps2 = 1e-6
    DTMAX = 2.0**-6
    so = OI.bootstrap(c["m"], c["x"], c["v"], order, eps2, dt_max=DTMAX)
    g = Integrator(c["m"], c["x"], c["v"], order, eps2, dt_max=DTMAX)
    for b in range(25):
        for k in range(8):
            g.D[k].copy_(U.dev(so.D[k]))
        for dst, src in ((g.t, so.t), (g.dt, so.dt), (g.x, so.x), (g.v, so.v), (g.pot, so.pot)):
            dst.copy_(U.dev(src))
        h_old = so.dt.copy()
        tn_o, idx_o = OI.block_step(so, eps2, 0.1, 2.0**-30, DTMAX, n_iter=2)
        tn_g, na_g = g.block_step(n_iter=2)
        torch.cuda.synchronize()
        assert tn_g == tn_o and na_g == idx_o.shape[0]
        assert np.array_equal(g.active[:na_g].cpu().numpy(), idx_o)
        assert np.array_equal(g.t.cpu().numpy(), so.t)
        # two evaluations: the second force sees the first corrector's (slightly different) x1, v1, so allow twice the bound
        bx, bv = U.corrector_bounds(order, h_old[idx_o], [d[idx_o] for d in so.D])
        ex = np.linalg.norm(g.x.cpu().numpy()[idx_o] - so.x[idx_o], axis=1)
        ev = np.linalg.norm(g.v.cpu().numpy()[idx_o] - so.v[idx_o], axis=1)
        assert np.all(ex <= 2 * bx + 1e-15) and np.all(ev <= 2 * bv + 1e-15)
    # energy behaviour on the GPU: Kepler ellipse, shared step, P(EC)^1 drifts, P(EC)^2 does not
    m = np.array([0.5, 0.5])
    x = np.array([[0.25, 0, 0], [-0.25, 0, 0]])
    v = np.array([[0, np.sqrt(3) / 2, 0], [0, -np.sqrt(3) / 2, 0]])

    def en(g):
        xx, vv = g.x.cpu().numpy(), g.v.cpu().numpy()
        return 0.5 * np.sum(m * np.sum(vv * vv, axis=1)) - 0.25 / np.linalg.norm(xx[0] - xx[1])

    err = {}
    for n_iter in (1, 2):
        g = Integrator(m, x, v, 4, 0.0, dt_min=2.0**-5, dt_max=2.0**-5)
        g.bootstrap(fixed_dt=2.0**-5)
        e0 = en(g)
        g.integrate(64.0, n_iter=n_iter)
        err[n_iter] = abs((en(g) - e0) / e0)
    assert err[2] < 0.5 * err[1], err


def test_corrector_order_limiter_bit_exact(nb, O):
    """R15 (oracle c-6b) on the CUDA path: same limited particles (count), same x1, v1, bit for bit; force inputs with a
    spike in the higher derivatives of every fifth particle (per derivative) so that all truncation orders occur."""
    import torch
    n = 3001
    for order in (4, 6, 8):
        c, D, t, dt = _state(3, n, order)
        t_now = 2.0**-10
        idx = W.active_list(n, 1500, W.rng_for(3, 23))
        xp, vp, ap, jp = O.predict(t_now, order, t, c["x"], c["v"], D)
        f = [None if a is None else a.copy() for a in O.force(c["m"], xp, vp, ap, jp, idx, order, c["eps2"])]
        for k in range(1, order // 2):  # spikes: term k+1 of particles k, k+5, ... grows past term k
            f[k][k::5] *= 1e9
        f[0][0::7] *= 50.0  # acceleration spikes: level 0 (predictor-only step)
        cnt = {}
        ot, odt, ox, ov, oD, op = t.copy(), dt.copy(), c["x"].copy(), c["v"].copy(), [d.copy() for d in D], np.zeros(n)
        O.correct(idx, order, t_now, 0.1, 2.0**-30, 2.0**-4, ot, odt, ox, ov, oD, op, *f, limit_order=1, counters=cnt)
        assert 0 < cnt["limited"] < idx.shape[0]
        ctx = nb.Context(n)
        ctx.set_option("corrector_order_limit", 1)
        gt, gdt, gx, gv, gD, gp = U.dev(t), U.dev(dt), U.dev(c["x"]), U.dev(c["v"]), [U.dev(d) for d in D], U.zeros(n)
        ctx.correct(U.dev(idx), idx.shape[0], order, t_now, 0.1, 2.0**-30, 2.0**-4, gt, gdt, gx, gv, gD, gp,
                    *[None if a is None else U.dev(a) for a in f])
        assert ctx.step_counters() == (0, cnt["limited"])
        for a, b in ((gt, ot), (gdt, odt), (gx, ox), (gv, ov), (gp, op)):
            assert np.array_equal(a.cpu().numpy(), b)
        for k in range(8):
            assert np.array_equal(gD[k].cpu().numpy(), oD[k])
        ctx.close()
