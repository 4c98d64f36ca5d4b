"""Helpers shared by the -m gpu parity tests: state upload, oracle-side inputs, error norms.  No method arithmetic."""
import numpy as np

# BASELINE.json north_star tolerances: max over particles of |delta|/|ref| per vector, relative pot error
TOL = dict(acc=1e-5, jerk=1e-4, snap=1e-3, crackle=1e-2, pot=1e-6)


def rel_vec(a, ref):
    """max over particles of |a - ref| / |ref| (Euclidean norms per particle)."""
    num = np.linalg.norm(np.asarray(a) - ref, axis=1)
    den = np.linalg.norm(ref, axis=1)
    return float(np.max(num / den))


def rel_scal(a, ref):
    return float(np.max(np.abs(np.asarray(a) - ref) / np.abs(ref)))


def dev(a, dtype=None):
    import torch
    t = torch.from_numpy(np.ascontiguousarray(a))
    if dtype is not None:
        t = t.to(dtype)
    return t.cuda()


def zeros(*shape, dtype=None):
    import torch
    return torch.zeros(*shape, dtype=dtype or torch.float64, device="cuda")


def oracle_bootstrap_derivs(c, n_derivs):
    """Physically consistent Taylor coefficients D_0..D_3 at tau = 0 from the oracle's own bootstrap
    (DESIGN.md input recipe, SURVEY.md 8(d) "primary"); higher D_k := small smooth continuation so that the
    predictor exercises every Horner term.  Used at small N only."""
    from oracle import oracle as O
    n = c["n"]
    idx = np.arange(n, dtype=np.int32)
    acc, jerk, _, _, _ = O.force(c["m"], c["x"], c["v"], None, None, idx, 4, c["eps2"])
    _, _, snap, crk, _ = O.force(c["m"], c["x"], c["v"], acc, jerk, idx, 8, c["eps2"])
    D = [acc, jerk, snap, crk]
    om = np.linalg.norm(jerk, axis=1) / np.maximum(np.linalg.norm(acc, axis=1), 1e-300)
    while len(D) < n_derivs:
        D.append(np.ascontiguousarray(-D[-2] * (om * om)[:, None]))
    return [np.ascontiguousarray(d) for d in D[:n_derivs]]


def gpu_force(ctx, n, order, eps2, t_now, t, m, x, v, D, active):
    """predict + force through the C ABI; returns numpy acc, jerk, snap, crackle, pot (None where undefined)."""
    import torch
    na = int(active.shape[0])
    dD = [dev(d) for d in D[: order - 2]]
    ctx.predict(n, t_now, order, dev(t), dev(m), dev(x), dev(v), dD)
    acc, jerk, pot = zeros(na, 3), zeros(na, 3), zeros(na)
    snap = zeros(na, 3) if order >= 6 else None
    crk = zeros(na, 3) if order >= 8 else None
    for a in (acc, jerk, pot, snap, crk):
        if a is not None:
            a.fill_(float("nan"))
    ctx.force(dev(active.astype(np.int32)), na, order, eps2, acc, jerk, snap, crk, pot)
    torch.cuda.synchronize()
    f = lambda a: None if a is None else a.cpu().numpy()
    return f(acc), f(jerk), f(snap), f(crk), f(pot)


def check_force(got, ref, order, tag=""):
    acc, jerk, snap, crk, pot = got
    racc, rjerk, rsnap, rcrk, rpot = ref
    errs = dict(acc=rel_vec(acc, racc), jerk=rel_vec(jerk, rjerk), pot=rel_scal(pot, rpot))
    if order >= 6:
        errs["snap"] = rel_vec(snap, rsnap)
    if order >= 8:
        errs["crackle"] = rel_vec(crk, rcrk)
    for k, e in errs.items():
        assert np.isfinite(e) and e <= TOL[k], "%s %s rel err %.3e > %.1e (all: %s)" % (tag, k, e, TOL[k], errs)
    return errs


def conditioning_report(got, ref, absn, radius, order):
    """Per quantity: max and 99.9th-percentile relative error over the sampled particles and, for the worst particle,
    its radius and kappa = Sum_j |term| / |Sum_j term|.  absn = oracle force_abs output."""
    names = ["acc", "jerk", "snap", "crackle"][: order // 2]
    rep = {}
    for k, nm in enumerate(names):
        den = np.linalg.norm(ref[k], axis=1)
        err = np.linalg.norm(np.asarray(got[k]) - ref[k], axis=1) / den
        kap = absn[k] / den
        w = int(np.argmax(err))
        rep[nm] = dict(max=float(err[w]), p999=float(np.percentile(err, 99.9)), median=float(np.median(err)),
                       worst_radius=float(radius[w]), worst_kappa=float(kap[w]), kappa_max=float(kap.max()),
                       kappa_median=float(np.median(kap)), tol=TOL[nm])
    e = np.abs(np.asarray(got[4]) - ref[4]) / np.abs(ref[4])
    w = int(np.argmax(e))
    rep["pot"] = dict(max=float(e[w]), p999=float(np.percentile(e, 99.9)), median=float(np.median(e)),
                      worst_radius=float(radius[w]), tol=TOL["pot"])
    return rep


def corrector_bounds(order, h, D1):
    """Per-particle bounds on |x_gpu - x_oracle| and |v_gpu - v_oracle| after ONE corrector step (R6) taken from
    identical states: the two sides differ only in the force-call values at t1, by at most BASELINE.json's tolerances
    (|da| <= 1e-5 |a1|, |dj| <= 1e-4 |j1|, |ds| <= 1e-3 |s1|, |dc| <= 1e-2 |c1|), which the corrector's own
    coefficients carry into v1 and x1:
        p=4: dv <= h/2 da + h^2/12 dj                        dx <= h/2 dv + h^2/12 da
        p=6: dv <= h/2 da + h^2/10 dj + h^3/120 ds           dx <= h/2 dv + h^2/10 da + h^3/120 dj
        p=8: dv <= h/2 da + 3h^2/28 dj + h^3/84 ds + h^4/1680 dc
             dx <= h/2 dv + 3h^2/28 da + h^3/84 dj + h^4/1680 ds
    h: step of each particle, D1[k]: the oracle's a^(k)(t1) rows of the same particles.  A few ulp of the state are
    added for the rounding of the sums themselves."""
    nr = [np.linalg.norm(D1[k], axis=1) for k in range(order // 2)]
    d = [TOL["acc"] * nr[0], TOL["jerk"] * nr[1]]
    if order >= 6:
        d.append(TOL["snap"] * nr[2])
    if order >= 8:
        d.append(TOL["crackle"] * nr[3])
    c = {4: [0.5, 1 / 12.0], 6: [0.5, 0.1, 1 / 120.0], 8: [0.5, 3 / 28.0, 1 / 84.0, 1 / 1680.0]}[order]
    dv = sum(c[k] * h ** (k + 1) * d[k] for k in range(order // 2))
    dx = 0.5 * h * dv + sum(c[k] * h ** (k + 1) * d[k - 1] for k in range(1, order // 2))
    return dx, dv


def check_corrected(order, idx, h, x_g, v_g, x_o, v_o, D1_o):
    """Assert the corrected rows `idx` agree within corrector_bounds (+ 8 ulp of the value)."""
    bx, bv = corrector_bounds(order, h, [d[idx] for d in D1_o])
    ex = np.linalg.norm(x_g[idx] - x_o[idx], axis=1)
    ev = np.linalg.norm(v_g[idx] - v_o[idx], axis=1)
    ulp = 8 * 2.2e-16
    okx = ex <= bx + ulp * np.linalg.norm(x_o[idx], axis=1)
    okv = ev <= bv + ulp * np.linalg.norm(v_o[idx], axis=1)
    assert np.all(okx), ("x", float(np.max(ex / (bx + 1e-300))))
    assert np.all(okv), ("v", float(np.max(ev / (bv + 1e-300))))
    return float(np.max(ex / (bx + 1e-300))), float(np.max(ev / (bv + 1e-300)))
