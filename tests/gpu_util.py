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
