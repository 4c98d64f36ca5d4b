"""Oracle-side block-time-step driver -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Plain restatement of the loop "pick block -> predict -> force -> correct -> new dt" (PAPER.md:15 abstract,
"individual hierarchically block time-steps with the high (4th, 6th and 8th) order Hermite integration
schemes"; section 2) on top of the fp64 C oracle.  The paper prints no algorithm; the steps are
SURVEY.md 8(c) items c-10 (bootstrap) and c-11 (block selection, energy).  Shares no code with the CUDA
package's scheduler.
"""
import numpy as np

from . import oracle as O


class State:
    """fp64 SoA state: t[n], dt[n], m[n], x,v[n][3], D[k] = a^(k) [n][3] for k = 0..order-1, pot[n]."""

    def __init__(self, m, x, v, order):
        n = m.shape[0]
        self.order = order
        self.m = np.ascontiguousarray(m, dtype=np.float64).copy()
        self.x = np.ascontiguousarray(x, dtype=np.float64).copy()
        self.v = np.ascontiguousarray(v, dtype=np.float64).copy()
        self.D = [np.zeros((n, 3)) for _ in range(8)]
        self.pot = np.zeros(n)
        self.t = np.zeros(n)
        self.dt = np.zeros(n)
        self.n = n


def bootstrap(m, x, v, order, eps2, eta_s=0.01, dt_min=2.0**-30, dt_max=2.0**-4, fixed_dt=None):
    """c-10: (i) order-4 force at tau = 0 -> a, j; (ii) for p >= 6 an order-8 force with those a, j as the
    particles' own a, j -> s, c (D_3 := c also for p = 6); higher D_k := 0; dt_i from eta_s |a|/|j|."""
    s = State(m, x, v, order)
    n = s.n
    idx = np.arange(n, dtype=np.int32)
    acc, jerk, _, _, pot = O.force(s.m, s.x, s.v, None, None, idx, 4, eps2)
    s.D[0][:], s.D[1][:], s.pot[:] = acc, jerk, pot
    if order >= 6:
        _, _, snap, crk, _ = O.force(s.m, s.x, s.v, acc, jerk, idx, 8, eps2)
        s.D[2][:], s.D[3][:] = snap, crk
    if fixed_dt is not None:
        s.dt[:] = fixed_dt
    else:
        s.dt[:] = O.initial_dt(acc, jerk, eta_s, dt_min, dt_max)
    return s


def block_step(s, eps2, eta, dt_min, dt_max, variant=0, crit_order=0, reject_ratio=0, n_iter=1, limit_order=0):
    """One block step (a-1 .. a-4).  Returns (t_next, active_idx).  With reject_ratio (c-9b) a rejected particle stays at
    its old time with a shorter step, so the next block time can lie before this one; s.rejected counts them.

    n_iter > 1 = P(EC)^n (the paper is silent): after the corrector, the active
    particles' corrected x1, v1 and their new a1, j1 (the first evaluation) stand in for their predicted values, the
    force on them is evaluated again, and the corrector is applied again FROM THE OLD STATE at t0 with the new force --
    n evaluations in all.  n -> infinity converges to the implicit (time-symmetric for a shared constant step) Hermite
    scheme."""
    p = s.order
    t_next, idx = O.next_block(s.t, s.dt)
    old = None
    if n_iter > 1:  # rows of the active particles at t0, restored before every re-correction
        old = dict(t=s.t[idx].copy(), dt=s.dt[idx].copy(), x=s.x[idx].copy(), v=s.v[idx].copy(), pot=s.pot[idx].copy(),
                   D=[d[idx].copy() for d in s.D])
    for it in range(n_iter):
        xp, vp, ap, jp = O.predict(t_next, p, s.t, s.x, s.v, s.D)  # corrected rows have t = t_next: tau = 0
        acc, jerk, snap, crk, pot = O.force(s.m, xp, vp, ap, jp, idx, p, eps2)
        if it > 0:
            s.t[idx], s.dt[idx], s.x[idx], s.v[idx], s.pot[idx] = old["t"], old["dt"], old["x"], old["v"], old["pot"]
            for k in range(8):
                s.D[k][idx] = old["D"][k]
        nrej = O.correct(idx, p, t_next, eta, dt_min, dt_max, s.t, s.dt, s.x, s.v, s.D, s.pot, acc, jerk, snap, crk,
                         pot, variant=variant, crit_order=crit_order,
                         reject_ratio=reject_ratio if it == n_iter - 1 else 0, limit_order=limit_order,
                         counters=s.__dict__.setdefault("counters", {}))
    s.rejected = getattr(s, "rejected", 0) + nrej
    return t_next, idx


def integrate(s, t_end, eps2, eta, dt_min, dt_max, variant=0, max_blocks=10**9, crit_order=0, reject_ratio=0, n_iter=1,
              limit_order=0):
    nb = 0
    pairs = 0
    while nb < max_blocks:
        if float(np.min(s.t + s.dt)) > t_end:
            break
        _, idx = block_step(s, eps2, eta, dt_min, dt_max, variant, crit_order, reject_ratio, n_iter, limit_order)
        nb += 1
        pairs += int(idx.shape[0]) * s.n * n_iter
    return nb, pairs


def total_energy(s, eps2):
    """c-11: E = Sum 1/2 m v^2 + 1/2 Sum m pot, pot from a synchronised order-4 all-active call.  All particles
    must sit at the same time."""
    assert np.all(s.t == s.t[0])
    idx = np.arange(s.n, dtype=np.int32)
    _, _, _, _, pot = O.force(s.m, s.x, s.v, None, None, idx, 4, eps2)
    k, w = O.energy(s.m, s.v, pot)
    return k + w
