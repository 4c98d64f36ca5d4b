"""Thin host block scheduler ("individual hierarchically block time-steps").

Holds the fp64 SoA state as torch CUDA tensors (device memory only -- no torch arithmetic on the path) and drives
the C-ABI calls.  Two drivers over the same kernels: block_step / integrate call next_block -> predict -> force ->
correct per block (one host round trip per block); run hands whole runs of blocks to the device-driven step
(nbody_run_blocks: one CUDA graph per block step, the host looks in every 4 .. 64 blocks).  Bootstrap = DESIGN.md R9b
(SURVEY c-10).
"""
import numpy as np
import torch

from . import nbody


class Integrator:
    def __init__(self, m, x, v, order, eps2, eta=0.1, eta_s=0.01, dt_min=2.0**-30, dt_max=2.0**-4, device=0,
                 ctx=None, dt_criterion_order=None, step_reject_ratio=0, corrector_order_limit=0):
        """dt_criterion_order: None / 0 = the library's automatic choice (pc = 4 for order >= 6, R8b: with
        fp32 pair arithmetic the order-p criterion of R8 is driven by rounding noise in the interpolated derivatives
        and collapses the steps); 4 | 6 | 8 = criterion order min(order, value) (value = order: R8)."""
        assert order in (4, 6, 8)
        self.order, self.eps2, self.eta, self.eta_s = order, float(eps2), float(eta), float(eta_s)
        self.dt_min, self.dt_max = float(dt_min), float(dt_max)
        self.dev = torch.device("cuda", device)
        n = int(np.asarray(m).shape[0])
        self.n = n
        self.ctx = ctx if ctx is not None else nbody.Context(n, device)
        self.ctx.set_option("dt_criterion_order", int(dt_criterion_order or 0))
        self.ctx.set_option("step_reject_ratio", int(step_reject_ratio))  # R14: 0 = the textbook scheme
        self.step_reject_ratio = int(step_reject_ratio)
        self.ctx.set_option("corrector_order_limit", int(corrector_order_limit))  # R15: 0 = off
        self.limited = 0
        self.rejected = 0
        self.dt_criterion_order = int(dt_criterion_order) if dt_criterion_order else (4 if order >= 6 else order)
        up = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).to(self.dev)
        self.m, self.x, self.v = up(m), up(x), up(v)
        z = lambda *s: torch.zeros(*s, dtype=torch.float64, device=self.dev)
        self.D = [z(n, 3) for _ in range(8)]
        self.pot = z(n)
        self.t = z(n)
        self.dt = z(n)
        # force outputs (active-list order) and the active list
        self.acc, self.jerk, self.snap, self.crk = z(n, 3), z(n, 3), z(n, 3), z(n, 3)
        self.fpot = z(n)
        self.active = torch.zeros(n, dtype=torch.int32, device=self.dev)
        self.all_idx = torch.arange(n, dtype=torch.int32, device=self.dev)
        self.time = 0.0
        self.blocks = 0
        self.pairs = 0

    # ---- R9b bootstrap: order-4 force at tau = 0, then (p >= 6) an order-8 force with those a, j ----
    def bootstrap(self, fixed_dt=None):
        c, n = self.ctx, self.n
        c.predict(n, 0.0, 4, self.t, self.m, self.x, self.v, self.D)
        c.force(self.all_idx, n, 4, self.eps2, self.acc, self.jerk, None, None, self.fpot)
        self.D[0].copy_(self.acc)
        self.D[1].copy_(self.jerk)
        self.pot.copy_(self.fpot)
        if self.order >= 6:
            # order-8 predictor at tau = 0 with D = (a, j, 0, 0, 0, 0) puts a, j into the j-store
            c.predict(n, 0.0, 8, self.t, self.m, self.x, self.v, self.D)
            c.force(self.all_idx, n, 8, self.eps2, self.acc, self.jerk, self.snap, self.crk, self.fpot)
            self.D[2].copy_(self.snap)
            self.D[3].copy_(self.crk)
        if fixed_dt is not None:
            self.dt.fill_(float(fixed_dt))
        else:
            c.initial_dt(n, self.D[0], self.D[1], self.eta_s, self.dt_min, self.dt_max, self.dt)

    def block_step(self, n_iter=1):
        """One host-driven block step.  n_iter > 1 = P(EC)^n (oracle/integrate.block_step): after the
        corrector the active particles' corrected state stands in for their prediction (the predictor gives exactly
        that at tau = 0), the force on them is evaluated again, their rows are put back to t0 (nbody_pack_rows /
        nbody_unpack_rows) and corrected again with the new force.  Same kernels, C-ABI calls only."""
        c, n, p = self.ctx, self.n, self.order
        snap, crk = (self.snap if p >= 6 else None), (self.crk if p >= 8 else None)
        t_next, n_act = c.next_block(n, self.t, self.dt, self.active)
        if n_iter > 1:
            if getattr(self, "_rows", None) is None:
                self._rows = torch.zeros(n, 9 + 3 * 8, dtype=torch.float64, device=self.dev)
            c.pack_rows(self.active, n_act, 8, self.t, self.dt, self.pot, self.x, self.v, self.D, self._rows)
        for it in range(n_iter):
            c.predict(n, t_next, p, self.t, self.m, self.x, self.v, self.D)
            c.force(self.active, n_act, p, self.eps2, self.acc, self.jerk, snap, crk, self.fpot)
            if it > 0:
                c.unpack_rows(self.active, n_act, 8, self.t, self.dt, self.pot, self.x, self.v, self.D, self._rows)
            if it < n_iter - 1 and self.step_reject_ratio:
                c.set_option("step_reject_ratio", 0)  # R14 applies to the last evaluation only
            c.correct(self.active, n_act, p, t_next, self.eta, self.dt_min, self.dt_max, self.t, self.dt, self.x, self.v,
                      self.D, self.pot, self.acc, self.jerk, snap, crk, self.fpot)
            if it < n_iter - 1 and self.step_reject_ratio:
                c.set_option("step_reject_ratio", self.step_reject_ratio)
        self.time = t_next
        self.blocks += 1
        self.pairs += n_act * n * n_iter
        return t_next, n_act

    def integrate(self, t_end, max_blocks=10**9, n_iter=1):
        """Host-driven integration: advance until the next block time would exceed t_end.  Returns the block-size
        histogram {floor(log2 n_act): count}."""
        hist = {}
        while self.blocks < max_blocks:
            # peek: the selection itself tells us t_next; stop when it passes t_end (block_step selects again: the
            # selection is idempotent)
            t_next, n_act = self.ctx.next_block(self.n, self.t, self.dt, self.active)
            if t_next > t_end:
                break
            self.block_step(n_iter)
            b = int(n_act).bit_length() - 1
            hist[b] = hist.get(b, 0) + 1
        return hist

    def run(self, t_end, max_blocks=10**12, max_n_act=None):
        """Device-driven integration (nbody_run_blocks): executes blocks while t_next <= t_end (and n_act <= max_n_act
        when given).  Returns the library's result dict; bit-identical to integrate()."""
        p = self.order
        r = self.ctx.run_blocks(self.n, p, self.eps2, self.eta, self.dt_min, self.dt_max, t_end, max_blocks,
                                self.n if max_n_act is None else max_n_act, self.t, self.dt, self.m, self.x, self.v,
                                self.D, self.pot, self.active, self.acc, self.jerk, self.snap if p >= 6 else None,
                                self.crk if p >= 8 else None, self.fpot)
        self.blocks += r["blocks"]
        self.pairs += r["pairs"]
        self.rejected += r["rejected"]
        self.limited += r["limited"]
        if r["blocks"]:
            self.time = float(self.t.max())  # diagnostic read (the last executed block's time)
        return r

    def energy(self):
        """E = Sum 1/2 m v^2 + 1/2 Sum m pot with pot from a synchronised order-4 all-active call (c-11).  The
        two dot products are diagnostics taken on the host in fp64."""
        assert bool((self.t == self.t[0]).all())
        t0 = float(self.t[0])
        self.ctx.predict(self.n, t0, 4, self.t, self.m, self.x, self.v, self.D)
        self.ctx.force(self.all_idx, self.n, 4, self.eps2, self.acc, self.jerk, None, None, self.fpot)
        m = self.m.cpu().numpy()
        v = self.v.cpu().numpy()
        pot = self.fpot.cpu().numpy()
        return float(0.5 * np.sum(m * np.sum(v * v, axis=1)) + 0.5 * np.sum(m * pot))
