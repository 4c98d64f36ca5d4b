"""Multi-GPU plumbing of the block step (eq. (1) beta-term: one exchange per block).

i-sharding with a replicated state: every rank predicts all N, computes force + correct for its contiguous slice of
the sorted active list, then ONE all-gather of the corrected rows keeps the replicas identical.  The per-particle
summation order does not depend on the partition, so the result is bit-identical to the single-GPU step.
Only torch.distributed collectives and index copies live here (no method arithmetic); the gloo CPU tests cover it.
"""
import torch
import torch.distributed as dist


def shard_bounds(n_act: int, rank: int, world: int):
    """Contiguous slice [lo, hi) of the active list owned by `rank`; sizes differ by at most one."""
    base, rem = divmod(int(n_act), int(world))
    lo = rank * base + min(rank, rem)
    hi = lo + base + (1 if rank < rem else 0)
    return lo, hi


def state_columns(order: int) -> int:
    """doubles per particle in the exchanged record: t, dt, pot, x[3], v[3], a^(0..order-1)[3]."""
    return 3 + 6 + 3 * order


def pack_rows(idx, t, dt, pot, x, v, D, order, out):
    """out[k] = record of particle idx[k] (idx: int64 tensor).  Returns out[:len(idx)]."""
    k = idx.shape[0]
    o = out[:k]
    o[:, 0] = t[idx]
    o[:, 1] = dt[idx]
    o[:, 2] = pot[idx]
    o[:, 3:6] = x[idx]
    o[:, 6:9] = v[idx]
    for d in range(order):
        o[:, 9 + 3 * d: 12 + 3 * d] = D[d][idx]
    return o


def unpack_rows(idx, rec, t, dt, pot, x, v, D, order):
    t[idx] = rec[:, 0]
    dt[idx] = rec[:, 1]
    pot[idx] = rec[:, 2]
    x[idx] = rec[:, 3:6]
    v[idx] = rec[:, 6:9]
    for d in range(order):
        D[d][idx] = rec[:, 9 + 3 * d: 12 + 3 * d]


def exchange_corrected(active, n_act, rank, world, t, dt, pot, x, v, D, order, group=None):
    """All-gather the rows each rank corrected (its slice of active[:n_act]) and apply the others' rows locally.
    Returns the bytes this rank sent.  Works on CPU (gloo) and CUDA (nccl) tensors alike."""
    if world == 1 or n_act == 0:
        return 0
    chunk = (n_act + world - 1) // world
    ncol = state_columns(order)
    send = torch.zeros(chunk, ncol, dtype=torch.float64, device=t.device)
    lo, hi = shard_bounds(n_act, rank, world)
    act64 = active[:n_act].to(torch.int64)
    if hi > lo:
        pack_rows(act64[lo:hi], t, dt, pot, x, v, D, order, send)
    recv = torch.empty(world * chunk, ncol, dtype=torch.float64, device=t.device)
    dist.all_gather_into_tensor(recv, send, group=group)
    for r in range(world):
        if r == rank:
            continue
        rlo, rhi = shard_bounds(n_act, r, world)
        if rhi > rlo:
            unpack_rows(act64[rlo:rhi], recv[r * chunk: r * chunk + (rhi - rlo)], t, dt, pot, x, v, D, order)
    return (hi - lo) * ncol * 8


def sharded_block_step(integ, rank: int, world: int, group=None):
    """One block step of `integ` (scheduler.Integrator) with the force + corrector work i-sharded over `world`
    ranks.  Returns (t_next, n_act, exchanged_bytes)."""
    c, n, p = integ.ctx, integ.n, integ.order
    t_next, n_act = c.next_block(n, integ.t, integ.dt, integ.active)
    c.predict(n, t_next, p, integ.t, integ.m, integ.x, integ.v, integ.D)
    lo, hi = shard_bounds(n_act, rank, world)
    if hi > lo:
        act = integ.active[lo:hi]
        snap = integ.snap if p >= 6 else None
        crk = integ.crk if p >= 8 else None
        c.force(act, hi - lo, p, integ.eps2, integ.acc, integ.jerk, snap, crk, integ.fpot)
        c.correct(act, hi - lo, p, t_next, integ.eta, integ.dt_min, integ.dt_max, integ.t, integ.dt, integ.x, integ.v,
                  integ.D, integ.pot, integ.acc, integ.jerk, snap, crk, integ.fpot)
    sent = exchange_corrected(integ.active, n_act, rank, world, integ.t, integ.dt, integ.pot, integ.x, integ.v,
                              integ.D, p, group)
    integ.time = t_next
    integ.blocks += 1
    integ.pairs += n_act * n
    return t_next, n_act, sent
