"""Multi-GPU plumbing of the block step (SURVEY.md 8(e); PAPER.md:43 "Both use MPI", :65 eq. (1) beta-term: one
exchange per block; NVLink 5 / NVSwitch through torch.distributed's NCCL backend).

i-sharding with a replicated state: every rank predicts all N, computes force + correct for its contiguous slice of
the sorted active list, then ONE all-gather of the corrected rows keeps the replicas identical.  Every rank passes
the size of the WHOLE block to the library ("geometry_n_act"), so the j-lane variant and the j-split -- the only
things the summation order of a particle depends on -- are those of the unsharded call and the sharded step
reproduces the single-GPU step bit for bit (tests/test_gpu_parallel.py).  Blocks smaller than REDUNDANT_BELOW are
computed redundantly by every rank with no collective; runs of such blocks go through the
device-driven step (nbody_run_blocks).

Only collectives, slicing and C-ABI calls live here (no method arithmetic).  On CUDA tensors the row records are
packed / unpacked by the library's kernels (nbody_pack_rows / nbody_unpack_rows: one gather, one all-gather, one
scatter per block); the torch-indexing variant below serves the gloo CPU tests of this plumbing only.

No scaling curve has been measured: this run has one GPU.
"""
import torch
import torch.distributed as dist

REDUNDANT_BELOW = 64  # blocks with fewer active particles are computed by every rank, no exchange


def shard_bounds(n_act: int, rank: int, world: int):
    """Contiguous slice [lo, hi) of the active list owned by `rank`: fixed chunks of ceil(n_act / world), the last
    non-empty one shorter.  With this layout the all-gathered buffer IS the record array of active[0 .. n_act) in
    order, so one scatter applies it."""
    chunk = (int(n_act) + int(world) - 1) // int(world)
    lo = min(rank * chunk, int(n_act))
    hi = min(lo + chunk, int(n_act))
    return lo, hi


def state_columns(order: int) -> int:
    """doubles per particle in the exchanged record: t, dt, pot, x[3], v[3], a^(0..order-1)[3]."""
    return 3 + 6 + 3 * order


def pack_rows(idx, t, dt, pot, x, v, D, order, out):
    """CPU plumbing (gloo tests): out[k] = record of particle idx[k] (idx: int64 tensor).  Returns out[:len(idx)]."""
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


def exchange_corrected(active, n_act, rank, world, t, dt, pot, x, v, D, order, group=None, ctx=None, force=False):
    """All-gather the rows each rank corrected (its slice of active[:n_act]) and apply them locally.  Returns the
    bytes this rank sent.  CUDA tensors need `ctx` (the library's pack / unpack kernels); CPU tensors (gloo tests)
    use torch indexing.  `force` runs the collective even for a single rank (tests of the NCCL path)."""
    if (world == 1 and not force) or n_act == 0:
        return 0
    chunk = (n_act + world - 1) // world
    ncol = state_columns(order)
    lo, hi = shard_bounds(n_act, rank, world)
    send = torch.zeros(chunk, ncol, dtype=torch.float64, device=t.device)
    recv = torch.empty(world * chunk, ncol, dtype=torch.float64, device=t.device)
    if t.is_cuda:
        if ctx is None:
            raise RuntimeError("exchange_corrected: CUDA tensors need the nbody Context (no torch fallback on the GPU path)")
        if hi > lo:
            ctx.pack_rows(active[lo:hi], hi - lo, order, t, dt, pot, x, v, D, send)
        dist.all_gather_into_tensor(recv, send, group=group)
        ctx.unpack_rows(active, n_act, order, t, dt, pot, x, v, D, recv)
    else:
        act64 = active[:n_act].to(torch.int64)
        if hi > lo:
            pack_rows(act64[lo:hi], t, dt, pot, x, v, D, order, send)
        dist.all_gather_into_tensor(recv, send, group=group)
        unpack_rows(act64, recv[:n_act], t, dt, pot, x, v, D, order)
    return (hi - lo) * ncol * 8


def sharded_block_step(integ, rank: int, world: int, group=None, force_exchange=False):
    """One block step of `integ` (scheduler.Integrator) with the force + corrector work i-sharded over `world`
    ranks.  Returns (t_next, n_act, exchanged_bytes)."""
    c, n, p = integ.ctx, integ.n, integ.order
    t_next, n_act = c.next_block(n, integ.t, integ.dt, integ.active)
    c.predict(n, t_next, p, integ.t, integ.m, integ.x, integ.v, integ.D)
    snap = integ.snap if p >= 6 else None
    crk = integ.crk if p >= 8 else None
    if n_act < REDUNDANT_BELOW and not force_exchange:  # small block: every rank computes all of it, no collective
        lo, hi, sent = 0, n_act, 0
    else:
        lo, hi = shard_bounds(n_act, rank, world)
    if hi > lo:
        act = integ.active[lo:hi]
        c.set_option("geometry_n_act", n_act)  # summation order of the unsharded call
        try:
            c.force(act, hi - lo, p, integ.eps2, integ.acc, integ.jerk, snap, crk, integ.fpot)
        finally:
            c.set_option("geometry_n_act", 0)
        c.correct(act, hi - lo, p, t_next, integ.eta, integ.dt_min, integ.dt_max, integ.t, integ.dt, integ.x, integ.v,
                  integ.D, integ.pot, integ.acc, integ.jerk, snap, crk, integ.fpot)
    if n_act >= REDUNDANT_BELOW or force_exchange:
        sent = exchange_corrected(integ.active, n_act, rank, world, integ.t, integ.dt, integ.pot, integ.x, integ.v,
                                  integ.D, p, group, ctx=c, force=force_exchange)
    integ.time = t_next
    integ.blocks += 1
    integ.pairs += n_act * n
    return t_next, n_act, sent


def sharded_run(integ, t_end, rank: int, world: int, group=None, max_blocks=10**12):
    """Integrate to t_end on `world` ranks: runs of small blocks go through the device-driven step on every rank
    (redundant, no collective, no host round trip per block); a block of REDUNDANT_BELOW or more particles is
    i-sharded with one all-gather.  Returns (blocks, exchanged_bytes)."""
    sent_total, blocks0 = 0, integ.blocks
    while integ.blocks - blocks0 < max_blocks:
        r = integ.run(t_end, max_blocks=max_blocks - (integ.blocks - blocks0),
                      max_n_act=(REDUNDANT_BELOW - 1) if world > 1 else None)
        if r["stop_reason"] != 2:
            break
        _, _, sent = sharded_block_step(integ, rank, world, group)
        sent_total += sent
    return integ.blocks - blocks0, sent_total
