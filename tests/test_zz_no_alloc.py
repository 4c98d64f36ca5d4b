"""-m gpu, collected last on purpose (the suite runs with pytest -x): nbody_force_static, the allocation-free variant of
nbody_force whose j-split scratch is a static device array inside libnbody.so (include/nbody.h).

Checked against the existing path (nbody_force, ctx-owned scratch) on the same predicted state: the two use the same
kernels and the same geometry rule, so the comparison is bit for bit (the determinism contract of nbody_force: a result
depends on the j-lane variant and the j-split count only) -- tighter than the BASELINE.json tolerances in gpu_util.TOL,
which are asserted as well.  Two calls in a row on one stream, of different size and order, so that the second one
runs on the first one's leftovers in the shared array; then the same pair again with the free device memory read
before and after (nothing may be allocated); then the documented rejection beyond the array's size."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_1312_1789_b200 import workloads as W
import gpu_util as U

N = 20011  # 79 j-tiles, ragged tail


def _outputs(n_act, order):
    out = [U.zeros(n_act, 3), U.zeros(n_act, 3), U.zeros(n_act, 3) if order >= 6 else None,
           U.zeros(n_act, 3) if order >= 8 else None, U.zeros(n_act)]
    for a in out:
        if a is not None:
            a.fill_(float("nan"))
    return out


def _same(got, ref, order, tag):
    names = ("acc", "jerk", "snap", "crackle", "pot")
    for name, a, b in zip(names, got, ref):
        if a is None:
            assert b is None
            continue
        a, b = a.cpu().numpy(), b.cpu().numpy()
        assert np.isfinite(a).all(), "%s %s: not fully written" % (tag, name)
        assert np.array_equal(a, b), "%s %s differs from nbody_force (max |d| = %.3e)" % (tag, name, np.abs(a - b).max())
    f = lambda a: None if a is None else a.cpu().numpy()
    U.check_force([f(a) for a in got], [f(a) for a in ref], order, tag)  # the tolerances the parity tests use


def test_force_static_matches_force_twice_in_a_row_without_allocating():
    import torch
    from paper_1312_1789_b200 import nbody as nb
    c = W.cluster(3, N)
    D = W.smooth_field_derivs(c, 6)
    t, _ = W.predictor_times(c["x"])
    t_now = 2.0**-10
    ctx = nb.Context(N)
    ctx.predict(N, t_now, 8, U.dev(t), U.dev(c["m"]), U.dev(c["x"]), U.dev(c["v"]), [U.dev(d) for d in D])
    ctx.force_static(None, 0, 8, c["eps2"], None, None, None, None, None)  # set-up call: resolves the array's address

    # (n_act, order): the largest block the limit guarantees (1024 at order 8: S x 13 x 1024 doubles), then a small
    # 4th-order block behind it that leaves most of the first call's partials in the array
    cases = [(1024, 8), (37, 4)]
    idx = [U.dev(W.active_list(N, na, W.rng_for(3, 40 + k))) for k, (na, _) in enumerate(cases)]
    ref, splits = [], []
    for (na, order), ix in zip(cases, idx):  # the existing path
        o = _outputs(na, order)
        ctx.force(ix, na, order, c["eps2"], *o)
        splits.append(ctx.last_force_geometry()["j_splits"])
        ref.append(o)
    torch.cuda.synchronize()
    assert min(splits) > 1, "both launches must be j-split (else the scratch is not exercised): %s" % splits
    need = [s * (3 * order // 2 + 1) * na * 8 for s, (na, order) in zip(splits, cases)]
    assert max(need) <= nb.FORCE_STATIC_SCRATCH_BYTES and need[0] > nb.FORCE_STATIC_SCRATCH_BYTES // 4

    for rep in range(2):
        got = [_outputs(na, order) for na, order in cases]
        if rep == 1:  # every kernel variant is loaded by now: nothing may change the free device memory from here on
            torch.cuda.synchronize()
            free0 = torch.cuda.mem_get_info()[0]
        for (na, order), ix, o in zip(cases, idx, got):  # two calls in a row on one stream, no synchronisation between
            ctx.force_static(ix, na, order, c["eps2"], *o)
            assert ctx.last_force_geometry()["j_splits"] == splits[cases.index((na, order))]
        torch.cuda.synchronize()
        if rep == 1:
            assert torch.cuda.mem_get_info()[0] == free0, "nbody_force_static changed the free device memory"
        for (na, order), o, r in zip(cases, got, ref):
            _same(o, r, order, "force_static rep %d n_act %d order %d" % (rep, na, order))

    # beyond the static array: a forced split of the all-active block (S x 13 x N x 8 bytes > 16 MiB) is refused with
    # its own code, launches nothing and leaves the outputs alone; nbody_force with the ctx scratch still takes it
    s_big = nb.FORCE_STATIC_SCRATCH_BYTES // (13 * N * 8) + 1
    ctx.set_option("force_split", s_big)
    all_idx = torch.arange(N, dtype=torch.int32, device="cuda")
    o = _outputs(N, 8)
    l0 = ctx.launch_count()
    with pytest.raises(nb.NBodyError) as e:
        ctx.force_static(all_idx, N, 8, c["eps2"], *o)
    assert e.value.code == nb.ESCRATCH and "NBODY_FORCE_STATIC_SCRATCH_BYTES" in str(e.value)
    assert ctx.launch_count() == l0
    torch.cuda.synchronize()
    assert all(bool(torch.isnan(a).all()) for a in o)
    ctx.force(all_idx, N, 8, c["eps2"], *o)
    r = o
    ctx.set_option("force_split", s_big - 1)  # the largest split that fits
    o = _outputs(N, 8)
    ctx.force_static(all_idx, N, 8, c["eps2"], *o)
    torch.cuda.synchronize()
    assert np.isfinite(o[0].cpu().numpy()).all()
    ctx.force(all_idx, N, 8, c["eps2"], *r)
    _same(o, r, 8, "force_static forced split %d" % (s_big - 1))
    ctx.close()
