"""-m gpu: the device-driven block step (nbody_run_blocks): K blocks replayed as CUDA graphs with
n_act known only on the device must be bit-identical -- t, dt, membership, state -- to K calls of the host-driven
path (nbody_next_block + predict + force + correct), which the other tests pin against the oracle; and the executed
blocks' membership is compared with the oracle's selection on identical inputs."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_1312_1789_b200 import workloads as W
import gpu_util as U


def _pair(config, n, order, **kw):
    from paper_1312_1789_b200.scheduler import Integrator
    import torch
    c = W.cluster(config, n)
    a = Integrator(c["m"], c["x"], c["v"], order, c["eps2"], **kw)
    b = Integrator(c["m"], c["x"], c["v"], order, c["eps2"], **kw)
    a.bootstrap()
    b.bootstrap()
    torch.cuda.synchronize()
    return c, a, b


def _same_state(a, b, order):
    for nm in ("t", "dt", "x", "v", "pot"):
        assert np.array_equal(getattr(a, nm).cpu().numpy(), getattr(b, nm).cpu().numpy()), nm
    for k in range(order):
        assert np.array_equal(a.D[k].cpu().numpy(), b.D[k].cpu().numpy()), "a^(%d)" % k


@pytest.mark.parametrize("order,use_graph,use_fused,n", [(4, 1, 1, 3001), (6, 1, 1, 3001), (8, 1, 1, 3001), (6, 0, 1, 3001),
                                                         (6, 1, 0, 3001), (8, 1, 1, 4096), (4, 0, 0, 2048)])
def test_run_blocks_bit_identical_to_host_driven_path(order, use_graph, use_fused, n):
    """use_fused = 1: blocks that fit one i-tile go through the fused step (N1: predict-in-force + last-CTA reduce and
    correct, raw state by TMA; n = 3001 also exercises the ragged last tile, n = 4096 all-TMA tiles), larger blocks
    through the general graph; use_fused = 0: every block through the general graph."""
    import torch
    K = 150
    c, a, b = _pair(5, n, order, dt_max=2.0**-5)
    sizes = []
    for _ in range(K):
        _, na = a.block_step()
        sizes.append(na)
    b.ctx.set_option("use_graph", use_graph)
    b.ctx.set_option("use_fused", use_fused)
    r = b.run(1.0, max_blocks=K)
    torch.cuda.synchronize()
    assert r["blocks"] == K and r["stop_reason"] == 3
    assert r["pairs"] == sum(sizes) * a.n
    hist = [0] * 40
    for s in sizes:
        hist[int(s).bit_length() - 1] += 1
    assert r["hist_log2"] == hist
    assert len(set(sizes)) > 5 and max(sizes) > 1024 and min(sizes) < 8  # every lane variant, both step flavours
    _same_state(a, b, order)
    # the block that stopped the run is the next block of the host-driven path
    tn, na = a.ctx.next_block(a.n, a.t, a.dt, a.active)
    assert r["t_next"] == tn and r["n_act_next"] == na
    assert np.array_equal(a.active[:na].cpu().numpy(), b.active[:na].cpu().numpy())


def test_fused_step_with_unaligned_state_arrays():
    """State arrays that are only 8-byte aligned cannot come in by TMA bulk copies (16-byte rule): the fused step reads
    them with plain loads instead; results stay bit-identical."""
    import torch
    order = 6
    c, a, b = _pair(3, 2048, order, dt_max=2.0**-6)

    def shifted(tn):
        flat = torch.zeros(tn.numel() + 1, dtype=torch.float64, device="cuda")
        view = flat[1:].view(tn.shape)
        view.copy_(tn)
        assert view.data_ptr() % 16 == 8
        return view

    b.x, b.v, b.t = shifted(b.x), shifted(b.v), shifted(b.t)
    b.D = [shifted(d) for d in b.D]
    for _ in range(60):
        a.block_step()
    r = b.run(1.0, max_blocks=60)
    assert r["blocks"] == 60
    _same_state(a, b, order)


def test_run_blocks_stop_reasons_and_resume():
    import torch
    order = 6
    c, a, b = _pair(3, 2049, order, dt_max=2.0**-6)
    T = 2.0**-6
    a.integrate(T)
    r = b.run(T)
    assert r["stop_reason"] == 1 and r["t_next"] > T and r["blocks"] == a.blocks
    assert bool((b.t == T).all())
    _same_state(a, b, order)
    # max_n_act: the run stops in front of the first block that is too large, state untouched by that block
    c, a, b = _pair(3, 2049, order, dt_max=2.0**-6)
    r = b.run(T, max_n_act=40)
    assert r["stop_reason"] == 2 and r["n_act_next"] > 40
    for _ in range(r["blocks"]):
        a.block_step()
    _same_state(a, b, order)
    tn, na = b.block_step()  # the host-driven path takes the big block; then the run resumes
    assert na == r["n_act_next"] and tn == r["t_next"]
    a.block_step()
    r2 = b.run(T, max_blocks=7)
    for _ in range(r2["blocks"]):
        a.block_step()
    _same_state(a, b, order)


def test_run_blocks_membership_matches_oracle_selection():
    """On identical inputs the blocks the device executes are the oracle's blocks (a-1, bit-exact membership): the
    particles whose time changed during a one-block run are exactly oracle_next_block's list."""
    import torch
    from oracle import oracle as O
    order = 4
    c, a, b = _pair(2, 4099, order, dt_max=2.0**-5)
    for _ in range(25):
        t0, dt0 = b.t.cpu().numpy().copy(), b.dt.cpu().numpy().copy()
        tn, idx = O.next_block(t0, dt0)
        r = b.run(1.0, max_blocks=1)
        assert r["blocks"] == 1
        t1 = b.t.cpu().numpy()
        changed = np.nonzero(t1 != t0)[0].astype(np.int32)
        assert np.array_equal(changed, idx) and np.all(t1[idx] == tn)


def test_run_blocks_errors():
    from paper_1312_1789_b200 import nbody
    c, a, b = _pair(1, 256, 4)
    with pytest.raises(nbody.NBodyError) as e:
        b.ctx.run_blocks(b.n, 4, b.eps2, 0.1, 0.3, 0.5, 1.0, 10, b.n, b.t, b.dt, b.m, b.x, b.v, b.D, b.pot, b.active,
                         b.acc, b.jerk, None, None, b.fpot)
    assert e.value.code == nbody.EINVAL  # dt_min not a power of two
    b.ctx.set_option("diff_mode", 1)
    with pytest.raises(nbody.NBodyError) as e:
        b.run(1.0, max_blocks=1)
    assert e.value.code == nbody.ESTATE
