"""Pins of the oracle's nearest-neighbour output (oracle_nearest, c-17 = DESIGN R16) against things other than itself:
a chain whose neighbours and distances have closed forms, an fp64 brute force on random points, the tie rule, the
precision in which the difference is formed, the degenerate sizes.  CPU only."""
import numpy as np

from oracle import oracle as O
from paper_1312_1789_b200 import workloads as W


def test_chain_with_closed_form_neighbours():
    """Particles at x_k = k^2 on a line (k = 0 .. 63, shuffled in memory): the gaps grow, so the nearest neighbour of
    k >= 1 is k - 1 at distance 2k - 1, and that of 0 is 1 at distance 1.  All values are exact in fp32."""
    k = np.arange(64)
    perm = W.rng_for(1, 90).permutation(64)  # memory slot s holds chain member perm[s]
    x = np.zeros((64, 3))
    x[:, 1] = (perm.astype(np.float64)) ** 2
    x[:, 0] = 7.0  # constant offsets drop out of the differences
    x[:, 2] = -3.0
    who, r2 = O.nearest(x, k.astype(np.int32))
    slot_of = np.argsort(perm)  # chain member -> memory slot
    for s in range(64):
        kk = perm[s]
        want = slot_of[1] if kk == 0 else slot_of[kk - 1]
        assert who[s] == want
        assert r2[s] == (1.0 if kk == 0 else float(2 * kk - 1) ** 2)


def test_against_fp64_brute_force():
    """Random cluster: the index equals numpy's fp64 argmin wherever the two smallest fp64 distances differ by more than
    fp32 rounding could bridge (they do for every particle here), and r2 is the fp64 value to fp32 accuracy.  Only a
    subset is active, in descending order: outputs follow the active list."""
    c = W.cluster(2, 700)
    x = c["x"]
    idx = np.arange(699, -1, -3).astype(np.int32)
    who, r2 = O.nearest(x, idx)
    d2 = ((x[None, :, :] - x[idx][:, None, :]) ** 2).sum(axis=2)
    d2[np.arange(idx.shape[0]), idx] = np.inf
    best = np.argmin(d2, axis=1)
    two = np.partition(d2, 1, axis=1)[:, :2]
    assert (two[:, 1] / two[:, 0] > 1.0 + 1e-5).all()  # no near-ties: the argmin is unique at fp32 accuracy
    assert np.array_equal(who, best.astype(np.int32))
    assert np.max(np.abs(r2 / two[:, 0] - 1.0)) < 3e-7  # three fp32 roundings
    assert np.all(r2 == r2.astype(np.float32))  # the stored value is an fp32 number


def test_ties_go_to_the_lowest_index():
    x = np.array([[0.0, 0.0, 0.0], [1.0, 0.0, 0.0], [-1.0, 0.0, 0.0], [0.0, 1.0, 0.0], [0.0, 0.0, -1.0]])
    who, r2 = O.nearest(x, np.arange(5, dtype=np.int32))
    assert who[0] == 1 and r2[0] == 1.0  # four neighbours at distance 1: the first in memory wins
    assert list(who[1:]) == [0, 0, 0, 0]
    x = x[::-1].copy()
    who, r2 = O.nearest(x, np.arange(5, dtype=np.int32))
    assert who[4] == 0 and r2[4] == 1.0


def test_difference_is_formed_in_fp64_then_rounded():
    """Two particles 2^-30 apart at x = 1000 (an fp32 position would swallow the offset: ulp_32(1000) = 2^-14), a third
    one 2^-20 away: the fp64 difference resolves both, r2 = 2^-60 exactly; a difference of fp32-rounded positions would
    give 0 for both and pick the wrong (lower-index) neighbour."""
    x = np.array([[1000.0 + 2.0**-20, 5.0, 5.0], [1000.0, 5.0, 5.0], [1000.0 + 2.0**-30, 5.0, 5.0]])
    who, r2 = O.nearest(x, np.arange(3, dtype=np.int32))
    assert list(who) == [2, 2, 1]
    assert r2[1] == 2.0**-60 and r2[2] == 2.0**-60
    assert r2[0] == float(np.float32(2.0**-20 - 2.0**-30)) ** 2  # (fl32(d))^2 is exact here (24-bit d, squared in fp32: check)
    # components are rounded one by one before the fp32 sum: a difference that is not an fp32 number
    x = np.array([[0.0, 0.0, 0.0], [1.0 + 2.0**-40, 0.0, 0.0]])
    who, r2 = O.nearest(x, np.arange(2, dtype=np.int32))
    assert r2[0] == 1.0 and r2[1] == 1.0


def test_degenerate_sizes():
    who, r2 = O.nearest(np.array([[1.0, 2.0, 3.0]]), np.array([0], dtype=np.int32))
    assert who[0] == -1 and np.isinf(r2[0])
    who, r2 = O.nearest(np.array([[1.0, 2.0, 3.0], [1.0, 2.0, 3.0]]), np.array([1, 0], dtype=np.int32))
    assert list(who) == [0, 1] and list(r2) == [0.0, 0.0]  # coincident particles: distance 0, still a neighbour
    who, r2 = O.nearest(np.zeros((4, 3)), np.array([], dtype=np.int32))
    assert who.shape == (0,) and r2.shape == (0,)
