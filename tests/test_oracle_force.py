"""Pins of the CPU oracle's force with derivatives (SURVEY.md 8(c) c-1 .. c-4) against things other than itself:
the worked example W3 (40-digit mpmath, tests/golden/w3.txt), mpmath differentiation of the plain softened
acceleration on random tiny systems, the circular two-body closed form, momentum-like invariants Sum m a^(k) = 0,
the Plummer potential energy -3 pi G M^2 / (32 a) and the N = 1 special case.  CPU only."""
import math
import os

import mpmath as mp
import numpy as np
import pytest

from oracle import oracle as O
from oracle import integrate as OI
from paper_1312_1789_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "w3.txt")


def _read_w3():
    out = {}
    with open(GOLD) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            tok = line.split()
            out[(int(tok[0]), tok[1])] = np.array([float(s) for s in tok[2:]])
    return out


def _two_pass(m, x, v, eps2):
    """c-10 bootstrap: order-4 pass then order-8 pass with pass-1 acc, jerk as the particles' a, j."""
    idx = np.arange(m.shape[0], dtype=np.int32)
    acc, jerk, _, _, pot = O.force(m, x, v, None, None, idx, 4, eps2)
    a8, j8, snap, crk, pot8 = O.force(m, x, v, acc, jerk, idx, 8, eps2)
    assert np.array_equal(a8, acc) and np.array_equal(j8, jerk) and np.array_equal(pot, pot8)
    a6, j6, s6, _, _ = O.force(m, x, v, acc, None, idx, 6, eps2)
    assert np.array_equal(a6, acc) and np.array_equal(j6, jerk) and np.array_equal(s6, snap)
    return acc, jerk, snap, crk, pot


def test_w3_worked_example():
    g = _read_w3()
    m = np.array([0.5, 0.3, 0.2])
    x = np.array([[1, 0, 0], [-0.5, 0.7, 0.1], [0.2, -0.9, -0.4]], dtype=np.float64)
    v = np.array([[0, 0.4, 0.1], [-0.3, -0.2, 0.2], [0.5, 0.1, -0.3]], dtype=np.float64)
    acc, jerk, snap, crk, pot = _two_pass(m, x, v, 0.01)
    for i in range(3):
        for name, arr in (("acc", acc), ("jerk", jerk), ("snap", snap), ("crackle", crk)):
            ref = g[(i, name)]
            assert np.linalg.norm(arr[i] - ref) <= 1e-13 * np.linalg.norm(ref), (i, name)
        assert abs(pot[i] - g[(i, "pot")][0]) <= 1e-14 * abs(g[(i, "pot")][0])
    # SURVEY.md pinned W = 1/2 Sum m pot
    assert abs(0.5 * np.dot(m, pot) - (-0.2018357925419243)) < 1e-15


@pytest.mark.parametrize("n,seed", [(2, 1), (5, 2), (8, 3)])
def test_mpmath_bruteforce_random(n, seed):
    """Independent derivation: d^k/dt^k of the plain softened acceleration along cubic trajectories whose
    2nd/3rd Taylor coefficients are RANDOM a_k, j_k (not forces) -- exercises r.a, v.a, r.j terms in general."""
    rng = np.random.default_rng(seed)
    m = rng.uniform(0.1, 1.0, n)
    x = rng.normal(0, 1, (n, 3))
    v = rng.normal(0, 1, (n, 3))
    a = rng.normal(0, 1, (n, 3))
    jj = rng.normal(0, 1, (n, 3))
    eps2 = 0.0025
    idx = np.arange(n, dtype=np.int32)
    acc, jerk, snap, crk, pot = O.force(m, x, v, a, jj, idx, 8, eps2)
    mp.mp.dps = 40
    mm = [mp.mpf(float(s)) for s in m]
    conv = lambda arr: [[mp.mpf(float(s)) for s in r] for r in arr]
    X, V, A, Jm = conv(x), conv(v), conv(a), conv(jj)
    e2 = mp.mpf(eps2)

    def acc_of(i, c, t):
        s = mp.mpf(0)
        for j in range(n):
            if j == i:
                continue
            r = [(X[j][d] - X[i][d]) + (V[j][d] - V[i][d]) * t + (A[j][d] - A[i][d]) * t**2 / 2
                 + (Jm[j][d] - Jm[i][d]) * t**3 / 6 for d in range(3)]
            s += mm[j] * r[c] / (r[0] ** 2 + r[1] ** 2 + r[2] ** 2 + e2) ** mp.mpf("1.5")
        return s

    for i in range(n):
        for k, arr in enumerate((acc, jerk, snap, crk)):
            ref = np.array([float(mp.diff(lambda t: acc_of(i, c, t), 0, k)) for c in range(3)])
            assert np.linalg.norm(arr[i] - ref) <= 1e-12 * np.linalg.norm(ref), (i, k)
        pref = -sum(mm[j] / mp.sqrt(sum((X[j][d] - X[i][d]) ** 2 for d in range(3)) + e2) for j in range(n) if j != i)
        assert abs(pot[i] - float(pref)) <= 1e-14 * abs(float(pref))


def test_two_body_circular_closed_form():
    """eps = 0, circular orbit: acc_1 = m_2 r/d^3, jerk_1 = m_2 v/d^3, snap = -w^2 acc, crackle = -w^2 jerk."""
    m1, m2, d = 0.7, 0.3, 2.0
    w2 = (m1 + m2) / d**3
    vrel = math.sqrt((m1 + m2) / d)
    x = np.array([[-m2 / (m1 + m2) * d, 0, 0], [m1 / (m1 + m2) * d, 0, 0]])
    v = np.array([[0, -m2 / (m1 + m2) * vrel, 0], [0, m1 / (m1 + m2) * vrel, 0]])
    m = np.array([m1, m2])
    acc, jerk, snap, crk, pot = _two_pass(m, x, v, 0.0)
    r, vv = x[1] - x[0], v[1] - v[0]
    np.testing.assert_allclose(acc[0], m2 * r / d**3, rtol=1e-15, atol=1e-17)
    np.testing.assert_allclose(jerk[0], m2 * vv / d**3, rtol=1e-15, atol=1e-17)
    np.testing.assert_allclose(snap[0], -w2 * acc[0], rtol=1e-13, atol=1e-17)
    np.testing.assert_allclose(crk[0], -w2 * jerk[0], rtol=1e-13, atol=1e-17)
    np.testing.assert_allclose(acc[1], -m1 * r / d**3, rtol=1e-15, atol=1e-17)
    np.testing.assert_allclose(pot, [-m2 / d, -m1 / d], rtol=1e-15)


def test_n1_all_zero():
    out = O.force(np.array([1.0]), np.zeros((1, 3)), np.ones((1, 3)), np.ones((1, 3)), np.ones((1, 3)),
                  np.array([0], dtype=np.int32), 8, 1e-4)
    for a in out:
        assert np.all(a == 0.0)


def test_self_excluded_by_index_not_by_position():
    """c-2: a DIFFERENT particle at the same position is included: adds 0 to acc and -m/eps to pot."""
    m = np.array([0.5, 0.25, 0.25])
    x = np.array([[0, 0, 0], [0, 0, 0], [1.0, 0, 0]])
    v = np.zeros((3, 3))
    eps2 = 0.01
    acc, jerk, _, _, pot = O.force(m, x, v, None, None, np.array([0], dtype=np.int32), 4, eps2)
    assert pot[0] == pytest.approx(-0.25 / 0.1 - 0.25 / math.sqrt(1.01), rel=1e-15)
    assert acc[0, 0] == pytest.approx(0.25 / 1.01**1.5, rel=1e-15)


def test_active_list_order_and_subset():
    c = W.cluster(1, n=200)
    idx_all = np.arange(200, dtype=np.int32)
    full = O.force(c["m"], c["x"], c["v"], None, None, idx_all, 4, c["eps2"])
    sub = np.array([3, 17, 150, 199], dtype=np.int32)
    part = O.force(c["m"], c["x"], c["v"], None, None, sub, 4, c["eps2"])
    for f, p in zip(full, part):
        if f is not None:
            assert np.array_equal(f[sub], p)


def test_sum_m_times_derivatives_vanish():
    """Pairwise antisymmetry: Sum_i m_i {acc, jerk, snap, crackle}_i = 0 when everybody is active at one time."""
    c = W.cluster(5, n=600)  # Plummer + central BH
    acc, jerk, snap, crk, pot = _two_pass(c["m"], c["x"], c["v"], c["eps2"])
    for arr in (acc, jerk, snap, crk):
        tot = (c["m"][:, None] * arr).sum(axis=0)
        scale = (c["m"][:, None] * np.abs(arr)).sum()
        assert np.linalg.norm(tot) <= 1e-12 * scale


def test_plummer_potential_energy_closed_form():
    """W = 1/2 Sum m pot -> -3 pi G M^2 / (32 a_P) = -1/2 in Henon units (large-N limit; the generator truncates
    0.1 % of the mass).  Three seeds, N = 4096: mean within 1.5 %."""
    ws = []
    for s in range(3):
        rng = W.rng_for(1, 10 + s)
        m, x, v = W.plummer(4096, rng)
        idx = np.arange(4096, dtype=np.int32)
        pot = O.force(m, x, v, None, None, idx, 4, 1e-8)[4]
        ws.append(0.5 * np.dot(m, pot))
    expect = -3.0 * math.pi / (32.0 * W.A_PLUMMER)
    assert expect == pytest.approx(-0.5, abs=1e-15)
    assert abs(np.mean(ws) - expect) < 0.015 * abs(expect), ws


def test_plummer_virial_and_energy():
    """Henon units: E = T + W = -1/4 and 2T + W = 0 to O(N^-1/2)."""
    c = W.cluster(2, n=8192)
    idx = np.arange(c["n"], dtype=np.int32)
    pot = O.force(c["m"], c["x"], c["v"], None, None, idx, 4, c["eps2"])[4]
    k, w = O.energy(c["m"], c["v"], pot)
    assert abs((k + w) + 0.25) < 0.01
    assert abs(2 * k / (-w) - 1.0) < 0.03


def test_total_energy_helper_matches_definition():
    c = W.cluster(1, n=64)
    s = OI.bootstrap(c["m"], c["x"], c["v"], 4, c["eps2"])
    e = OI.total_energy(s, c["eps2"])
    n = c["n"]
    w = 0.0
    for i in range(n):
        for j in range(i + 1, n):
            w -= c["m"][i] * c["m"][j] / math.sqrt(np.sum((c["x"][i] - c["x"][j]) ** 2) + c["eps2"])
    k = 0.5 * np.sum(c["m"] * np.sum(c["v"] ** 2, axis=1))
    assert e == pytest.approx(k + w, rel=1e-13)


def test_force_abs_conditioning_numbers():
    """c-16 diagnostic: kappa = Sum|term| / |Sum term| is exactly 1 for N = 2 (one term), >= 1 always (triangle
    inequality), and large for a particle in the middle of a symmetric pair (near-total cancellation)."""
    rng = np.random.default_rng(2)
    m = np.array([0.5, 0.5])
    x = np.array([[1.0, 0.2, 0.0], [-0.3, 0.0, 0.1]])
    v = rng.normal(size=(2, 3))
    a = rng.normal(size=(2, 3))
    j = rng.normal(size=(2, 3))
    idx = np.arange(2, dtype=np.int32)
    f = O.force(m, x, v, a, j, idx, 8, 0.01)
    ab = O.force_abs(m, x, v, a, j, idx, 8, 0.01)
    for k in range(4):
        np.testing.assert_allclose(ab[k], np.linalg.norm(f[k], axis=1), rtol=1e-14)
    n = 40
    m = rng.uniform(0.1, 1.0, n)
    x, v, a, j = (rng.normal(size=(n, 3)) for _ in range(4))
    idx = np.arange(n, dtype=np.int32)
    f = O.force(m, x, v, a, j, idx, 8, 0.01)
    ab = O.force_abs(m, x, v, a, j, idx, 8, 0.01)
    for k in range(4):
        assert np.all(ab[k] >= np.linalg.norm(f[k], axis=1) * (1 - 1e-14))
    # a test particle midway between two equal masses at rest: acc cancels, kappa_acc is huge
    m = np.array([1e-12, 1.0, 1.0])
    x = np.array([[0.0, 0.0, 1e-9], [1.0, 0.0, 0.0], [-1.0, 0.0, 0.0]])
    z = np.zeros((3, 3))
    f = O.force(m, x, z, None, None, np.array([0], dtype=np.int32), 4, 0.0)
    ab = O.force_abs(m, x, z, None, None, np.array([0], dtype=np.int32), 4, 0.0)
    assert ab[0][0] / np.linalg.norm(f[0][0]) > 1e8 and abs(ab[0][0] - 2.0) < 1e-9
