"""Pins of the CPU oracle's predictor, corrector, interpolated derivatives, time-step rule, quantisation and
block selection (SURVEY.md 8(c) c-5 .. c-11) against polynomial exactness, closed forms, property tests, the
convergence table B2 and Kepler / energy invariants.  CPU only."""
import math
from fractions import Fraction

import numpy as np
import pytest

from oracle import oracle as O
from oracle import integrate as OI
from paper_1312_1789_b200 import workloads as W

FACT = [math.factorial(k) for k in range(12)]


def _poly_derivs(coef, t, kmax):
    """coef[k] = k-th derivative at 0 of a polynomial (Taylor form); returns derivatives 0..kmax at time t."""
    out = []
    for d in range(kmax + 1):
        s = 0.0
        for k in range(d, len(coef)):
            s = s + coef[k] * t ** (k - d) / FACT[k - d]
        out.append(s)
    return out


# ------------------------------------------------------------------------------------------------- c-5
@pytest.mark.parametrize("order", [4, 6, 8])
def test_predictor_polynomial_exactness(order):
    """Exact for x(t) a polynomial of degree <= p-1 (x, v, then a^(0..p-3) as Taylor coefficients)."""
    rng = np.random.default_rng(order)
    n = 7
    # Taylor coefficients of x(t) about t_i: c[0]=x, c[1]=v, c[k+2]=D_k
    c = [rng.normal(0, 1, (n, 3)) for _ in range(order)]
    t = -np.ldexp(1.0, -rng.integers(1, 6, n))
    t_now = 0.0
    xp, vp, ap, jp = O.predict(t_now, order, t, c[0], c[1], c[2:])
    tau = (t_now - t)[:, None]
    d = _poly_derivs(c, tau, 3)
    np.testing.assert_allclose(xp, d[0], rtol=1e-14, atol=1e-15)
    np.testing.assert_allclose(vp, d[1], rtol=1e-14, atol=1e-15)
    if order >= 6:
        np.testing.assert_allclose(ap, d[2], rtol=1e-14, atol=1e-15)
    else:
        assert ap is None
    if order >= 8:
        np.testing.assert_allclose(jp, d[3], rtol=1e-14, atol=1e-15)
    else:
        assert jp is None


@pytest.mark.parametrize("order", [4, 6, 8])
def test_predictor_truncation_is_exactly_order_p(order):
    """A degree-p term must NOT be captured by x_p (truncation after tau^(p-1)), checked with exact rationals."""
    n = 1
    D = [np.full((n, 3), float(k + 1)) for k in range(order - 2)]
    x = np.full((n, 3), 0.5)
    v = np.full((n, 3), -0.25)
    tau = 0.125
    xp, vp, ap, jp = O.predict(tau, order, np.zeros(n), x, v, D)
    ex = Fraction(1, 2) + Fraction(-1, 4) * Fraction(1, 8)
    ev = Fraction(-1, 4)
    for k in range(order - 2):
        ex += Fraction(k + 1) * Fraction(1, 8) ** (k + 2) / FACT[k + 2]
        ev += Fraction(k + 1) * Fraction(1, 8) ** (k + 1) / FACT[k + 1]
    assert xp[0, 0] == pytest.approx(float(ex), rel=2e-16)
    assert vp[0, 0] == pytest.approx(float(ev), rel=2e-16)


def test_predictor_tau_zero_returns_state():
    rng = np.random.default_rng(0)
    n = 5
    x, v = rng.normal(0, 1, (n, 3)), rng.normal(0, 1, (n, 3))
    D = [rng.normal(0, 1, (n, 3)) for _ in range(6)]
    t = np.full(n, 0.375)
    xp, vp, ap, jp = O.predict(0.375, 8, t, x, v, D)
    assert np.array_equal(xp, x) and np.array_equal(vp, v) and np.array_equal(ap, D[0]) and np.array_equal(jp, D[1])


# ------------------------------------------------------------------------------------------- c-6, c-7
def _run_corrector_on_polynomial(order, deg_a, h, variant=0, seed=0):
    """a(t) = polynomial of degree deg_a (random Taylor coefficients at t0 = 0).  Feed the corrector the exact
    a^(0..K-1) at both ends; return (x1, v1, D_new, exact derivs at t1, exact x1, exact v1)."""
    K = order // 2
    rng = np.random.default_rng(100 * order + deg_a + seed)
    # Taylor coefficients of x about 0: x0, v0, then a^(k)(0) for k = 0..deg_a
    cx = [rng.normal(0, 1, (1, 3)) for _ in range(deg_a + 3)]
    a0 = _poly_derivs(cx[2:], 0.0, order)
    a1 = _poly_derivs(cx[2:], h, order)
    x1e, v1e = _poly_derivs(cx, h, 1)
    t, dt = np.zeros(1), np.full(1, h)
    x, v = cx[0].copy(), cx[1].copy()
    D = [np.zeros((1, 3)) for _ in range(8)]
    for k in range(K):
        D[k][:] = a0[k]
    pot_state = np.zeros(1)
    f = [np.ascontiguousarray(a1[k]) if k < K else None for k in range(4)]
    O.correct(np.array([0], dtype=np.int32), order, h, 0.1, 2.0**-40, 1.0, t, dt, x, v, D, pot_state,
              f[0], f[1], f[2], f[3], np.array([-1.5]), variant=variant)
    assert t[0] == h and pot_state[0] == -1.5
    return x, v, D, a1, x1e, v1e


@pytest.mark.parametrize("order", [4, 6, 8])
def test_corrector_polynomial_exactness(order):
    K = order // 2
    h = 0.25
    # degree 2K-1: v exact, interpolated derivatives exact, compact x NOT exact (c-6 "Ambiguity")
    x, v, D, a1, x1e, v1e = _run_corrector_on_polynomial(order, 2 * K - 1, h)
    np.testing.assert_allclose(v, v1e, rtol=1e-13, atol=1e-14)
    for k in range(K, 2 * K):
        # the formulas difference O(1) numbers times coefficients up to 1e5 and divide by h^k
        np.testing.assert_allclose(D[k], a1[k], rtol=0, atol=2e-11 / h**k)
    for k in range(K):
        assert np.array_equal(D[k], a1[k])
    # ... while compact x is NOT exact at degree 2K-1 (error ~ h^(2K+1) a^(2K-1) / big: use a long step to see it)
    xl, vl, _, _, xle, vle = _run_corrector_on_polynomial(order, 2 * K - 1, 4.0)
    np.testing.assert_allclose(vl, vle, rtol=1e-12, atol=1e-12)
    assert np.max(np.abs(xl - xle)) > 1e-6 * np.max(np.abs(xle))
    # degree 2K-2: x (compact) exact too
    x, v, D, a1, x1e, v1e = _run_corrector_on_polynomial(order, 2 * K - 2, h)
    np.testing.assert_allclose(v, v1e, rtol=1e-13, atol=1e-14)
    np.testing.assert_allclose(x, x1e, rtol=1e-13, atol=1e-14)


def test_corrector_p4_compact_vs_double_integral_difference():
    """c-6: the two readings differ by h^5 a^(3) / 720 at p = 4; the double-integral variant (1) is exact at
    degree 3."""
    h = 0.5
    xc, _, D, a1, x1e, _ = _run_corrector_on_polynomial(4, 3, h, variant=0)
    xd, _, _, _, _, _ = _run_corrector_on_polynomial(4, 3, h, variant=1)
    np.testing.assert_allclose(xd, x1e, rtol=1e-13, atol=1e-14)
    np.testing.assert_allclose(np.abs(xc - xd), np.abs(h**5 * D[3] / 720.0), rtol=1e-8)


@pytest.mark.parametrize("order", [4, 6, 8])
def test_corrector_time_reversal_prescribed_field(order):
    """+h then -h with a prescribed a(t) returns (x0, v0) to rounding (both formulas are symmetric under
    (0 <-> 1, h -> -h))."""
    K = order // 2
    rng = np.random.default_rng(order)
    cx = [rng.normal(0, 1, (1, 3)) for _ in range(12)]  # degree-9 acceleration: NOT integrated exactly
    h = 0.125
    a0 = _poly_derivs(cx[2:], 0.0, K)
    a1 = _poly_derivs(cx[2:], h, K)
    x, v = cx[0].copy(), cx[1].copy()
    t, dt = np.zeros(1), np.full(1, h)
    D = [np.zeros((1, 3)) for _ in range(8)]
    for k in range(K):
        D[k][:] = a0[k]
    ps = np.zeros(1)
    idx = np.array([0], dtype=np.int32)
    f = [np.ascontiguousarray(a1[k]) if k < K else None for k in range(4)]
    O.correct(idx, order, h, 0.1, 2.0**-40, 1.0, t, dt, x, v, D, ps, f[0], f[1], f[2], f[3], np.zeros(1))
    assert np.max(np.abs(x - cx[0])) > 1e-3
    dt[:] = -h  # step back: "old" end is now t1, force end is t0
    f = [np.ascontiguousarray(a0[k]) if k < K else None for k in range(4)]
    O.correct(idx, order, 0.0, 0.1, 2.0**-40, 1.0, t, dt, x, v, D, ps, f[0], f[1], f[2], f[3], np.zeros(1))
    np.testing.assert_allclose(x, cx[0], rtol=0, atol=1e-15)
    np.testing.assert_allclose(v, cx[1], rtol=0, atol=1e-15)


# ------------------------------------------------------------------------------------------- c-8, c-9
@pytest.mark.parametrize("order", [4, 6, 8])
def test_dt_criterion_exponential_pin(order):
    """a(t) = a_0 e^(lambda t) => |a^(k)| = lambda^k |a| => dt_crit = eta / lambda exactly; the quantised step
    is 2^floor(log2(eta/lambda)) (lambda chosen away from power-of-two boundaries)."""
    a0 = np.array([0.3, -0.4, 1.2])
    for lam, eta in ((3.0, 0.1), (17.0, 0.02), (0.7, 0.1), (1000.0, 0.1)):
        derivs = [a0 * lam**k for k in range(order)]
        want = 2.0 ** math.floor(math.log2(eta / lam))
        got = O.new_dt(order, derivs, 0.0, want, eta, 2.0**-40, 1.0)  # dt_old = want: no doubling limit, t1 = 0
        assert got == want, (order, lam, eta)


def test_dt_exact_power_of_two_tie():
    """dt_crit exactly 2^k => 2^k (eta = 2^-3, lambda = 2 => 2^-4)."""
    a0 = np.array([1.0, 0.0, 0.0])
    for order in (4, 6, 8):
        derivs = [a0 * 2.0**k for k in range(order)]
        assert O.new_dt(order, derivs, 0.0, 2.0**-4, 0.125, 2.0**-40, 1.0) == 2.0**-4


def test_dt_quantisation_properties():
    rng = np.random.default_rng(5)
    dt_min, dt_max = 2.0**-20, 2.0**-3
    for order in (4, 6, 8):
        q = order - 3
        for _ in range(300):
            derivs = [rng.normal(0, 1, 3) * 10.0 ** rng.uniform(-2, 2) * 30.0**k for k in range(order)]
            kold = int(rng.integers(-18, -3))
            dt_old = 2.0**kold
            t1 = dt_old * int(rng.integers(1, 1000))
            eta = 0.1
            got = O.new_dt(order, derivs, t1, dt_old, eta, dt_min, dt_max)
            # independent evaluation of dt_crit in extended precision
            nr = [math.sqrt(sum(float(c) ** 2 for c in d)) for d in derivs]
            A1 = math.sqrt(nr[0] * nr[2] + nr[1] ** 2)
            Ap = math.sqrt(nr[order - 3] * nr[order - 1] + nr[order - 2] ** 2)
            crit = eta * (A1 / Ap) ** (1.0 / q)
            m, e = math.frexp(got)
            assert m == 0.5 and dt_min <= got <= dt_max
            assert got <= 2 * dt_old
            assert math.fmod(t1, got) == 0.0
            if got > dt_min:
                assert got <= crit * (1 + 1e-12)
            want = 2.0 ** math.floor(math.log2(crit))
            want = min(want, 2 * dt_old)
            if want == 2 * dt_old and math.fmod(t1, want) != 0.0:
                want = dt_old
            want = max(min(want, dt_max), dt_min)
            if abs(math.log2(crit) - round(math.log2(crit))) > 1e-9:
                assert got == want


def test_dt_degenerate_cases():
    z = np.zeros(3)
    a = np.array([1.0, 0, 0])
    # A^(p-2) == 0 => +inf => limited by 2 dt_old / dt_max
    assert O.new_dt(4, [a, a, z, z], 0.0, 2.0**-6, 0.1, 2.0**-20, 2.0**-3) == 2.0**-5
    assert O.new_dt(4, [a, a, z, z], 0.0, 2.0**-3, 0.1, 2.0**-20, 2.0**-3) == 2.0**-3
    # NaN => dt_min
    nan = np.array([np.nan, 0, 0])
    assert O.new_dt(6, [a, a, a, nan, a, a], 0.0, 2.0**-6, 0.1, 2.0**-20, 2.0**-3) == 2.0**-20
    # commensurability: may not double at odd multiples
    big = [a, a * 1e-3, a * 1e-6, a * 1e-9]
    assert O.new_dt(4, big, 3 * 2.0**-6, 2.0**-6, 0.1, 2.0**-20, 1.0) == 2.0**-6
    assert O.new_dt(4, big, 4 * 2.0**-6, 2.0**-6, 0.1, 2.0**-20, 1.0) == 2.0**-5


def test_initial_dt():
    acc = np.array([[3.0, 0, 0], [1.0, 0, 0], [1.0, 0, 0]])
    jerk = np.array([[0, 4.0, 0], [0, 0, 0], [0, 1e9, 0]])
    dt = O.initial_dt(acc, jerk, 0.01, 2.0**-20, 2.0**-4)
    assert dt[0] == 2.0 ** math.floor(math.log2(0.01 * 0.75))
    assert dt[1] == 2.0**-4 and dt[2] == 2.0**-20


def test_next_block_bit_exact():
    rng = np.random.default_rng(3)
    n = 1000
    k = rng.integers(3, 12, n)
    dt = np.ldexp(1.0, -k)
    t = dt * rng.integers(0, 5, n)
    tn, idx = O.next_block(t, dt)
    s = t + dt
    assert tn == s.min()
    assert np.array_equal(idx, np.nonzero(s == s.min())[0].astype(np.int32))
    assert idx.dtype == np.int32 and np.all(np.diff(idx) > 0)


# ------------------------------------------------------------------------------ B2 convergence, Kepler
B2 = {  # SURVEY.md 8(c) "Convergence pin B2": |dE/E| at t = 8, dt = 2^-4 .. 2^-7
    4: [3.1e-05, 5.4e-06, 5.6e-07, 4.2e-08],
    6: [5.1e-07, 1.6e-08, 4.5e-10, 8.6e-12],
    8: [5.2e-06, 4.1e-09, 8.2e-12, 2.9e-14],
}


def _binary(ecc=0.5):
    m = np.array([0.5, 0.5])
    rp = 1.0 - ecc
    vp = math.sqrt((1 + ecc) / (1 - ecc))  # relative speed at pericentre, a = 1, M = 1
    x = np.array([[rp / 2, 0, 0], [-rp / 2, 0, 0]])
    v = np.array([[0, vp / 2, 0], [0, -vp / 2, 0]])
    return m, x, v


def _energy2(m, x, v):
    return 0.5 * np.sum(m * np.sum(v * v, axis=1)) - m[0] * m[1] / np.linalg.norm(x[0] - x[1])


@pytest.mark.parametrize("order", [4, 6, 8])
def test_convergence_table_b2(order):
    m, x, v = _binary()
    e0 = _energy2(m, x, v)
    errs = []
    for k in (4, 5, 6, 7):
        dt = 2.0**-k
        s = OI.bootstrap(m, x, v, order, 0.0, fixed_dt=dt)
        OI.integrate(s, 8.0, 0.0, 1e-30, dt, dt)  # eta tiny + dt_min = dt_max = dt: shared constant step
        assert np.all(s.t == 8.0)
        errs.append(abs((_energy2(s.m, s.x, s.v) - e0) / e0))
    for got, want in zip(errs[:3] if order == 8 else errs, B2[order]):
        assert want / 1.6 < got < want * 1.6, (order, errs)
    if order == 8:
        assert errs[3] < 3e-13  # rounding floor
    slope = math.log2(errs[1] / errs[2])
    assert slope > order - 1.0, (order, errs)


def test_p4_double_integral_variant_matches_its_own_table():
    """the double-integral 4th-order variant gives 5.0e-05, 4.2e-06, 4.9e-07, 3.8e-08."""
    m, x, v = _binary()
    e0 = _energy2(m, x, v)
    want = [5.0e-05, 4.2e-06, 4.9e-07, 3.8e-08]
    for k, w in zip((4, 5, 6, 7), want):
        dt = 2.0**-k
        s = OI.bootstrap(m, x, v, 4, 0.0, fixed_dt=dt)
        OI.integrate(s, 8.0, 0.0, 1e-30, dt, dt, variant=1)
        got = abs((_energy2(s.m, s.x, s.v) - e0) / e0)
        assert w / 1.6 < got < w * 1.6


@pytest.mark.parametrize("order", [4, 6, 8])
def test_kepler_orbit_closes(order):
    """Circular two-body orbit, period T = 2 pi sqrt(a^3/M) : position after one period returns, error falls at
    the scheme's order when dt halves (T is not dyadic, so integrate to the last block time and finish with the
    analytic rotation angle)."""
    m = np.array([0.5, 0.5])
    x = np.array([[0.5, 0, 0], [-0.5, 0, 0]])
    v = np.array([[0, 0.5, 0], [0, -0.5, 0]])  # separation 1, M = 1 => omega = 1, T = 2 pi
    errs = []
    for k in (4, 5):
        dt = 2.0**-k
        s = OI.bootstrap(m, x, v, order, 0.0, fixed_dt=dt)
        nsteps = int(2 * math.pi / dt)
        OI.integrate(s, nsteps * dt, 0.0, 1e-30, dt, dt)
        ang = nsteps * dt  # omega = 1
        ref = 0.5 * np.array([math.cos(ang), math.sin(ang), 0.0])
        errs.append(np.linalg.norm(s.x[0] - ref))
    assert errs[0] < 1e-3
    assert errs[0] / errs[1] > 2.0 ** (order - 1.2), (order, errs)


@pytest.mark.parametrize("order", [4, 6, 8])
def test_block_timestep_energy_conservation_plummer(order):
    """Short block-time-step integration of a small softened Plummer sphere: every particle lands on t_end,
    times stay commensurate, energy is conserved to the accuracy eta buys."""
    c = W.cluster(1, n=128)
    eps2 = 1e-4
    dt_min, dt_max = 2.0**-24, 2.0**-5
    s = OI.bootstrap(c["m"], c["x"], c["v"], order, eps2, dt_min=dt_min, dt_max=dt_max)
    e0 = OI.total_energy(s, eps2)
    nb, pairs = OI.integrate(s, 0.125, eps2, 0.1, dt_min, dt_max)
    assert np.all(s.t == 0.125)
    assert nb > 4
    assert np.all(np.fmod(s.t, s.dt) == 0.0)
    e1 = OI.total_energy(s, eps2)
    assert abs((e1 - e0) / e0) < {4: 1e-6, 6: 1e-7, 8: 1e-7}[order]


# ------------------------------------------------------------------------------------------- c-8b (R8b)
@pytest.mark.parametrize("order,pc", [(6, 4), (8, 4), (8, 6)])
def test_dt_criterion_order_option(order, pc):
    """crit_order pc < p: the corrector's new step equals the order-pc criterion evaluated on the lowest pc
    derivatives at t1 (which the corrector stores, so they can be read back), everything else is untouched;
    it still reproduces eta/lambda on an exponential, and it differs from the order-p criterion in general.  For
    p = 6, pc = 4 the fourth entry is the mean crackle (s1 - s0)/h: only directly computed derivatives decide."""
    rng = np.random.default_rng(8)
    n = 64
    idx = np.arange(n, dtype=np.int32)
    h = 2.0**-6
    mk = lambda: np.ascontiguousarray(rng.normal(0, 1, (n, 3)))
    base = dict(t=np.zeros(n), dt=np.full(n, h), x=mk(), v=mk(), D=[mk() * 3.0**k for k in range(8)], pot=np.zeros(n))
    f = [mk() * 3.0**k for k in range(4)]
    out = {}
    for co in (0, pc):
        s = dict(t=base["t"].copy(), dt=base["dt"].copy(), x=base["x"].copy(), v=base["v"].copy(),
                 D=[d.copy() for d in base["D"]], pot=base["pot"].copy())
        O.correct(idx, order, h, 0.1, 2.0**-30, 2.0**-2, s["t"], s["dt"], s["x"], s["v"], s["D"], s["pot"],
                  f[0], f[1], f[2], f[3], np.zeros(n), crit_order=co)
        out[co] = s
    a, b = out[0], out[pc]
    assert np.array_equal(a["x"], b["x"]) and np.array_equal(a["v"], b["v"])
    for k in range(order):
        assert np.array_equal(a["D"][k], b["D"][k])
    want_p = np.array([O.new_dt(order, [a["D"][k][i] for k in range(order)], h, h, 0.1, 2.0**-30, 2.0**-2) for i in range(n)])
    low = [a["D"][k] for k in range(pc)]
    if order == 6 and pc == 4:  # mean crackle of the step from the two directly computed snaps
        low[3] = (f[2] - base["D"][2]) / h
    want_pc = np.array([O.new_dt(pc, [low[k][i] for k in range(pc)], h, h, 0.1, 2.0**-30, 2.0**-2) for i in range(n)])
    assert np.array_equal(a["dt"], want_p)
    assert np.array_equal(b["dt"], want_pc)
    assert np.any(want_p != want_pc)


def test_block_timestep_energy_conservation_criterion_order4():
    """8th-order scheme stepped with Aarseth's four-derivative criterion (R8b): still lands on t_end and conserves
    energy (fp64 oracle; the CUDA path needs this variant, R8b)."""
    c = W.cluster(1, n=128)
    eps2 = 1e-4
    dt_min, dt_max = 2.0**-24, 2.0**-5
    s = OI.bootstrap(c["m"], c["x"], c["v"], 8, eps2, dt_min=dt_min, dt_max=dt_max)
    e0 = OI.total_energy(s, eps2)
    OI.integrate(s, 0.125, eps2, 0.1, dt_min, dt_max, crit_order=4)
    assert np.all(s.t == 0.125)
    e1 = OI.total_energy(s, eps2)
    assert abs((e1 - e0) / e0) < 1e-7
