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
            # the quantised value itself is pinned without any skipped case in test_dt_quantisation_exact_rational



def _norm3(d):
    """|d| in fp64 in the order c-8 states ((x^2 + y^2) + z^2, IEEE sqrt): python floats are IEEE fp64."""
    return math.sqrt((float(d[0]) * float(d[0]) + float(d[1]) * float(d[1])) + float(d[2]) * float(d[2]))


def _exact_k(order, derivs, eta):
    """c-9 step 1 with exact rational arithmetic: the largest integer k with Ap 2^(k q) <= fl(A1 E), where A1, Ap,
    E are the fp64 numbers c-8/c-9 define (norms, sqrt, E = eta^q by repeated fp64 products) and everything from
    there on is exact (fractions.Fraction: no log, no pow, no ldexp search, no rounding).  None if Ap == 0."""
    q = order - 3
    n = [_norm3(d) for d in derivs]
    A1 = math.sqrt(n[0] * n[2] + n[1] * n[1])
    Ap = math.sqrt(n[order - 3] * n[order - 1] + n[order - 2] * n[order - 2])
    E = 1.0
    for _ in range(q):
        E = E * eta
    rhs = A1 * E
    if Ap == 0.0:
        return None
    ratio = Fraction(rhs) / Fraction(Ap)  # exact
    if ratio <= 0:
        return -10**9
    # largest k with 2^(k q) <= ratio
    k = (ratio.numerator.bit_length() - ratio.denominator.bit_length()) // q + 2
    while Fraction(2) ** (k * q) > ratio:
        k -= 1
    return k


def _quantise(k, t1, dt_old, dt_min, dt_max):
    """c-9 steps 2-4 on exact dyadic numbers."""
    kmin, kmax = int(round(math.log2(dt_min))), int(round(math.log2(dt_max)))
    want = Fraction(2) ** max(min(k, kmax + 1), kmin - 1) if k is not None else Fraction(2) ** (kmax + 1)
    two_old = 2 * Fraction(dt_old)
    want = min(want, two_old)
    if want == two_old and (Fraction(t1) / want).denominator != 1:
        want = Fraction(dt_old)
    want = min(want, Fraction(dt_max))
    want = max(want, Fraction(dt_min))
    return float(want)


def test_dt_quantisation_exact_rational():
    """c-9 against exact rational arithmetic (no tolerance, no skipped case): 2400 random derivative sets for
    p = 4, 6, 8, plus constructed ties and one-ulp near-ties where a log2-based floor would go wrong."""
    rng = np.random.default_rng(11)
    dt_min, dt_max = 2.0**-24, 2.0**-2
    for order in (4, 6, 8):
        for _ in range(800):
            derivs = [rng.normal(0, 1, 3) * 10.0 ** rng.uniform(-2, 2) * 25.0**k for k in range(order)]
            kold = int(rng.integers(-20, -3))
            dt_old = 2.0**kold
            t1 = dt_old * int(rng.integers(1, 1000))
            eta = float(rng.choice([0.1, 0.02, 0.3, 2.0**-3]))
            got = O.new_dt(order, derivs, t1, dt_old, eta, dt_min, dt_max)
            want = _quantise(_exact_k(order, derivs, eta), t1, dt_old, dt_min, dt_max)
            assert got == want, (order, eta, derivs)
    # constructed ties and near-ties: derivatives along x with |a^(k)| = lambda^k => A1/Ap = lambda^-(q) * (exact
    # powers of two), dt_crit = eta / lambda; eta one ulp either side of a power of two flips the floor
    ex = np.array([1.0, 0.0, 0.0])
    for order in (4, 6, 8):
        for lam_log2 in (0, 1, 3):
            lam = 2.0**lam_log2
            derivs = [ex * lam**k for k in range(order)]
            for k_eta in (-3, -5):
                e0 = 2.0**k_eta
                for eta, kk in ((e0, k_eta - lam_log2), (np.nextafter(e0, 0.0), k_eta - lam_log2 - 1),
                                (np.nextafter(e0, 1.0), k_eta - lam_log2)):
                    assert _exact_k(order, derivs, float(eta)) == kk
                    got = O.new_dt(order, derivs, 0.0, 2.0**kk, float(eta), 2.0**-40, 1.0)
                    assert got == 2.0**kk, (order, lam, eta)


def test_dt_mean_crackle_closed_form_pin():
    """c-8b, p = 6 with the 4-derivative criterion (the library default, R8b): for a(t) = a0 e^(lambda t)
    the mean crackle of the step is cbar = (s1 - s0)/h = lambda^2 a1 (1 - e^(-lambda h))/h = lambda^2 a1 g, so
    A^(1) = sqrt(2) lambda |a1|, A^(2) = lambda^(3/2) |a1| sqrt(g + lambda) and
        dt_crit = eta sqrt(2 / (lambda (g + lambda)))        (-> eta/lambda as h -> 0),
    evaluated here with 50-digit mpmath and quantised by hand; the oracle never sees this formula.  The cases
    include ones where the true crackle (dt_crit = eta/lambda) and the interpolated a3 of c-7 would land on a
    different power of two, so a corrector that fed either of those to the criterion fails."""
    import mpmath as mp
    mp.mp.dps = 50
    u = np.array([0.6, -0.48, 0.64])  # unit vector
    discriminates_true, discriminates_interp, sens_half, sens_double = 0, 0, 0, 0
    cases = [(52.0, 0.1, -6), (40.0, 0.1, -6), (90.0, 0.1, -7), (11.0, 0.05, -5), (300.0, 0.2, -8), (23.0, 0.1, -5),
             (6.5, 0.1, -3), (52.78, 0.1, -8), (26.4, 0.05, -7), (105.5, 0.2, -9), (13.2, 0.1, -6), (3.3, 0.1, -4)]
    for lam, eta, hlog in cases:
        h = 2.0**hlog
        a0n = 0.37
        L, H = mp.mpf(lam), mp.mpf(h)
        g = (1 - mp.e ** (-L * H)) / H
        crit = mp.mpf(eta) * mp.sqrt(2 / (L * (g + L)))
        lg = mp.log(crit, 2)
        assert abs(lg - mp.nint(lg)) > mp.mpf("1e-6")  # the case does not sit on a power-of-two boundary
        k = int(mp.floor(lg))
        assert 2.0**k < 2 * h  # no doubling limit in play
        # state at t0 and "force" at t1 = h: exact exponential derivatives
        e1 = math.exp(lam * h)
        D = [np.ascontiguousarray((a0n * lam**kk) * u[None, :]) for kk in range(6)] + [np.zeros((1, 3)), np.zeros((1, 3))]
        f = [np.ascontiguousarray((a0n * lam**kk * e1) * u[None, :]) for kk in range(3)]
        t, dt = np.zeros(1), np.full(1, h)
        x, v, ps = np.zeros((1, 3)), np.zeros((1, 3)), np.zeros(1)
        for crit_order in (4, 0):  # explicit and automatic mean the same thing for p = 6
            tt, dd = t.copy(), dt.copy()
            DD = [d.copy() for d in D]
            O.correct(np.array([0], dtype=np.int32), 6, h, eta, 2.0**-40, 1.0, tt, dd, x.copy(), v.copy(), DD, ps.copy(),
                      f[0], f[1], f[2], None, np.zeros(1), crit_order=crit_order)
            assert dd[0] == 2.0**k, (lam, eta, h, dd[0], 2.0**k)
        # what the other two candidate fourth entries would have produced (mpmath, c-7's a3 formula)
        k_true = int(mp.floor(mp.log(mp.mpf(eta) / L, 2)))
        a1 = mp.mpf(a0n) * mp.e ** (L * H)
        a0m, j0, s0 = mp.mpf(a0n), mp.mpf(a0n) * L, mp.mpf(a0n) * L**2
        j1, s1 = a1 * L, a1 * L**2
        a3 = -3 * (20 * (a0m - a1) + 8 * H * j0 + 12 * H * j1 + H**2 * s0 - 3 * H**2 * s1) / H**3
        crit_i = mp.mpf(eta) * mp.sqrt((a1 * s1 + j1**2) / (j1 * abs(a3) + s1**2))
        k_int = int(mp.floor(mp.log(crit_i, 2)))
        discriminates_true += k_true != k
        discriminates_interp += k_int != k
        # a factor-2 slip in cbar (e.g. dividing by 2h, or h/2) must change the result in several cases
        for scale, which in ((mp.mpf("0.5"), "half"), (mp.mpf(2), "double")):
            km = int(mp.floor(mp.log(mp.mpf(eta) * mp.sqrt(2 / (L * (scale * g + L))), 2)))
            if which == "half":
                sens_half += km != k
            else:
                sens_double += km != k
    assert discriminates_true >= 2 and discriminates_interp >= 1, (discriminates_true, discriminates_interp)
    assert sens_half >= 3 and sens_double >= 1, (sens_half, sens_double)


def test_dt_criterion_automatic_option_value():
    """crit_order 0 = automatic = the library's "dt_criterion_order" 0 (include/nbody.h): order p for p = 4, the
    4-derivative criterion for p = 6, 8.  Checked by equality with the explicit values on random inputs."""
    rng = np.random.default_rng(21)
    n = 32
    idx = np.arange(n, dtype=np.int32)
    h = 2.0**-6
    mk = lambda: np.ascontiguousarray(rng.normal(0, 1, (n, 3)))
    for order, same_as, differs_from in ((4, 4, None), (6, 4, 6), (8, 4, 8)):
        base = dict(x=mk(), v=mk(), D=[mk() * 3.0**k for k in range(8)])
        f = [mk() * 3.0**k for k in range(4)]
        res = {}
        for co in {0, same_as, differs_from or same_as}:
            t, dt = np.zeros(n), np.full(n, h)
            x, v, D = base["x"].copy(), base["v"].copy(), [d.copy() for d in base["D"]]
            O.correct(idx, order, h, 0.1, 2.0**-30, 2.0**-2, t, dt, x, v, D, np.zeros(n), f[0], f[1],
                      f[2] if order >= 6 else None, f[3] if order >= 8 else None, np.zeros(n), crit_order=co)
            res[co] = dt
        assert np.array_equal(res[0], res[same_as])
        if differs_from:
            assert np.any(res[0] != res[differs_from])


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
    nb, pairs = OI.integrate(s, 0.125, eps2, 0.1, dt_min, dt_max, crit_order=order)  # c-8, order-p criterion
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
    for co in (order, pc):  # value = order: the order-p criterion of c-8 (0 would mean "automatic", R8b)
        s = dict(t=base["t"].copy(), dt=base["dt"].copy(), x=base["x"].copy(), v=base["v"].copy(),
                 D=[d.copy() for d in base["D"]], pot=base["pot"].copy())
        O.correct(idx, order, h, 0.1, 2.0**-30, 2.0**-2, s["t"], s["dt"], s["x"], s["v"], s["D"], s["pot"],
                  f[0], f[1], f[2], f[3], np.zeros(n), crit_order=co)
        out[co] = s
    a, b = out[order], out[pc]
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


# ------------------------------------------------------------------------------------------- c-9b (R14)
def _flyby(order, reject_ratio, h0=2.0**-4):
    """Two equal masses (M = 1e-3) on a hyperbolic orbit, impact parameter b = 1e-3, v_inf = 1: closest approach
    (r_min = 4.1e-4) falls on the END of the first step h0 = 2^-4 that both particles are started with."""
    m = np.array([5e-4, 5e-4])
    b = 1e-3
    x = np.array([[-h0 / 2, b / 2, 0.0], [h0 / 2, -b / 2, 0.0]])
    v = np.array([[0.5, 0.0, 0.0], [-0.5, 0.0, 0.0]])
    s = OI.bootstrap(m, x, v, order, 0.0, fixed_dt=h0, dt_min=2.0**-40, dt_max=h0)
    e0 = _energy2(s.m, s.x, s.v)
    l0 = np.sum(s.m[:, None] * np.cross(s.x, s.v), axis=0)[2]
    nb, _ = OI.integrate(s, 2 * h0, 0.0, 0.1, 2.0**-40, h0, reject_ratio=reject_ratio)
    assert np.all(s.t == 2 * h0)
    e1 = _energy2(s.m, s.x, s.v)
    l1 = np.sum(s.m[:, None] * np.cross(s.x, s.v), axis=0)[2]
    return abs((e1 - e0) / e0), abs((l1 - l0) / l0), s, nb


@pytest.mark.parametrize("order", [4, 6, 8])
def test_step_rejection_flyby_pin(order):
    """c-9b against the two-body invariants and the closed-form deflection: an encounter whose closest approach sits on
    the end point of a long step wrecks the textbook scheme (the end-point derivatives m v^k / r^(k+2) are extrapolated
    over the whole step: |dE/E| > 1e4), while with reject_ratio = 4 the step is refused, redone on h/4, and energy and
    angular momentum are conserved; the velocity turns by theta = 2 atan(M / (b v_inf^2)) = 90 degrees."""
    bad_e, bad_l, _, _ = _flyby(order, 0)
    good_e, good_l, s, nb = _flyby(order, 4)
    assert bad_e > 1e3
    assert good_e < {4: 1e-6, 6: 1e-9, 8: 1e-10}[order] and good_l < {4: 1e-6, 6: 1e-9, 8: 1e-10}[order]
    assert s.rejected >= 1 and nb > 100
    ang = math.degrees(math.atan2(s.v[0][1], s.v[0][0]))  # started along +x
    assert abs(abs(ang) - 90.0) < 2.5, ang  # asymptotic value 90; the run ends 0.06 = 60 b after the pericentre
    assert abs(np.linalg.norm(s.v[0] - s.v[1]) - 1.0) < 0.02  # |v_rel| back to v_inf (up to the residual potential)


def test_step_rejection_rule_details():
    """c-9b mechanics: a rejected particle keeps x, v, D, pot, t and only gets dt = h/R; the rule never fires when it
    is off, when dt_new > h/R, or when h/R would fall below dt_min."""
    n = 3
    idx = np.arange(n, dtype=np.int32)
    h = 2.0**-6
    ex = np.array([1.0, 0.0, 0.0])
    lam = np.array([1.0, 2.0**9, 2.0**9])  # particle 0: smooth; 1 and 2: dt_crit = eta / lam = 2^-3 / 2^9 = 2^-12
    f = [np.ascontiguousarray(np.outer(lam**k * np.exp(lam * h), ex)) for k in range(2)]  # a(t) = e^(lam t)
    mk = lambda: dict(t=np.zeros(n), dt=np.full(n, h), x=np.ones((n, 3)), v=np.ones((n, 3)),
                      D=[np.ascontiguousarray(np.outer(lam**k, ex)) for k in range(8)], pot=np.zeros(n))
    for R, dtmin, expect in ((0, 2.0**-30, [False, False, False]), (4, 2.0**-30, [False, True, True]),
                             (4, 2.0**-7, [False, False, False]), (2.0**7, 2.0**-30, [False, False, False])):
        s = mk()
        ref = mk()
        nrej = O.correct(idx, 4, h, 0.125, dtmin, 2.0**-2, s["t"], s["dt"], s["x"], s["v"], s["D"], s["pot"], f[0], f[1],
                         None, None, np.full(n, -1.0), crit_order=4, reject_ratio=int(R))
        assert nrej == sum(expect)
        for i in range(n):
            if expect[i]:
                assert s["t"][i] == 0.0 and s["dt"][i] == h / R and s["pot"][i] == 0.0
                assert np.array_equal(s["x"][i], ref["x"][i]) and np.array_equal(s["D"][2][i], ref["D"][2][i])
            else:
                assert s["t"][i] == h and s["pot"][i] == -1.0


# ------------------------------------------------------------------------------------------- N4: P(EC)^n
@pytest.mark.parametrize("order", [4, 6])
def test_pec_n_iteration_removes_secular_energy_drift(order):
    """P(EC)^n (oracle/integrate.block_step n_iter): with a shared constant step the iterated corrector converges to the
    implicit, time-symmetric Hermite scheme, whose energy error on a Kepler ellipse (e = 0.5) stays bounded, while the
    single-pass P(EC)^1 drifts linearly with time -- the textbook property, no formula of ours involved."""
    m = np.array([0.5, 0.5])
    x = np.array([[0.25, 0, 0], [-0.25, 0, 0]])
    v = np.array([[0, math.sqrt(3) / 2, 0], [0, -math.sqrt(3) / 2, 0]])
    dt = 2.0**-5
    drift = {}
    for n_iter in (1, 2, 3):
        s = OI.bootstrap(m, x, v, order, 0.0, fixed_dt=dt)
        e0 = _energy2(s.m, s.x, s.v)
        errs = []
        for T in (16.0, 64.0):
            OI.integrate(s, T, 0.0, 1e-30, dt, dt, crit_order=order, n_iter=n_iter)
            errs.append(abs((_energy2(s.m, s.x, s.v) - e0) / e0))
        drift[n_iter] = errs
    assert drift[1][1] / drift[1][0] > 10.0      # secular growth (4 x the time: ~ 50 x here, the phase error feeds back)
    assert drift[2][1] / drift[2][0] < 1.5 and drift[3][1] / drift[3][0] < 1.5   # bounded
    assert abs(drift[3][1] - drift[2][1]) < 0.05 * drift[2][1]                 # n = 2 is already converged to a few %
    assert drift[2][1] < drift[1][1]


# ------------------------------------------------------------------------------------------- c-6b (R15)
def test_corrector_order_limiter_mechanics():
    """c-6b: M = number of leading quadrature terms with non-increasing norms; a limited step takes x1, v1 from the
    corrector of order 2M.  Checked against the oracle's own LOWER-ORDER correctors on the same inputs (those are pinned
    by polynomial exactness above) and against the trapezoid rule written out; smooth data are left alone."""
    rng = np.random.default_rng(12)
    n = 40
    idx = np.arange(n, dtype=np.int32)
    h = 2.0**-5
    mk = lambda sc: np.ascontiguousarray(rng.normal(0, 1, (n, 3)) * sc)
    for order in (6, 8):
        K = order // 2
        for M in range(1, K + 1):
            # derivative scales: terms T_k ~ h^k |a^(k-1)| fall off up to term M, then jump up
            sc = [1.0, 1.0 / h * 0.1, 1.0 / h**2 * 0.01, 1.0 / h**3 * 0.001]
            for k in range(M, K):
                sc[k] = 1e6 / h**k
            D = [mk(sc[k]) if k < K else mk(1.0) for k in range(8)]
            f = [mk(sc[k]) for k in range(4)]
            f[0] = D[0] + 0.01 * f[0]  # a smooth acceleration: |a1 - a0| << |a0| (level 0 does not fire)
            x0, v0 = mk(1.0), mk(1.0)
            st = lambda: dict(t=np.zeros(n), dt=np.full(n, h), x=x0.copy(), v=v0.copy(), D=[d.copy() for d in D], pot=np.zeros(n))
            a, b = st(), st()
            cnt = {}
            O.correct(idx, order, h, 0.1, 2.0**-40, 1.0, a["t"], a["dt"], a["x"], a["v"], a["D"], a["pot"], f[0], f[1], f[2],
                      f[3] if order == 8 else None, np.zeros(n), limit_order=1, counters=cnt)
            O.correct(idx, order, h, 0.1, 2.0**-40, 1.0, b["t"], b["dt"], b["x"], b["v"], b["D"], b["pot"], f[0], f[1], f[2],
                      f[3] if order == 8 else None, np.zeros(n))
            assert cnt["limited"] == (n if M < K else 0), (order, M, cnt)
            for k in range(order):  # stored derivatives and the new step are those of the unlimited corrector
                assert np.array_equal(a["D"][k], b["D"][k])
            assert np.array_equal(a["dt"], b["dt"])
            if M == K:
                assert np.array_equal(a["x"], b["x"]) and np.array_equal(a["v"], b["v"])
            elif M >= 2:  # equals the order-2M corrector of the oracle on the same inputs
                lo = st()
                O.correct(idx, 2 * M, h, 0.1, 2.0**-40, 1.0, lo["t"], lo["dt"], lo["x"], lo["v"], lo["D"], lo["pot"], f[0], f[1],
                          f[2] if 2 * M >= 6 else None, None, np.zeros(n))
                assert np.array_equal(a["x"], lo["x"]) and np.array_equal(a["v"], lo["v"])
            else:  # trapezoid
                v1 = v0 + (h / 2.0) * (D[0] + f[0])
                x1 = x0 + (h / 2.0) * (v0 + v1)
                assert np.array_equal(a["v"], v1) and np.array_equal(a["x"], x1)


def test_corrector_order_limiter_level_zero_is_the_predictor():
    """c-6b level 0: an end-point acceleration spike (|a1 - a0| > 2 |a0|) makes the step fall back on the particle's own
    Taylor prediction -- exactly oracle_predict's x_p, v_p at tau = h -- while the stored derivatives and the new step
    are still those of the end-point force."""
    rng = np.random.default_rng(13)
    n = 16
    idx = np.arange(n, dtype=np.int32)
    h = 2.0**-6
    mk = lambda: np.ascontiguousarray(rng.normal(0, 1, (n, 3)))
    for order in (4, 6, 8):
        D = [mk() for _ in range(8)]
        f = [mk() for _ in range(4)]
        f[0] = 10.0 * D[0]
        x0, v0 = mk(), mk()
        t, dt, x, v, pot = np.zeros(n), np.full(n, h), x0.copy(), v0.copy(), np.zeros(n)
        Dn = [d.copy() for d in D]
        cnt = {}
        O.correct(idx, order, h, 0.1, 2.0**-40, 1.0, t, dt, x, v, Dn, pot, f[0], f[1], f[2] if order >= 6 else None,
                  f[3] if order >= 8 else None, np.zeros(n), limit_order=1, counters=cnt)
        assert cnt["limited"] == n
        xp, vp, _, _ = O.predict(h, order, np.zeros(n), x0, v0, D)
        assert np.array_equal(x, xp) and np.array_equal(v, vp)
        for k in range(order // 2):
            assert np.array_equal(Dn[k], f[k])
        assert np.all(t == h)


def test_corrector_order_limiter_is_inert_on_smooth_runs_and_tames_the_flyby():
    """c-6b never fires in a benign cluster integration (bit-identical state with and without it), and on the fly-by
    whose closest approach sits on the end point of a long step it cuts the energy error by orders of magnitude without
    going back in time (it cannot restore the accuracy of a resolved encounter: that needs short steps BEFORE the
    encounter, which no end-point rule can give)."""
    c = W.cluster(5, 256)
    runs = []
    for lim in (0, 1):
        s = OI.bootstrap(c["m"], c["x"], c["v"], 8, c["eps2"], dt_max=2.0**-5)
        OI.integrate(s, 2.0**-5, c["eps2"], 0.1, 2.0**-30, 2.0**-5, limit_order=lim)
        runs.append((s.x.copy(), s.v.copy(), s.dt.copy(), s.counters.get("limited", 0)))
    assert runs[1][3] == 0
    for a, b in zip(runs[0][:3], runs[1][:3]):
        assert np.array_equal(a, b)
    for order in (4, 6, 8):
        h0 = 2.0**-4
        errs = []
        for lim in (0, 1):
            m = np.array([5e-4, 5e-4])
            x = np.array([[-h0 / 2, 5e-4, 0.0], [h0 / 2, -5e-4, 0.0]])
            v = np.array([[0.5, 0.0, 0.0], [-0.5, 0.0, 0.0]])
            s = OI.bootstrap(m, x, v, order, 0.0, fixed_dt=h0, dt_min=2.0**-40, dt_max=h0)
            e0 = _energy2(s.m, s.x, s.v)
            OI.integrate(s, 2 * h0, 0.0, 0.1, 2.0**-40, h0, limit_order=lim)
            errs.append(abs((_energy2(s.m, s.x, s.v) - e0) / e0))
            if lim:
                assert s.counters["limited"] >= 1
        assert errs[1] < errs[0] / 1e4 and errs[1] < 3.0, (order, errs)  # O(1) of the TWO-BODY energy: the unresolved pericentre
