"""Seeded synthetic cluster generators -- the ONLY module shared by the CPU oracle's tests and the CUDA path.

It holds none of the method's arithmetic (no predictor, force, corrector or time-step rule): it only draws
initial conditions, Taylor-coefficient inputs, particle times and active lists.  The arrays it returns are
handed unchanged to both sides.

The paper publishes no initial-condition file ("star clusters and galactic nuclei with supermassive black
holes", "real core-halo density structure", "up to a few million bodies": PAPER.md:15 abstract, :23 section 1,
:70 section 3).  BASELINE.json `configs` restates its workloads as seeded synthetic clusters; the recipes below
 stand in for the paper's own files.  Everything is fp64 numpy, one PCG64 stream per
config, seed = 13121789 + config number (1-based).

Units: G = 1, Henon units for the Plummer models (M = 1, E = -1/4, a_P = 3 pi / 16).
"""
from __future__ import annotations

import math

import numpy as np

SEED0 = 13121789
A_PLUMMER = 3.0 * math.pi / 16.0


def rng_for(config: int, stream: int = 0) -> np.random.Generator:
    """Independent PCG64 stream for (config number, purpose)."""
    return np.random.Generator(np.random.PCG64([SEED0 + int(config), int(stream)]))


# ----------------------------------------------------------------------------------------------------
# mass profiles (used only to draw radii and to give the smooth-field Taylor inputs a sensible scale)
# ----------------------------------------------------------------------------------------------------
def plummer_mass(r):
    r = np.asarray(r, dtype=np.float64)
    return r**3 / (r * r + A_PLUMMER**2) ** 1.5


def dehnen1_mass(r):
    r = np.asarray(r, dtype=np.float64)
    return r * r / (1.0 + r) ** 2


def _isotropic(rng, n):
    z = rng.uniform(-1.0, 1.0, n)
    phi = rng.uniform(0.0, 2.0 * math.pi, n)
    s = np.sqrt(1.0 - z * z)
    return np.stack([s * np.cos(phi), s * np.sin(phi), z], axis=1)


def plummer(n: int, rng: np.random.Generator, r_in: float = 0.0, x_out: float = 0.999, mass_total: float = 1.0):
    """Equal-mass Plummer sphere, Henon units, radii truncated at M(<r) = x_out (r <= 22.8 a_P-units).

    r = a_P (X^(-2/3) - 1)^(-1/2), X ~ U(M(<r_in), x_out); speed q sqrt(2) (r^2 + a_P^2)^(-1/4) with q drawn by
    rejection from q^2 (1 - q^2)^(7/2) (envelope 0.1).  Centre-of-mass position and velocity are removed by
    the caller (after any black holes are added)."""
    x_in = float(plummer_mass(r_in)) if r_in > 0.0 else 0.0
    X = rng.uniform(x_in, x_out, n)
    X = np.maximum(X, 1e-300)
    r = A_PLUMMER / np.sqrt(X ** (-2.0 / 3.0) - 1.0)
    pos = r[:, None] * _isotropic(rng, n)
    q = np.empty(n)
    todo = np.arange(n)
    while todo.size:
        qq = rng.uniform(0.0, 1.0, todo.size)
        yy = rng.uniform(0.0, 0.1, todo.size)
        ok = yy < qq * qq * (1.0 - qq * qq) ** 3.5
        q[todo[ok]] = qq[ok]
        todo = todo[~ok]
    speed = q * math.sqrt(2.0) * (r * r + A_PLUMMER**2) ** (-0.25)
    vel = speed[:, None] * _isotropic(rng, n)
    m = np.full(n, mass_total / n)
    return m, pos, vel


def dehnen1(n: int, rng: np.random.Generator, m_bh: float = 0.0, r_in: float = 2e-3, r_out: float = 20.0):
    """Dehnen gamma = 1 (Hernquist) cusp, scale radius 1, stellar mass exactly 1 inside [r_in, r_out].

    r = sqrt(X) / (1 - sqrt(X)), X ~ U(M(<r_in), M(<r_out)); isotropic Gaussian velocities with 1-D
    sigma^2 = (M(<r) + m_bh) / (3 r), speed capped at 0.95 v_esc (not an exact equilibrium; irrelevant for a
    force evaluation)."""
    X = rng.uniform(float(dehnen1_mass(r_in)), float(dehnen1_mass(r_out)), n)
    s = np.sqrt(X)
    r = s / (1.0 - s)
    pos = r[:, None] * _isotropic(rng, n)
    sig = np.sqrt((dehnen1_mass(r) + m_bh) / (3.0 * r))
    vel = rng.normal(0.0, 1.0, (n, 3)) * sig[:, None]
    vesc = np.sqrt(2.0 * (1.0 / (1.0 + r) + m_bh / r))
    sp = np.linalg.norm(vel, axis=1)
    f = np.minimum(1.0, 0.95 * vesc / np.maximum(sp, 1e-300))
    vel = vel * f[:, None]
    m = np.full(n, 1.0 / n)
    return m, pos, vel


def _remove_com(m, x, v):
    M = m.sum()
    x -= (m[:, None] * x).sum(axis=0) / M
    v -= (m[:, None] * v).sum(axis=0) / M


# ----------------------------------------------------------------------------------------------------
# BASELINE.json configs (1-based numbering as in SURVEY.md 8(d))
# ----------------------------------------------------------------------------------------------------
CONFIG_N = {1: 1024, 2: 65536, 3: 262144, 4: 1048576, 5: 2097152}
CONFIG_ORDER = {1: 4, 2: 4, 3: 6, 4: 6, 5: 8}
CONFIG_EPS = {1: 1e-4, 2: 1e-4, 3: 1e-5, 4: 1e-5, 5: 1e-5}


def cluster(config: int, n: int | None = None):
    """Initial conditions of BASELINE.json config `config` (1..5), optionally at a reduced total N (a scaled
    twin with the same structure, used by the parity tests).  N counts the black holes.

    Returns dict(m, x, v [fp64], bh = indices of black holes, model = 'plummer'|'dehnen1', m_bh = total BH mass,
    order, eps2, n)."""
    n = int(CONFIG_N[config] if n is None else n)
    rng = rng_for(config, 0)
    if config in (1, 2):
        m, x, v = plummer(n, rng)
        bh = np.zeros(0, dtype=np.int64)
        model, m_bh = "plummer", 0.0
    elif config == 3:
        m_bh = 0.01
        ms, xs, vs = dehnen1(n - 1, rng, m_bh=m_bh)
        m = np.concatenate([[m_bh], ms])
        x = np.concatenate([np.zeros((1, 3)), xs])
        v = np.concatenate([np.zeros((1, 3)), vs])
        bh = np.array([0])
        model = "dehnen1"
    elif config == 4:
        m_bh = 0.01
        ms, xs, vs = plummer(n - 2, rng, r_in=0.02)
        m = np.concatenate([[0.005, 0.005], ms])
        x = np.concatenate([[[0.005, 0.0, 0.0], [-0.005, 0.0, 0.0]], xs])
        v = np.concatenate([[[0.0, 0.5, 0.0], [0.0, -0.5, 0.0]], vs])
        bh = np.array([0, 1])
        model = "plummer"
    elif config == 5:
        m_bh = 0.01
        ms, xs, vs = plummer(n - 1, rng)
        m = np.concatenate([[m_bh], ms])
        x = np.concatenate([np.zeros((1, 3)), xs])
        v = np.concatenate([np.zeros((1, 3)), vs])
        bh = np.array([0])
        model = "plummer"
    else:
        raise ValueError("config must be 1..5")
    m = np.ascontiguousarray(m, dtype=np.float64)
    x = np.ascontiguousarray(x, dtype=np.float64)
    v = np.ascontiguousarray(v, dtype=np.float64)
    if bh.size == 0:
        _remove_com(m, x, v)
    else:
        # keep the black holes where the config puts them: remove the stars' own centre of mass only
        s = np.ones(n, dtype=bool)
        s[bh] = False
        ms_ = m[s]
        x[s] -= (ms_[:, None] * x[s]).sum(axis=0) / ms_.sum()
        v[s] -= (ms_[:, None] * v[s]).sum(axis=0) / ms_.sum()
    return dict(m=m, x=x, v=v, bh=bh, model=model, m_bh=m_bh, order=CONFIG_ORDER[config],
                eps2=CONFIG_EPS[config] ** 2, n=n, config=config)


def smooth_field_derivs(c: dict, n_derivs: int, stream: int = 1):
    """Quick Taylor-coefficient inputs D_k = a^(k)(t_i), k = 0 .. n_derivs-1 (SURVEY.md 8(d) "quick variant"):
    D_0 = -(M(<r) + M_bh) x / r^3 (smooth field of the model), D_k (k >= 1) isotropic Gaussian of rms
    |D_0| Omega^k with Omega^2 = (M(<r) + M_bh) / r^3.  Black holes: a central BH gets zeros; the members of a BH
    binary get their mutual circular two-body values (acc, jerk = m_o dx/d^3, m_o dv/d^3, then -omega^2 times
    the entry two below).  Input recipe only -- the physically consistent alternative is the oracle's own
    bootstrap (tests do that at small N)."""
    rng = rng_for(c["config"], stream)
    x, v, m, bh = c["x"], c["v"], c["m"], c["bh"]
    n = x.shape[0]
    r = np.linalg.norm(x, axis=1)
    rs = np.where(r > 0.0, r, 1.0)  # a particle at the origin (central BH) is zeroed below
    Mr = plummer_mass(rs) if c["model"] == "plummer" else dehnen1_mass(rs)
    om2 = (Mr + c["m_bh"]) / rs**3
    om2 = np.where(r > 0.0, om2, 0.0)
    D0 = -om2[:, None] * x
    n0 = np.linalg.norm(D0, axis=1)
    om = np.sqrt(om2)
    D = [D0]
    for k in range(1, n_derivs):
        g = rng.normal(0.0, 1.0, (n, 3)) / math.sqrt(3.0)
        D.append(g * (n0 * om**k)[:, None])
    if bh.size == 1:
        for k in range(n_derivs):
            D[k][bh[0]] = 0.0
    elif bh.size == 2:
        a, b = int(bh[0]), int(bh[1])
        dx, dv = x[b] - x[a], v[b] - v[a]
        d3 = np.linalg.norm(dx) ** 3
        w2 = (m[a] + m[b]) / d3
        for (i, mo, sg) in ((a, m[b], 1.0), (b, m[a], -1.0)):
            seq = [sg * mo * dx / d3, sg * mo * dv / d3]
            while len(seq) < n_derivs:
                seq.append(-w2 * seq[-2])
            for k in range(n_derivs):
                D[k][i] = seq[k]
    return [np.ascontiguousarray(d) for d in D]


def predictor_times(x: np.ndarray, t_now: float = 2.0**-10):
    """Particle times for predictor tests: dt_i = 2^-k_i, k_i = 10 + min(6, floor(-log2
    clamp(r_i, 2^-6, 1))), t_i = t_now - dt_i (so every particle is due exactly at t_now)."""
    r = np.clip(np.linalg.norm(x, axis=1), 2.0**-6, 1.0)
    k = 10 + np.minimum(6, np.floor(-np.log2(r))).astype(np.int64)
    dt = np.ldexp(1.0, -k)
    t = t_now - dt
    return np.ascontiguousarray(t), np.ascontiguousarray(dt)


def active_list(n: int, n_act: int, rng: np.random.Generator) -> np.ndarray:
    """Ascending unique int32 indices; n_act == n gives 0..n-1."""
    if n_act >= n:
        return np.arange(n, dtype=np.int32)
    return np.sort(rng.choice(n, size=n_act, replace=False)).astype(np.int32)


def oracle_sample(c: dict, size: int = 1024, n_edge: int = 32, stream: int = 2, n_outer: int | None = None) -> np.ndarray:
    """i-particles on which the oracle is evaluated when N is too large for all of them:
    a seeded uniform draw plus forced members -- every BH, the n_edge innermost and the n_outer (default n_edge)
    outermost particles and the n_edge particles nearest to each BH (where mixed-precision errors are largest).
    Ascending, unique."""
    rng = rng_for(c["config"], stream)
    x, bh = c["x"], c["bh"]
    n = x.shape[0]
    if size >= n:
        return np.arange(n, dtype=np.int32)
    r = np.linalg.norm(x, axis=1)
    forced = [np.asarray(bh, dtype=np.int64)]
    ne = min(n_edge, n)
    order = np.argpartition(r, ne - 1)[:ne]
    forced.append(order)
    no = min(n_edge if n_outer is None else n_outer, n)
    order = np.argpartition(-r, no - 1)[:no]
    forced.append(order)
    for b in bh:
        d = np.linalg.norm(x - x[b], axis=1)
        forced.append(np.argpartition(d, ne)[: ne + 1])
    forced = np.unique(np.concatenate(forced))
    rest = max(0, size - forced.size)
    draw = rng.choice(n, size=rest, replace=False)
    return np.unique(np.concatenate([forced, draw])).astype(np.int32)


def block_histogram(n: int, n_calls: int, rng: np.random.Generator) -> np.ndarray:
    """Block sizes for the config-4 histogram: N_act = floor(2^u), u ~ U(0, log2 n)."""
    u = rng.uniform(0.0, math.log2(n), n_calls)
    return np.minimum(n, np.floor(2.0**u)).astype(np.int64)
