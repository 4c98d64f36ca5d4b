"""ctypes access to oracle/liboracle.so -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

numpy-in / numpy-out wrappers, argument marshalling only; every formula lives in nbody_oracle.c
(which cites SURVEY.md 8(c) item by item; the paper itself, names the scheme only).
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import this.
It imports nothing from the CUDA package.
"""
import ctypes as C
import numpy as np

from . import build as _build

_lib = None
_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        L.oracle_num_threads.restype = C.c_int
        L.oracle_set_num_threads.argtypes = [C.c_int]
        L.oracle_predict.argtypes = [C.c_int64, C.c_double, C.c_int, _dp, _dp, _dp, C.POINTER(_dp), _dp, _dp, _dp, _dp]
        L.oracle_predict.restype = None
        L.oracle_force.argtypes = [C.c_int64, _dp, _dp, _dp, _dp, _dp, _ip, C.c_int64, C.c_int, C.c_double,
                                   _dp, _dp, _dp, _dp, _dp]
        L.oracle_force.restype = None
        L.oracle_force_abs.argtypes = [C.c_int64, _dp, _dp, _dp, _dp, _dp, _ip, C.c_int64, C.c_int, C.c_double,
                                       _dp, _dp, _dp, _dp]
        L.oracle_force_abs.restype = None
        L.oracle_nearest.argtypes = [C.c_int64, _dp, _ip, C.c_int64, _ip, _dp]
        L.oracle_nearest.restype = None
        L.oracle_new_dt.argtypes = [C.c_int, C.POINTER(_dp), C.c_double, C.c_double, C.c_double, C.c_double, C.c_double]
        L.oracle_new_dt.restype = C.c_double
        L.oracle_initial_dt.argtypes = [C.c_int64, _dp, _dp, C.c_double, C.c_double, C.c_double, _dp]
        L.oracle_initial_dt.restype = None
        L.oracle_correct.argtypes = [_ip, C.c_int64, C.c_int, C.c_double, C.c_double, C.c_double, C.c_double,
                                     _dp, _dp, _dp, _dp, C.POINTER(_dp), _dp, _dp, _dp, _dp, _dp, _dp, C.c_int, C.c_int,
                                     C.c_int, C.POINTER(C.c_int64), C.c_int, C.POINTER(C.c_int64)]
        L.oracle_correct.restype = None
        L.oracle_next_block.argtypes = [C.c_int64, _dp, _dp, _dp, _ip]
        L.oracle_next_block.restype = C.c_int64
        L.oracle_energy.argtypes = [C.c_int64, _dp, _dp, _dp, _dp, _dp]
        L.oracle_energy.restype = None
        _lib = L
    return _lib


def num_threads() -> int:
    return lib().oracle_num_threads()


def set_num_threads(n: int) -> None:
    lib().oracle_set_num_threads(int(n))


def _d(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a


def _p(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _ptr_array(arrs, n):
    t = (_dp * n)()
    for k in range(n):
        t[k] = _p(arrs[k]) if k < len(arrs) and arrs[k] is not None else None
    return t


def predict(t_now, order, t, x, v, D):
    """c-5.  D = list of a^(k) arrays, k = 0..order-3.  Returns xp, vp, ap, jp (None where not defined)."""
    t, x, v = _d(t), _d(x), _d(v)
    D = [_d(a) for a in D[: order - 2]]
    assert len(D) == order - 2
    n = t.shape[0]
    xp, vp = np.empty((n, 3)), np.empty((n, 3))
    ap = np.empty((n, 3)) if order >= 6 else None
    jp = np.empty((n, 3)) if order >= 8 else None
    lib().oracle_predict(n, float(t_now), order, _p(t), _p(x), _p(v), _ptr_array(D, 6), _p(xp), _p(vp), _p(ap), _p(jp))
    return xp, vp, ap, jp


def force(m, xp, vp, ap, jp, active_idx, order, eps2):
    """c-1..c-4.  Returns acc, jerk, snap, crackle, pot in active-list order (None where not defined)."""
    m, xp, vp = _d(m), _d(xp), _d(vp)
    ap = _d(ap) if ap is not None else None
    jp = _d(jp) if jp is not None else None
    if order >= 6:
        assert ap is not None
    if order >= 8:
        assert jp is not None
    idx = np.ascontiguousarray(active_idx, dtype=np.int32)
    n, na = m.shape[0], idx.shape[0]
    acc, jerk, pot = np.empty((na, 3)), np.empty((na, 3)), np.empty(na)
    snap = np.empty((na, 3)) if order >= 6 else None
    crk = np.empty((na, 3)) if order >= 8 else None
    lib().oracle_force(n, _p(m), _p(xp), _p(vp), _p(ap), _p(jp), idx.ctypes.data_as(_ip), na, order, float(eps2),
                       _p(acc), _p(jerk), _p(snap), _p(crk), _p(pot))
    return acc, jerk, snap, crk, pot


def force_abs(m, xp, vp, ap, jp, active_idx, order, eps2):
    """c-16: Sum_j |pair term| per active particle for acc, jerk, snap, crackle (None above the order); divide by the
    norm of oracle force's sum to get the conditioning number kappa >= 1."""
    m, xp, vp = _d(m), _d(xp), _d(vp)
    ap = _d(ap) if ap is not None else None
    jp = _d(jp) if jp is not None else None
    idx = np.ascontiguousarray(active_idx, dtype=np.int32)
    n, na = m.shape[0], idx.shape[0]
    a, j = np.empty(na), np.empty(na)
    s = np.empty(na) if order >= 6 else None
    c = np.empty(na) if order >= 8 else None
    lib().oracle_force_abs(n, _p(m), _p(xp), _p(vp), _p(ap), _p(jp), idx.ctypes.data_as(_ip), na, order, float(eps2),
                           _p(a), _p(j), _p(s), _p(c))
    return a, j, s, c


def nearest(xp, active_idx):
    """c-17: (index, squared distance in the force kernel's fp32) of the nearest other particle of each active one."""
    xp = _d(xp)
    idx = np.ascontiguousarray(active_idx, dtype=np.int32)
    who = np.empty(idx.shape[0], dtype=np.int32)
    r2 = np.empty(idx.shape[0])
    lib().oracle_nearest(xp.shape[0], _p(xp), idx.ctypes.data_as(_ip), idx.shape[0], who.ctypes.data_as(_ip), _p(r2))
    return who, r2


def new_dt(order, derivs, t1, dt_old, eta, dt_min, dt_max):
    """c-8 + c-9 for one particle; derivs = list of 3-vectors a^(0..order-1)(t1)."""
    d = [_d(a) for a in derivs[:order]]
    return lib().oracle_new_dt(order, _ptr_array(d, 8), float(t1), float(dt_old), float(eta), float(dt_min), float(dt_max))


def initial_dt(acc, jerk, eta_s, dt_min, dt_max):
    acc, jerk = _d(acc), _d(jerk)
    dt = np.empty(acc.shape[0])
    lib().oracle_initial_dt(acc.shape[0], _p(acc), _p(jerk), float(eta_s), float(dt_min), float(dt_max), _p(dt))
    return dt


def correct(active_idx, order, t_now, eta, dt_min, dt_max, t, dt, x, v, D, pot_state, acc, jerk, snap, crackle, pot,
            variant=0, crit_order=0, reject_ratio=0, limit_order=0, counters=None):
    """c-6..c-9 (+ c-8b crit_order, c-9b reject_ratio), IN PLACE on t, dt, x, v, D[0..order-1], pot_state (all must be
    C-contiguous float64 arrays).  crit_order: 0 = automatic (criterion order 4 for order >= 6, else the order), the same
    meaning as the library's "dt_criterion_order" 0; 4 | 6 | 8 = min(order, value) (value = order: the order-p criterion
    of c-8).  reject_ratio: 0 = no step rejection; R = 2^r >= 2 = c-9b.  limit_order: 1 = c-6b corrector order limiter.
    Returns the number of rejected steps; `counters` (a dict) gets "limited" += the number of order-limited steps."""
    idx = np.ascontiguousarray(active_idx, dtype=np.int32)
    for a in (t, dt, x, v, pot_state, *D[:order]):
        assert a.dtype == np.float64 and a.flags.c_contiguous
    acc, jerk, pot = _d(acc), _d(jerk), _d(pot)
    snap = _d(snap) if snap is not None else None
    crackle = _d(crackle) if crackle is not None else None
    nrej, nlim = C.c_int64(0), C.c_int64(0)
    lib().oracle_correct(idx.ctypes.data_as(_ip), idx.shape[0], order, float(t_now), float(eta), float(dt_min),
                         float(dt_max), _p(t), _p(dt), _p(x), _p(v), _ptr_array(D, 8), _p(pot_state),
                         _p(acc), _p(jerk), _p(snap), _p(crackle), _p(pot), int(variant), int(crit_order),
                         int(reject_ratio), C.byref(nrej), int(limit_order), C.byref(nlim))
    if counters is not None:
        counters["limited"] = counters.get("limited", 0) + int(nlim.value)
    return int(nrej.value)


def next_block(t, dt):
    """a-1 / c-11.  Returns (t_next, active_idx int32 ascending)."""
    t, dt = _d(t), _d(dt)
    n = t.shape[0]
    idx = np.empty(n, dtype=np.int32)
    tn = C.c_double()
    na = lib().oracle_next_block(n, _p(t), _p(dt), C.cast(C.byref(tn), _dp), idx.ctypes.data_as(_ip))
    return tn.value, idx[:na].copy()


def energy(m, v, pot):
    m, v, pot = _d(m), _d(v), _d(pot)
    k, w = C.c_double(), C.c_double()
    lib().oracle_energy(m.shape[0], _p(m), _p(v), _p(pot), C.cast(C.byref(k), _dp), C.cast(C.byref(w), _dp))
    return k.value, w.value
