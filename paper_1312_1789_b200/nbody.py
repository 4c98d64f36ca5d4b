"""Thin ctypes binding of libnbody.so (include/nbody.h) -- argument marshalling only.

Every step of the path runs in the CUDA kernels of csrc/; torch supplies device memory (`tensor.data_ptr()`) and
the current stream, nothing else.  Importing this module fails loudly when csrc/libnbody.so is missing: there
is no CPU fallback (BASELINE.json north_star), and nothing here imports `oracle/`.
Names follow the C ABI: Context.predict / force / correct / next_block / initial_dt / get_predicted / run_blocks /
pack_rows / unpack_rows / force_host / step_host (include/nbody.h) and probe_peak (include/nbody_bench.h).
"""
import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("NBODY_LIBRARY") or os.path.join(_HERE, "csrc", "libnbody.so")  # override: another build

if not os.path.exists(LIB_PATH):
    raise ImportError(
        "paper_1312_1789_b200: %s is missing -- build it with `python -m paper_1312_1789_b200.build` "
        "(or __graft_entry__.build()); there is no CPU fallback." % LIB_PATH)

_lib = C.CDLL(LIB_PATH)

OK, EINVAL, ESTATE, ECUDA, ENOMEM, ESCRATCH = 0, -1, -2, -3, -4, -5
FORCE_STATIC_SCRATCH_BYTES = 16 * 1024 * 1024  # NBODY_FORCE_STATIC_SCRATCH_BYTES (include/nbody.h)

_vp = C.c_void_p
_i64 = C.c_int64
_dbl = C.c_double

class RunResult(C.Structure):
    """nbody_run_result of include/nbody.h."""
    _fields_ = [("blocks", C.c_int64), ("pairs", C.c_int64), ("t_next", C.c_double), ("n_act_next", C.c_int64),
                ("stop_reason", C.c_int32), ("reserved", C.c_int32), ("rejected", C.c_int64), ("limited", C.c_int64),
                ("hist_log2", C.c_int64 * 40)]


# every symbol include/nbody.h and include/nbody_bench.h declare, with its signature
SIGNATURES = {
    "nbody_abi_version": (C.c_int, []),
    "nbody_strerror": (C.c_char_p, [C.c_int]),
    "nbody_create": (C.c_int, [C.POINTER(_vp), _i64, C.c_int]),
    "nbody_workspace_bytes": (_i64, [_i64]),
    "nbody_destroy": (C.c_int, [_vp]),
    "nbody_last_cuda_error": (C.c_int, [_vp]),
    "nbody_set_option": (C.c_int, [_vp, C.c_char_p, _i64]),
    "nbody_predict": (C.c_int, [_vp, _i64, _dbl, C.c_int, _vp, _vp, _vp, _vp, C.POINTER(_vp), _vp]),
    "nbody_force": (C.c_int, [_vp, _vp, _i64, C.c_int, _dbl, _vp, _vp, _vp, _vp, _vp, _vp]),
    "nbody_force_static": (C.c_int, [_vp, _vp, _i64, C.c_int, _dbl, _vp, _vp, _vp, _vp, _vp, _vp]),
    "nbody_correct": (C.c_int, [_vp, _vp, _i64, C.c_int, _dbl, _dbl, _dbl, _dbl, _vp, _vp, _vp, _vp, C.POINTER(_vp),
                                _vp, _vp, _vp, _vp, _vp, _vp, _vp]),
    "nbody_initial_dt": (C.c_int, [_vp, _i64, _vp, _vp, _dbl, _dbl, _dbl, _vp, _vp]),
    "nbody_next_block": (C.c_int, [_vp, _i64, _vp, _vp, _vp, C.POINTER(_dbl), C.POINTER(_i64), _vp]),
    "nbody_get_predicted": (C.c_int, [_vp, _vp, _vp, _vp, _vp, _vp, _vp]),
    "nbody_nearest": (C.c_int, [_vp, _vp, _i64, _vp, _vp, _vp]),
    "nbody_rejected_steps": (C.c_int, [_vp, C.c_int, C.POINTER(_i64), _vp]),
    "nbody_run_blocks": (C.c_int, [_vp, _i64, C.c_int, _dbl, _dbl, _dbl, _dbl, _dbl, _i64, _i64, _vp, _vp, _vp, _vp, _vp,
                                   C.POINTER(_vp), _vp, _vp, _vp, _vp, _vp, _vp, _vp, C.POINTER(RunResult), _vp]),
    "nbody_pack_rows": (C.c_int, [_vp, _vp, _i64, C.c_int, _vp, _vp, _vp, _vp, _vp, C.POINTER(_vp), _vp, _vp]),
    "nbody_unpack_rows": (C.c_int, [_vp, _vp, _i64, C.c_int, _vp, _vp, _vp, _vp, _vp, C.POINTER(_vp), _vp, _vp]),
    "nbody_force_host": (C.c_int, [_vp, _i64, _dbl, C.c_int, _vp, _vp, _vp, _vp, C.POINTER(_vp), _vp, _i64, _dbl,
                                   _vp, _vp, _vp, _vp, _vp, C.POINTER(_i64), C.POINTER(_i64)]),
    "nbody_step_host": (C.c_int, [_vp, _i64, C.c_int, _dbl, _dbl, _dbl, _dbl, _vp, _vp, _vp, _vp, _vp, C.POINTER(_vp),
                                  _vp, C.POINTER(_dbl), C.POINTER(_i64), C.POINTER(_i64), C.POINTER(_i64)]),
    "nbody_probe_peak": (C.c_int, [_vp, C.c_int, C.c_int, C.POINTER(_dbl)]),
    "nbody_launch_count": (_i64, [_vp]),
    "nbody_last_force_geometry": (C.c_int, [_vp, C.POINTER(C.c_int), C.POINTER(C.c_int), C.POINTER(C.c_int),
                                            C.POINTER(_i64)]),
}
for _name, (_res, _args) in SIGNATURES.items():
    _f = getattr(_lib, _name)  # AttributeError here = the library does not export what the header declares
    _f.restype = _res
    _f.argtypes = _args


class NBodyError(RuntimeError):
    def __init__(self, code, where, cuda_error=0):
        self.code = code
        self.cuda_error = cuda_error
        msg = _lib.nbody_strerror(code).decode()
        if cuda_error:
            msg += " [cudaError %d]" % cuda_error
        super().__init__("%s: %s (%d)" % (where, msg, code))


def strerror(code: int) -> str:
    return _lib.nbody_strerror(int(code)).decode()


def abi_version() -> int:
    return _lib.nbody_abi_version()


def workspace_bytes(n_capacity: int) -> int:
    return int(_lib.nbody_workspace_bytes(int(n_capacity)))


def _ptr(a):
    """Device (torch) or host (numpy) array -> address; None -> NULL."""
    if a is None:
        return None
    if hasattr(a, "data_ptr"):
        assert a.is_contiguous(), "nbody: tensors must be contiguous"
        return a.data_ptr()
    assert a.flags.c_contiguous, "nbody: arrays must be C-contiguous"
    return a.ctypes.data


def _ptr_array(arrs, n):
    t = (_vp * n)()
    for k in range(n):
        t[k] = _ptr(arrs[k]) if k < len(arrs) and arrs[k] is not None else None
    return t


def _stream(stream):
    if stream is not None:
        return int(stream)
    import torch
    return torch.cuda.current_stream().cuda_stream


class Context:
    """Owns one nbody_ctx (scratch only: packed j-store, split partials, staging)."""

    def __init__(self, n_capacity: int, device: int = 0):
        self._h = _vp()
        rc = _lib.nbody_create(C.byref(self._h), int(n_capacity), int(device))
        if rc != OK:
            self._h = _vp()
            raise NBodyError(rc, "nbody_create")
        self.capacity = int(n_capacity)
        self.device = int(device)

    def _check(self, rc, where):
        if rc != OK:
            raise NBodyError(rc, where, _lib.nbody_last_cuda_error(self._h))

    def close(self):
        if getattr(self, "_h", None) is not None and self._h:
            _lib.nbody_destroy(self._h)
            self._h = _vp()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_option(self, key: str, value: int):
        self._check(_lib.nbody_set_option(self._h, key.encode(), int(value)), "nbody_set_option")

    def predict(self, n, t_now, order, t, m, x, v, a_derivs, stream=None):
        self._check(_lib.nbody_predict(self._h, int(n), float(t_now), int(order), _ptr(t), _ptr(m), _ptr(x), _ptr(v),
                                       _ptr_array(a_derivs, 6), _stream(stream)), "nbody_predict")

    def force(self, active_idx, n_act, order, eps2, acc, jerk, snap, crackle, pot, stream=None):
        self._check(_lib.nbody_force(self._h, _ptr(active_idx), int(n_act), int(order), float(eps2), _ptr(acc),
                                     _ptr(jerk), _ptr(snap), _ptr(crackle), _ptr(pot), _stream(stream)), "nbody_force")

    def force_static(self, active_idx, n_act, order, eps2, acc, jerk, snap, crackle, pot, stream=None):
        """nbody_force with the j-split scratch in the library's static device array (no allocation; the launch
        must need <= FORCE_STATIC_SCRATCH_BYTES, else NBODY_ESCRATCH)."""
        self._check(_lib.nbody_force_static(self._h, _ptr(active_idx), int(n_act), int(order), float(eps2), _ptr(acc),
                                            _ptr(jerk), _ptr(snap), _ptr(crackle), _ptr(pot), _stream(stream)),
                    "nbody_force_static")

    def correct(self, active_idx, n_act, order, t_now, eta, dt_min, dt_max, t, dt, x, v, a_derivs, pot_state,
                acc, jerk, snap, crackle, pot, stream=None):
        self._check(_lib.nbody_correct(self._h, _ptr(active_idx), int(n_act), int(order), float(t_now), float(eta),
                                       float(dt_min), float(dt_max), _ptr(t), _ptr(dt), _ptr(x), _ptr(v),
                                       _ptr_array(a_derivs, 8), _ptr(pot_state), _ptr(acc), _ptr(jerk), _ptr(snap),
                                       _ptr(crackle), _ptr(pot), _stream(stream)), "nbody_correct")

    def nearest(self, active_idx, n_act, nn_idx, nn_r2, stream=None):
        """N4 neighbour output: index (int32) and squared distance (fp64 holding the fp32 value) of the nearest other
        particle of each active one, at the positions of the last predict."""
        self._check(_lib.nbody_nearest(self._h, _ptr(active_idx), int(n_act), _ptr(nn_idx), _ptr(nn_r2), _stream(stream)),
                    "nbody_nearest")

    def initial_dt(self, n, acc, jerk, eta_s, dt_min, dt_max, dt, stream=None):
        self._check(_lib.nbody_initial_dt(self._h, int(n), _ptr(acc), _ptr(jerk), float(eta_s), float(dt_min),
                                          float(dt_max), _ptr(dt), _stream(stream)), "nbody_initial_dt")

    def next_block(self, n, t, dt, active_idx, stream=None):
        """Returns (t_next, n_act); active_idx[:n_act] is filled on the device."""
        tn, na = _dbl(), _i64()
        self._check(_lib.nbody_next_block(self._h, int(n), _ptr(t), _ptr(dt), _ptr(active_idx), C.byref(tn),
                                          C.byref(na), _stream(stream)), "nbody_next_block")
        return tn.value, na.value

    def get_predicted(self, xp, vp, ap, jp, m32, stream=None):
        self._check(_lib.nbody_get_predicted(self._h, _ptr(xp), _ptr(vp), _ptr(ap), _ptr(jp), _ptr(m32),
                                             _stream(stream)), "nbody_get_predicted")

    def run_blocks(self, n, order, eps2, eta, dt_min, dt_max, t_end, max_blocks, max_n_act, t, dt, m, x, v, a_derivs,
                   pot_state, active_idx, acc, jerk, snap, crackle, pot, stream=None):
        """Device-driven block steps (nbody_run_blocks).  Returns dict(blocks, pairs, t_next, n_act_next, stop_reason,
        hist_log2)."""
        r = RunResult()
        self._check(_lib.nbody_run_blocks(self._h, int(n), int(order), float(eps2), float(eta), float(dt_min),
                                          float(dt_max), float(t_end), int(max_blocks), int(max_n_act), _ptr(t),
                                          _ptr(dt), _ptr(m), _ptr(x), _ptr(v), _ptr_array(a_derivs, 8), _ptr(pot_state),
                                          _ptr(active_idx), _ptr(acc), _ptr(jerk), _ptr(snap), _ptr(crackle), _ptr(pot),
                                          C.byref(r), _stream(stream)), "nbody_run_blocks")
        return dict(blocks=r.blocks, pairs=r.pairs, t_next=r.t_next, n_act_next=r.n_act_next,
                    stop_reason=r.stop_reason, rejected=r.rejected, limited=r.limited, hist_log2=list(r.hist_log2))

    def rejected_steps(self, reset=False, stream=None) -> int:
        return self.step_counters(reset, stream)[0]

    def step_counters(self, reset=False, stream=None):
        """(steps refused by R14, steps order-limited by R15) since the last reset."""
        v = (_i64 * 2)()
        self._check(_lib.nbody_rejected_steps(self._h, int(bool(reset)), v, _stream(stream)), "nbody_rejected_steps")
        return int(v[0]), int(v[1])

    def pack_rows(self, idx, n_rows, order, t, dt, pot_state, x, v, a_derivs, rec, stream=None):
        self._check(_lib.nbody_pack_rows(self._h, _ptr(idx), int(n_rows), int(order), _ptr(t), _ptr(dt), _ptr(pot_state),
                                         _ptr(x), _ptr(v), _ptr_array(a_derivs, 8), _ptr(rec), _stream(stream)),
                    "nbody_pack_rows")

    def unpack_rows(self, idx, n_rows, order, t, dt, pot_state, x, v, a_derivs, rec, stream=None):
        self._check(_lib.nbody_unpack_rows(self._h, _ptr(idx), int(n_rows), int(order), _ptr(t), _ptr(dt),
                                           _ptr(pot_state), _ptr(x), _ptr(v), _ptr_array(a_derivs, 8), _ptr(rec),
                                           _stream(stream)), "nbody_unpack_rows")

    def force_host(self, n, t_now, order, t, m, x, v, a_derivs, active_idx, n_act, eps2, acc, jerk, snap, crackle, pot):
        """HOST (numpy) buffers in and out; returns (h2d_bytes, d2h_bytes)."""
        up, down = _i64(), _i64()
        self._check(_lib.nbody_force_host(self._h, int(n), float(t_now), int(order), _ptr(t), _ptr(m), _ptr(x),
                                          _ptr(v), _ptr_array(a_derivs, 6), _ptr(active_idx), int(n_act), float(eps2),
                                          _ptr(acc), _ptr(jerk), _ptr(snap), _ptr(crackle), _ptr(pot),
                                          C.byref(up), C.byref(down)), "nbody_force_host")
        return up.value, down.value

    def step_host(self, n, order, eps2, eta, dt_min, dt_max, t, dt, m, x, v, a_derivs, pot_state):
        """One whole block step on HOST (numpy) state, in place; returns (t_next, n_act, h2d_bytes, d2h_bytes)."""
        tn, na, up, down = _dbl(), _i64(), _i64(), _i64()
        self._check(_lib.nbody_step_host(self._h, int(n), int(order), float(eps2), float(eta), float(dt_min),
                                         float(dt_max), _ptr(t), _ptr(dt), _ptr(m), _ptr(x), _ptr(v),
                                         _ptr_array(a_derivs, 8), _ptr(pot_state), C.byref(tn), C.byref(na),
                                         C.byref(up), C.byref(down)), "nbody_step_host")
        return tn.value, na.value, up.value, down.value

    def probe_peak(self, kind: int, millis: int = 200):
        """Returns (1e12 thread-ops/s, SM MHz measured inside the probe kernel)."""
        r = (_dbl * 2)()
        self._check(_lib.nbody_probe_peak(self._h, int(kind), int(millis), r), "nbody_probe_peak")
        return r[0], r[1]

    def launch_count(self) -> int:
        return int(_lib.nbody_launch_count(self._h))

    def last_force_geometry(self):
        r, jl, s, ctas = C.c_int(), C.c_int(), C.c_int(), _i64()
        self._check(_lib.nbody_last_force_geometry(self._h, C.byref(r), C.byref(jl), C.byref(s), C.byref(ctas)),
                    "nbody_last_force_geometry")
        return dict(i_per_thread=r.value, j_lanes=jl.value, j_splits=s.value, ctas=ctas.value)
