"""ctypes wrapper around oracle/hermite_oracle.c -- TEST INFRASTRUCTURE, not product.

Argument marshalling only; every formula lives in the C file, which cites the paper passage it follows.
Parity unpinned (paper silent): the value of dt_min only.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "hermite_oracle.c"
_LIB = _HERE / "libhermite_oracle.so"

#: reading R6: largest / smallest block step, exact powers of two
DT_MAX = 2.0 ** -3
DT_MIN = 2.0 ** -23

_lib = None


def build(force: bool = False) -> Path:
    """Compile the oracle with gcc (-O2, no contraction, no fast-math)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".tmp{os.getpid()}.so")
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fvisibility=hidden",
               "-shared", "-fPIC", "-std=c11", "-o", str(tmp), str(_SRC), "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)
_lp = C.POINTER(C.c_int64)


class _State(C.Structure):
    _fields_ = [
        ("n", C.c_int64),
        ("eps2", C.c_double), ("eta", C.c_double), ("dt_min", C.c_double), ("dt_max", C.c_double),
        ("halving_mode", C.c_int32), ("acc_mode", C.c_int32),
        ("t", C.c_double),
        ("m", _dp), ("x", _dp), ("v", _dp), ("a", _dp), ("j", _dp), ("t_i", _dp), ("dt", _dp),
        ("xp", _dp), ("vp", _dp), ("a1", _dp), ("j1", _dp),
        ("active", _ip),
        ("n_act", C.c_int64),
        ("block_steps", C.c_int64), ("particle_steps", C.c_int64),
        ("diag", C.c_int64 * 2),
        ("min_margin", C.c_double),
        ("level_hist", C.c_int64 * 64),
        ("sec_force", C.c_double), ("sec_total", C.c_double),
    ]


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(str(build()))
        lib.orc_num_threads.restype = C.c_int
        lib.orc_set_num_threads.argtypes = [C.c_int]
        lib.orc_pairsum.argtypes = [C.c_int64, _dp, _dp, _dp, C.c_double, _ip, C.c_int64, _dp, _dp, C.c_int]
        lib.orc_pairsum.restype = None
        lib.orc_pairsum_longdouble.argtypes = [C.c_int64, _dp, _dp, _dp, C.c_double, C.c_void_p, C.c_void_p]
        lib.orc_pairsum_longdouble.restype = None
        lib.orc_block_init.argtypes = [C.c_double] * 3
        lib.orc_block_init.restype = C.c_double
        lib.orc_block_update.argtypes = [C.c_double] * 5 + [C.c_int]
        lib.orc_block_update.restype = C.c_double
        lib.orc_initial_dt.argtypes = [C.c_int64, _dp, _dp, C.c_double, C.c_double, C.c_double, _dp]
        lib.orc_initial_dt.restype = None
        lib.orc_next_block.argtypes = [C.c_int64, _dp, _dp, _ip, _lp]
        lib.orc_next_block.restype = C.c_double
        lib.orc_predict.argtypes = [C.c_int64, C.c_double, _dp, _dp, _dp, _dp, _dp, _dp, _dp]
        lib.orc_predict.restype = None
        lib.orc_correct.argtypes = [C.c_int64, _ip, C.c_double, C.c_double, C.c_double, C.c_double, C.c_int,
                                    _dp, _dp, _dp, _dp, _dp, _dp, _dp, _dp, _dp, _dp, _lp, _dp, _dp]
        lib.orc_correct.restype = None
        lib.orc_energy.argtypes = [C.c_int64, _dp, _dp, _dp, C.c_double, _dp, _dp]
        lib.orc_energy.restype = None
        lib.orc_state_size.restype = C.c_int64
        lib.orc_init.argtypes = [C.POINTER(_State)]
        lib.orc_init.restype = None
        lib.orc_step.argtypes = [C.POINTER(_State)]
        lib.orc_step.restype = C.c_double
        lib.orc_run.argtypes = [C.POINTER(_State), C.c_double, C.c_int64, _dp, _lp, C.POINTER(C.c_uint64), C.c_int64]
        lib.orc_run.restype = C.c_int64
        assert lib.orc_state_size() == C.sizeof(_State), "orc_state layout mismatch"
        _lib = lib
    return _lib


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def _p(a: np.ndarray):
    return a.ctypes.data_as(_dp)


def num_threads() -> int:
    return int(_load().orc_num_threads())


def set_num_threads(n: int) -> None:
    _load().orc_set_num_threads(int(n))


def pairsum(m, x, v, eps, idx=None, mode: str = "compensated"):
    """(a, jerk) for the particles in ``idx`` (all if None) summed over all sources; arrays [n_act,3]."""
    lib = _load()
    m, x, v = _f64(m), _f64(x), _f64(v)
    n = m.shape[0]
    if idx is None:
        ip, n_act = None, n
    else:
        idx = np.ascontiguousarray(idx, dtype=np.int32)
        ip, n_act = idx.ctypes.data_as(_ip), idx.shape[0]
    a = np.zeros((n_act, 3))
    j = np.zeros((n_act, 3))
    lib.orc_pairsum(n, _p(m), _p(x), _p(v), float(eps) ** 2, ip, n_act, _p(a), _p(j),
                    {"plain": 0, "compensated": 1}[mode])
    return a, j


def pairsum_longdouble(m, x, v, eps):
    """All-long-double brute force (N <= a few hundred); returns numpy longdouble arrays."""
    lib = _load()
    m, x, v = _f64(m), _f64(x), _f64(v)
    n = m.shape[0]
    a = np.zeros((n, 3), dtype=np.longdouble)
    j = np.zeros((n, 3), dtype=np.longdouble)
    assert a.itemsize == 16
    lib.orc_pairsum_longdouble(n, _p(m), _p(x), _p(v), float(eps) ** 2, a.ctypes.data, j.ctypes.data)
    return a, j


def block_init(value: float, dt_min: float = DT_MIN, dt_max: float = DT_MAX) -> float:
    return float(_load().orc_block_init(value, dt_min, dt_max))


def block_update(h, dt_req, t_new, dt_min=DT_MIN, dt_max=DT_MAX, halving_mode=1) -> float:
    return float(_load().orc_block_update(h, dt_req, t_new, dt_min, dt_max, halving_mode))


def initial_dt(a, j, eta, dt_min=DT_MIN, dt_max=DT_MAX):
    a, j = _f64(a), _f64(j)
    out = np.zeros(a.shape[0])
    _load().orc_initial_dt(a.shape[0], _p(a), _p(j), eta, dt_min, dt_max, _p(out))
    return out


def next_block(t_i, dt):
    t_i, dt = _f64(t_i), _f64(dt)
    n = t_i.shape[0]
    act = np.zeros(n, dtype=np.int32)
    cnt = C.c_int64(0)
    tn = _load().orc_next_block(n, _p(t_i), _p(dt), act.ctypes.data_as(_ip), C.byref(cnt))
    return float(tn), act[:cnt.value].copy()


def predict(t, x, v, a, j, t_i):
    x, v, a, j, t_i = map(_f64, (x, v, a, j, t_i))
    xp, vp = np.zeros_like(x), np.zeros_like(v)
    _load().orc_predict(x.shape[0], float(t), _p(x), _p(v), _p(a), _p(j), _p(t_i), _p(xp), _p(vp))
    return xp, vp


def correct(active, t_new, eta, x, v, a, j, t_i, dt, xp, vp, a1, j1, dt_min=DT_MIN, dt_max=DT_MAX,
            halving_mode=1):
    """Corrector + time-step update for the active list; returns new copies (x, v, a, j, t_i, dt, dt_req)."""
    active = np.ascontiguousarray(active, dtype=np.int32)
    x, v, a, j, t_i, dt = (_f64(u).copy() for u in (x, v, a, j, t_i, dt))
    xp, vp, a1, j1 = map(_f64, (xp, vp, a1, j1))
    dt_req = np.zeros(active.shape[0])
    diag = np.zeros(2, dtype=np.int64)
    margin = C.c_double(np.inf)
    _load().orc_correct(active.shape[0], active.ctypes.data_as(_ip), float(t_new), float(eta), dt_min, dt_max,
                        int(halving_mode), _p(x), _p(v), _p(a), _p(j), _p(t_i), _p(dt), _p(xp), _p(vp),
                        _p(a1), _p(j1), diag.ctypes.data_as(_lp), C.byref(margin), _p(dt_req))
    return x, v, a, j, t_i, dt, dt_req


def energy(m, x, v, eps):
    """(K, U) with the softened potential."""
    m, x, v = _f64(m), _f64(x), _f64(v)
    k, u = C.c_double(0), C.c_double(0)
    _load().orc_energy(m.shape[0], _p(m), _p(x), _p(v), float(eps) ** 2, C.byref(k), C.byref(u))
    return k.value, u.value


class HermiteOracle:
    """The whole integrator: INIT then block steps, state in numpy arrays owned here."""

    def __init__(self, m, x, v, eps, eta, dt_min=DT_MIN, dt_max=DT_MAX, halving_mode=1,
                 acc_mode: str = "compensated"):
        self._lib = _load()
        self.m, self.x, self.v = _f64(m).copy(), _f64(x).copy(), _f64(v).copy()
        n = self.m.shape[0]
        self.n = n
        self.eps = float(eps)
        self.a, self.j = np.zeros((n, 3)), np.zeros((n, 3))
        self.t_i, self.dt = np.zeros(n), np.zeros(n)
        self.xp, self.vp = np.zeros((n, 3)), np.zeros((n, 3))
        self.a1, self.j1 = np.zeros((n, 3)), np.zeros((n, 3))
        self._active = np.zeros(n, dtype=np.int32)
        s = _State()
        s.n = n
        s.eps2, s.eta, s.dt_min, s.dt_max = self.eps ** 2, float(eta), float(dt_min), float(dt_max)
        s.halving_mode = int(halving_mode)
        s.acc_mode = {"plain": 0, "compensated": 1}[acc_mode]
        for name in ("m", "x", "v", "a", "j", "t_i", "dt", "xp", "vp", "a1", "j1"):
            setattr(s, name, _p(getattr(self, name)))
        s.active = self._active.ctypes.data_as(_ip)
        self._s = s
        self._lib.orc_init(C.byref(s))

    # --- stepping -------------------------------------------------------------------------------
    def step(self) -> float:
        return float(self._lib.orc_step(C.byref(self._s)))

    def run(self, t_end: float = np.inf, max_steps: int = -1, record: bool = False):
        """Advance; with record=True returns (t[], n_act[], hash[]) for the steps taken."""
        cap = 0
        rt = rn = rh = None
        if record:
            cap = max_steps if max_steps >= 0 else 1 << 22
            rt, rn, rh = np.zeros(cap), np.zeros(cap, dtype=np.int64), np.zeros(cap, dtype=np.uint64)
        k = self._lib.orc_run(C.byref(self._s), float(t_end), int(max_steps),
                              _p(rt) if record else None,
                              rn.ctypes.data_as(_lp) if record else None,
                              rh.ctypes.data_as(C.POINTER(C.c_uint64)) if record else None, cap)
        if record:
            k = min(k, cap)
            return rt[:k], rn[:k], rh[:k]
        return int(k)

    # --- views ----------------------------------------------------------------------------------
    @property
    def t(self) -> float:
        return float(self._s.t)

    @property
    def active(self) -> np.ndarray:
        return self._active[: self._s.n_act].copy()

    @property
    def block_steps(self) -> int:
        return int(self._s.block_steps)

    @property
    def particle_steps(self) -> int:
        return int(self._s.particle_steps)

    @property
    def nan_count(self) -> int:
        return int(self._s.diag[0])

    @property
    def dtmin_clamps(self) -> int:
        return int(self._s.diag[1])

    @property
    def min_margin(self) -> float:
        return float(self._s.min_margin)

    @property
    def seconds(self) -> tuple[float, float]:
        """(wall seconds inside PAIRSUM, wall seconds inside INIT + the block steps) so far (force ~ 95 %)."""
        return float(self._s.sec_force), float(self._s.sec_total)

    @property
    def level_hist(self) -> np.ndarray:
        return np.array(list(self._s.level_hist), dtype=np.int64)

    def energy(self):
        """(K, U) at the current time: every particle predicted to t (reading R9), softened U (R8)."""
        xp, vp = predict(self.t, self.x, self.v, self.a, self.j, self.t_i)
        return energy(self.m, xp, vp, self.eps)
