"""ctypes binding of include/gravidy_b200.h -- argument marshalling only.

Every step of the path runs in the CUDA kernels of libgravidy_b200.so; this module only turns torch CUDA
tensors into device pointers (torch is used for device memory and streams, nothing else) and numpy arrays
into host pointers.  There is no CPU fallback: if the library is missing or no CUDA device is present the
calls raise.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np

_PKG = Path(__file__).resolve().parent
LIB_PATH = _PKG / "libgravidy_b200.so"

GD_OK, GD_EINVAL, GD_ESTATE, GD_ECUDA = 0, -1, -2, -3

#: every symbol include/gravidy_b200.h declares: name -> (restype, argtypes)
_vp, _i64, _dbl, _int, _sz = C.c_void_p, C.c_int64, C.c_double, C.c_int, C.c_size_t
_pi64, _pdbl = C.POINTER(C.c_int64), C.POINTER(C.c_double)
SYMBOLS = {
    "gd_version": (C.c_char_p, []),
    "gd_workspace_bytes": (_sz, [_i64]),
    "gd_init": (_int, [C.POINTER(_vp), _i64, _vp, _vp, _vp, _dbl, _dbl, _vp, _sz, _vp]),
    "gd_init_host": (_int, [C.POINTER(_vp), _i64, _vp, _vp, _vp, _dbl, _dbl, _vp, _sz, _vp]),
    "gd_destroy": (None, [_vp]),
    "gd_last_error": (C.c_char_p, [_vp]),
    "gd_set_option": (_int, [_vp, C.c_char_p, _dbl]),
    "gd_next_block": (_int, [_vp, _pdbl, _pi64]),
    "gd_predict": (_int, [_vp, _dbl]),
    "gd_force_jerk": (_int, [_vp, _vp, _i64, _vp, _vp]),
    "gd_force_jerk_host": (_int, [_i64, _vp, _vp, _vp, _dbl, _vp, _i64, _vp, _vp, _vp, _sz, _vp]),
    "gd_correct_and_timestep": (_int, [_vp]),
    "gd_energy": (_int, [_vp, _pdbl, _pdbl]),
    "gd_energy_static": (_int, [_i64, _vp, _vp, _vp, _dbl, _vp, _vp]),
    "gd_energy_static_last_error": (C.c_char_p, []),
    "gd_step": (_int, [_vp, _i64, _pi64]),
    "gd_run_until": (_int, [_vp, _dbl, _i64, _pi64, _pi64]),
    "gd_time": (_dbl, [_vp]),
    "gd_n": (_i64, [_vp]),
    "gd_n_active": (_i64, [_vp]),
    "gd_block_steps": (_i64, [_vp]),
    "gd_particle_steps": (_i64, [_vp]),
    "gd_last_force_kernel": (_int, [_vp]),
    "gd_kernel_launches": (_i64, [_vp]),
    "gd_last_force_geometry": (_int, [_vp, _vp]),
    "gd_get_state": (_int, [_vp] * 7),
    "gd_get_state_host": (_int, [_vp] * 7),
    "gd_get_predicted": (_int, [_vp, _vp, _vp]),
    "gd_get_active": (_int, [_vp, _vp, _i64]),
    "gd_get_level_histogram": (_int, [_vp, _vp, _vp]),
    "gd_get_profile": (_int, [_vp, _vp]),
    "gd_get_loop_profile": (_int, [_vp, _vp]),
    "gd_get_loop_histogram": (_int, [_vp, _vp]),
    "gd_get_level_census": (_int, [_vp, _vp]),
    "gd_core_radius": (_int, [_vp, _int, _pdbl, _vp, _vp]),
    "gd_lagrange_radii": (_int, [_vp, _vp, _vp, _int, _vp, _vp]),
    "gd_fp64_peak_probe": (_int, [_int, _pdbl, _pdbl]),
    "gd_selftest_div_const": (_int, [C.c_int64, C.c_uint64, _vp]),
}

_lib = None


class GravidyError(RuntimeError):
    def __init__(self, code: int, text: str):
        super().__init__(f"gravidy_b200 error {code}: {text}")
        self.code = code


def load() -> C.CDLL:
    """dlopen the in-tree library and declare the prototypes; raises if it has not been built."""
    global _lib
    if _lib is None:
        if not LIB_PATH.exists():
            raise FileNotFoundError(f"{LIB_PATH} is missing: run `python -m paper_1702_00440_b200.build` "
                                    "(there is no fallback path)")
        lib = C.CDLL(str(LIB_PATH))
        for name, (res, args) in SYMBOLS.items():
            fn = getattr(lib, name)
            fn.restype, fn.argtypes = res, args
        _lib = lib
    return _lib


def version() -> str:
    return load().gd_version().decode()


def workspace_bytes(n: int) -> int:
    return int(load().gd_workspace_bytes(int(n)))


def fp64_peak_probe(iters: int = 1 << 15) -> tuple[float, float]:
    """(flop/s, ms) of the register-only DFMA loop on the current device."""
    f, ms = C.c_double(0), C.c_double(0)
    rc = load().gd_fp64_peak_probe(int(iters), C.byref(f), C.byref(ms))
    if rc:
        raise GravidyError(rc, "gd_fp64_peak_probe failed (no CUDA device?)")
    return f.value, ms.value


def selftest_div_const(n: int = 1 << 24, seed: int = 1) -> int:
    """Mismatches between the corrector's division by 6, 24, 120 (multiply + two FMAs) and x / c on n random operands."""
    bad = C.c_int64(-1)
    rc = load().gd_selftest_div_const(int(n), int(seed), C.byref(bad))
    if rc:
        raise GravidyError(rc, "gd_selftest_div_const failed (no CUDA device?)")
    return int(bad.value)


#: largest n gd_energy_static accepts (GD_ENERGY_STATIC_MAX_N of the header)
ENERGY_STATIC_MAX_N = 1 << 21


def energy_static(m, x, v, eps: float, out, stream=None):
    """gd_energy_static: K and U (Eq. 2) of the particles m [n], x [n,3], v [n,3] into out[0], out[1].

    This is the call for code that may not allocate on the GPU -- a driver whose pool already owns all of HBM, a loop
    that cannot afford the device-wide wait of cudaMalloc, a plug-in whose host forbids allocations -- so the wrapper
    allocates nothing either: m, x, v and out (two doubles) must already be contiguous float64 CUDA tensors.  The
    reduction's scratch lives in a fixed array inside the library, hence n <= ENERGY_STATIC_MAX_N and the rule that
    two calls must not run concurrently on one GPU (calls on one stream are fine).  Asynchronous on `stream` (default:
    torch's current stream); returns `out`.  The first call per GPU should happen outside stream capture."""
    torch = _torch()
    n = int(m.shape[0])
    for t, shape in ((m, (n,)), (x, (n, 3)), (v, (n, 3)), (out, (2,))):
        assert t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and tuple(t.shape) == shape, \
            "energy_static takes contiguous float64 CUDA tensors m [n], x [n,3], v [n,3], out [2] and converts nothing"
    sp = (torch.cuda.current_stream() if stream is None else stream).cuda_stream
    rc = load().gd_energy_static(n, m.data_ptr(), x.data_ptr(), v.data_ptr(), float(eps), out.data_ptr(), sp)
    if rc:
        raise GravidyError(rc, load().gd_energy_static_last_error().decode())
    return out


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("gravidy_b200 needs a CUDA device; there is no CPU fallback")
    return torch


def _dev_f64(t, shape=None):
    torch = _torch()
    if isinstance(t, np.ndarray):
        t = torch.from_numpy(np.ascontiguousarray(t, dtype=np.float64)).cuda()
    assert t.is_cuda and t.dtype == torch.float64 and t.is_contiguous(), "need a contiguous float64 CUDA tensor"
    if shape is not None:
        assert tuple(t.shape) == tuple(shape), f"shape {tuple(t.shape)} != {tuple(shape)}"
    return t


def _host_f64(a, shape=None):
    a = np.ascontiguousarray(a, dtype=np.float64)
    if shape is not None:
        assert a.shape == tuple(shape)
    return a


def _alloc_workspace(n: int):
    torch = _torch()
    nbytes = workspace_bytes(n)
    ws = torch.empty(nbytes + 256, dtype=torch.uint8, device="cuda")
    off = (-ws.data_ptr()) % 256
    return ws, ws.data_ptr() + off, nbytes


def force_jerk_host(m, x, v, eps: float, idx=None):
    """One-shot a, jerk on HOST numpy arrays through gd_force_jerk_host (copies inside the call)."""
    torch = _torch()
    m, x, v = _host_f64(m), _host_f64(x), _host_f64(v)
    n = m.shape[0]
    if idx is not None:
        idx = np.ascontiguousarray(idx, dtype=np.int32)
    n_act = n if idx is None else idx.shape[0]
    a, j = np.empty((n_act, 3)), np.empty((n_act, 3))
    ws, ptr, nbytes = _alloc_workspace(n)
    rc = load().gd_force_jerk_host(n, m.ctypes.data, x.ctypes.data, v.ctypes.data, float(eps),
                                   idx.ctypes.data if idx is not None else None, n_act, a.ctypes.data, j.ctypes.data,
                                   ptr, nbytes, torch.cuda.current_stream().cuda_stream)
    if rc:
        raise GravidyError(rc, load().gd_last_error(None).decode())
    return a, j


class Hermite:
    """One integration context: the calls of the C-ABI with the same names (init, next_block, predict,
    force_jerk, correct_and_timestep, energy, ...)."""

    def __init__(self, m, x, v, eps: float, eta: float, host: bool = False, stream=None):
        torch = _torch()
        self._lib = load()
        self._h = _vp(None)
        n = int(m.shape[0])
        self.n = n
        self._ws, ptr, nbytes = _alloc_workspace(n)
        self._stream = torch.cuda.current_stream() if stream is None else stream
        sp = self._stream.cuda_stream
        if host:
            m, x, v = _host_f64(m, (n,)), _host_f64(x, (n, 3)), _host_f64(v, (n, 3))
            rc = self._lib.gd_init_host(C.byref(self._h), n, m.ctypes.data, x.ctypes.data, v.ctypes.data,
                                        float(eps), float(eta), ptr, nbytes, sp)
        else:
            m, x, v = _dev_f64(m, (n,)), _dev_f64(x, (n, 3)), _dev_f64(v, (n, 3))
            rc = self._lib.gd_init(C.byref(self._h), n, m.data_ptr(), x.data_ptr(), v.data_ptr(),
                                   float(eps), float(eta), ptr, nbytes, sp)
        if rc:
            raise GravidyError(rc, self._lib.gd_last_error(None).decode())

    # -- plumbing ---------------------------------------------------------------------------------
    def _check(self, rc: int):
        if rc:
            raise GravidyError(rc, self._lib.gd_last_error(self._h).decode())

    def close(self):
        h, lib = getattr(self, "_h", None), getattr(self, "_lib", None)
        if h is not None and h.value and lib is not None:
            lib.gd_destroy(h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:        # interpreter shutdown: ctypes may already be torn down
            pass

    def set_option(self, key: str, value: float):
        self._check(self._lib.gd_set_option(self._h, key.encode(), float(value)))

    # -- the stages -------------------------------------------------------------------------------
    def next_block(self) -> tuple[float, int]:
        t, k = C.c_double(0), C.c_int64(0)
        self._check(self._lib.gd_next_block(self._h, C.byref(t), C.byref(k)))
        return t.value, k.value

    def predict(self, t: float):
        self._check(self._lib.gd_predict(self._h, float(t)))

    def force_jerk(self, idx=None, a_out=None, j_out=None):
        """idx: int32 CUDA tensor (or None = internal active list).  With idx given, returns (a, j) tensors."""
        torch = _torch()
        if idx is None:
            self._check(self._lib.gd_force_jerk(self._h, None, 0,
                                                a_out.data_ptr() if a_out is not None else None,
                                                j_out.data_ptr() if j_out is not None else None))
            return a_out, j_out
        if isinstance(idx, np.ndarray):
            idx = torch.from_numpy(np.ascontiguousarray(idx, dtype=np.int32)).cuda()
        assert idx.is_cuda and idx.dtype == torch.int32 and idx.is_contiguous()
        k = idx.shape[0]
        if a_out is None:
            a_out = torch.empty((k, 3), dtype=torch.float64, device="cuda")
            j_out = torch.empty((k, 3), dtype=torch.float64, device="cuda")
        self._check(self._lib.gd_force_jerk(self._h, idx.data_ptr(), k, a_out.data_ptr(), j_out.data_ptr()))
        return a_out, j_out

    def correct_and_timestep(self):
        self._check(self._lib.gd_correct_and_timestep(self._h))

    def energy(self) -> tuple[float, float]:
        k, u = C.c_double(0), C.c_double(0)
        self._check(self._lib.gd_energy(self._h, C.byref(k), C.byref(u)))
        return k.value, u.value

    def step(self, n_steps: int = 1) -> int:
        ps = C.c_int64(0)
        self._check(self._lib.gd_step(self._h, int(n_steps), C.byref(ps)))
        return ps.value

    def run_until(self, t_end: float, max_steps: int = -1) -> tuple[int, int]:
        s, ps = C.c_int64(0), C.c_int64(0)
        self._check(self._lib.gd_run_until(self._h, float(t_end), int(max_steps), C.byref(s), C.byref(ps)))
        return s.value, ps.value

    # -- views ------------------------------------------------------------------------------------
    @property
    def t(self) -> float:
        return float(self._lib.gd_time(self._h))

    @property
    def n_active(self) -> int:
        return int(self._lib.gd_n_active(self._h))

    @property
    def block_steps(self) -> int:
        return int(self._lib.gd_block_steps(self._h))

    @property
    def particle_steps(self) -> int:
        return int(self._lib.gd_particle_steps(self._h))

    @property
    def last_force_kernel(self) -> str:
        return {0: "none", 1: "ipar", 2: "jsplit", 3: "ipar_small", 4: "slice"}[int(self._lib.gd_last_force_kernel(self._h))]

    @property
    def kernel_launches(self) -> int:
        return int(self._lib.gd_kernel_launches(self._h))

    @property
    def last_force_geometry(self) -> tuple:
        g = (C.c_int * 4)()
        self._check(self._lib.gd_last_force_geometry(self._h, g))
        return tuple(g)

    def state(self, names=("x", "v", "a", "j", "t", "dt")) -> dict:
        """Copies of the state as CUDA tensors."""
        torch = _torch()
        out = {}
        for k in names:
            out[k] = torch.empty((self.n, 3) if k in "xvaj" else (self.n,), dtype=torch.float64, device="cuda")
        p = [out[k].data_ptr() if k in out else None for k in ("x", "v", "a", "j", "t", "dt")]
        self._check(self._lib.gd_get_state(self._h, *p))
        return out

    def state_host(self, names=("x", "v", "a", "j", "t", "dt")) -> dict:
        """Copies of the state as numpy arrays through gd_get_state_host (D2H inside the call)."""
        out = {k: np.empty((self.n, 3) if k in "xvaj" else (self.n,)) for k in names}
        p = [out[k].ctypes.data if k in out else None for k in ("x", "v", "a", "j", "t", "dt")]
        self._check(self._lib.gd_get_state_host(self._h, *p))
        return out

    def predicted(self):
        torch = _torch()
        xp = torch.empty((self.n, 3), dtype=torch.float64, device="cuda")
        vp = torch.empty((self.n, 3), dtype=torch.float64, device="cuda")
        self._check(self._lib.gd_get_predicted(self._h, xp.data_ptr(), vp.data_ptr()))
        return xp, vp

    def active(self):
        torch = _torch()
        k = self.n_active
        idx = torch.empty((max(k, 1),), dtype=torch.int32, device="cuda")
        self._check(self._lib.gd_get_active(self._h, idx.data_ptr(), idx.shape[0]))
        return idx[:k]

    def profile(self) -> dict:
        """Event-timed force launches since the "profile" option was set: per kernel launches, ms, pairs."""
        p = np.zeros(20)
        self._check(self._lib.gd_get_profile(self._h, p.ctypes.data))
        return {k: {"launches": int(p[4 * i]), "ms": float(p[4 * i + 1]), "pairs": float(p[4 * i + 2]),
                    "ms2": float(p[4 * i + 3])} for i, k in enumerate(("ipar", "jsplit", "ipar_small", "loop", "slice"))}

    def lagrange_radii(self, fractions, center=None):
        """Radii about `center` (None: the centre of mass) holding the given mass fractions -> (radii, centre[3], M)."""
        f = np.ascontiguousarray(fractions, dtype=np.float64)
        r, co = np.zeros(f.shape[0]), np.zeros(4)
        c = None if center is None else np.ascontiguousarray(center, dtype=np.float64)
        self._check(self._lib.gd_lagrange_radii(self._h, c.ctypes.data if c is not None else None, f.ctypes.data,
                                                int(f.shape[0]), r.ctypes.data, co.ctypes.data))
        return r, co[:3].copy(), float(co[3])

    def level_census(self) -> np.ndarray:
        """Number of particles per CURRENT block step 2^-k (Fig. 13)."""
        h = np.zeros(64, dtype=np.int64)
        self._check(self._lib.gd_get_level_census(self._h, h.ctypes.data))
        return h

    def core_radius(self, k: int = 6, want_rho: bool = False):
        """(r_c, density centre[3]) or (r_c, centre, rho CUDA tensor [n]) -- Casertano & Hut (1985), R25."""
        torch = _torch()
        rc, xd = C.c_double(0), np.zeros(3)
        rho = torch.empty((self.n,), dtype=torch.float64, device="cuda") if want_rho else None
        self._check(self._lib.gd_core_radius(self._h, int(k), C.byref(rc), xd.ctypes.data, rho.data_ptr() if want_rho else None))
        return (rc.value, xd, rho) if want_rho else (rc.value, xd)

    def loop_profile(self) -> dict:
        o = np.zeros(11, dtype=np.int64)
        self._check(self._lib.gd_get_loop_profile(self._h, o.ctypes.data))
        keys = ("particle_steps", "block_steps", "ns", "ns_force", "ns_barrier1", "ns_correct", "ns_barrier2", "launches",
                "owner_steps", "ns_owner_correct", "ns_owner_publish")
        return {k: int(v) for k, v in zip(keys, o)}

    def loop_histogram(self) -> list[dict]:
        """Block steps of the persistent loop binned by active-set size: one row per non-empty bucket."""
        o = np.zeros((32, 6), dtype=np.int64)
        self._check(self._lib.gd_get_loop_histogram(self._h, o.ctypes.data))
        keys = ("block_steps", "particle_steps", "ns_force", "ns_barrier1", "ns_correct", "ns_barrier2")
        return [dict({"n_act_below": 1 << b}, **{k: int(v) for k, v in zip(keys, o[b])}) for b in range(32) if o[b, 0]]

    def level_histogram(self) -> tuple[np.ndarray, np.ndarray]:
        h, d = np.zeros(64, dtype=np.int64), np.zeros(2, dtype=np.int64)
        self._check(self._lib.gd_get_level_histogram(self._h, h.ctypes.data, d.ctypes.data))
        return h, d
