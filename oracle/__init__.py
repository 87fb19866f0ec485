"""ctypes binding of the CPU oracle (oracle/smaug_oracle.cpp) -- TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / ``--impl reference`` legs may import
this package; the product (paper_1710_06423_b200/) never does.  ``build()`` compiles the C++ source with
g++ (``-O2 -ffp-contract=off``, no fast-math; OpenMP is compiled in but every context starts with one
thread, and the row-parallel loops are result-neutral: no sum reductions, only max).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "smaug_oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle_smaug.so")
_SRC3 = os.path.join(_HERE, "smaug3d_oracle.cpp")       # the 3-D form: a separate library (no shared code)
_LIB3 = os.path.join(_HERE, "liboracle_smaug3d.so")

BC_PERIODIC, BC_OPEN, BC_FIXED = 0, 1, 2
(P_LX, P_LY, P_HD_ON, P_C_RHO, P_C_MOM, P_C_E, P_C_B, P_RK_ORDER, P_FIXED_DT) = range(9)
P_GX, P_GY = 10, 11
P_LZ, P_GZ = 13, 14
ENONFINITE = -4

_lib = None
_lib3 = None


def _cpu_has_fma() -> bool:
    try:
        with open("/proc/cpuinfo") as f:
            return " fma " in f.read().replace("\n", " ")
    except OSError:
        return False


def _compile(src: str, out: str, force: bool) -> str:
    if force or not os.path.exists(out) or os.path.getmtime(out) < os.path.getmtime(src):
        cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared"]
        if _cpu_has_fma():
            cmd.append("-mfma")      # std::fma -> one hardware instruction (same bits as the libm fallback)
        cmd += ["-o", out, src]
        subprocess.run(cmd, check=True)
    return out


def build(force: bool = False) -> str:
    """Compile liboracle_smaug.so (and the 3-D oracle's library) next to the sources if missing or stale."""
    _compile(_SRC3, _LIB3, force)
    return _compile(_SRC, _LIB, force)


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        dp, ip, vp = C.POINTER(C.c_double), C.POINTER(C.c_int), C.c_void_p
        L.oracle_last_error.restype = C.c_char_p
        L.oracle_create.argtypes = [C.c_int, C.c_int, C.c_double, ip, dp, C.POINTER(vp)]
        L.oracle_destroy.argtypes = [vp]
        L.oracle_destroy.restype = None
        L.oracle_set_param.argtypes = [vp, C.c_int, C.c_double]
        L.oracle_set_threads.argtypes = [vp, C.c_int]
        L.oracle_set_state.argtypes = [vp, dp]
        L.oracle_get_state.argtypes = [vp, dp]
        L.oracle_get_time.argtypes = [vp, dp, dp]
        L.oracle_step.argtypes = [vp, C.c_int, C.c_double]
        L.oracle_rhs.argtypes = [vp, dp]
        L.oracle_wavespeeds.argtypes = [vp, dp]
        L.oracle_get_padded.argtypes = [vp, C.c_int, dp]
        L.oracle_hyper_nu_1d.argtypes = [dp, C.c_int, C.c_double, C.c_double, C.c_double, dp]
        L.oracle_central_diff_1d.argtypes = [dp, C.c_int, C.c_double, dp]
        _lib = L
    return _lib


def _dp(a: np.ndarray):
    return a.ctypes.data_as(C.POINTER(C.c_double))


class OracleError(RuntimeError):
    def __init__(self, code: int):
        self.code = code
        super().__init__(f"oracle error {code}: {lib().oracle_last_error().decode()}")


def _check(rc: int) -> None:
    if rc != 0:
        raise OracleError(rc)


class Oracle:
    """One oracle context.  Arrays are numpy float64, state [6, ny, nx], background [4, ny, nx]."""

    def __init__(self, nx, ny, gamma, bc, bg=None, threads=1, **params):
        L = lib()
        self.nx, self.ny = int(nx), int(ny)
        bc_arr = (C.c_int * 4)(*[int(b) for b in bc])
        bgp = None
        if bg is not None:
            bg = np.ascontiguousarray(bg, dtype=np.float64)
            assert bg.shape == (4, ny, nx)
            bgp = _dp(bg)
        h = C.c_void_p()
        _check(L.oracle_create(nx, ny, float(gamma), bc_arr, bgp, C.byref(h)))
        self._h = h
        if threads != 1:
            _check(L.oracle_set_threads(self._h, int(threads)))
        for k, v in params.items():
            self.set_param(k, v)

    _KEYS = dict(lx=P_LX, ly=P_LY, hd_on=P_HD_ON, c_rho=P_C_RHO, c_mom=P_C_MOM, c_e=P_C_E, c_b=P_C_B,
                 rk_order=P_RK_ORDER, fixed_dt=P_FIXED_DT, gx=P_GX, gy=P_GY)

    def set_param(self, key, value):
        k = self._KEYS[key] if isinstance(key, str) else int(key)
        _check(lib().oracle_set_param(self._h, k, float(value)))

    def set_state(self, w):
        w = np.ascontiguousarray(w, dtype=np.float64)
        assert w.shape == (6, self.ny, self.nx)
        _check(lib().oracle_set_state(self._h, _dp(w)))

    def get_state(self):
        w = np.empty((6, self.ny, self.nx))
        _check(lib().oracle_get_state(self._h, _dp(w)))
        return w

    def step(self, n_steps, cfl=0.3):
        _check(lib().oracle_step(self._h, int(n_steps), float(cfl)))

    def time(self):
        t, dt = C.c_double(), C.c_double()
        _check(lib().oracle_get_time(self._h, C.byref(t), C.byref(dt)))
        return t.value, dt.value

    def rhs(self):
        r = np.empty((6, self.ny, self.nx))
        _check(lib().oracle_rhs(self._h, _dp(r)))
        return r

    def wavespeeds(self):
        o = np.empty(4)
        _check(lib().oracle_wavespeeds(self._h, _dp(o)))
        return o

    def padded(self, f):
        o = np.empty((self.ny + 6, self.nx + 6))
        _check(lib().oracle_get_padded(self._h, int(f), _dp(o)))
        return o

    def close(self):
        if getattr(self, "_h", None):
            lib().oracle_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def hyper_nu_1d(u_padded, coef, delta, vt):
    """c-5 coefficient along a 1-D line; u_padded has n+6 entries, returns the n+1 interfaces -1/2..n-1/2."""
    u = np.ascontiguousarray(u_padded, dtype=np.float64)
    n = u.size - 6
    out = np.empty(n + 1)
    _check(lib().oracle_hyper_nu_1d(_dp(u), n, float(coef), float(delta), float(vt), _dp(out)))
    return out


def central_diff_1d(f_padded, h):
    """c-3 along a 1-D line; f_padded has n+4 entries, returns n derivatives."""
    f = np.ascontiguousarray(f_padded, dtype=np.float64)
    n = f.size - 4
    out = np.empty(n)
    _check(lib().oracle_central_diff_1d(_dp(f), n, float(h), _dp(out)))
    return out


# ------------------------------------------------------------------------------------------------ three dimensions
def lib3() -> C.CDLL:
    global _lib3
    if _lib3 is None:
        L = C.CDLL(_compile(_SRC3, _LIB3, False))
        dp, ip, vp = C.POINTER(C.c_double), C.POINTER(C.c_int), C.c_void_p
        L.oracle3_last_error.restype = C.c_char_p
        L.oracle3_create.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, ip, C.POINTER(vp)]
        L.oracle3_destroy.argtypes = [vp]
        L.oracle3_destroy.restype = None
        L.oracle3_set_param.argtypes = [vp, C.c_int, C.c_double]
        L.oracle3_set_threads.argtypes = [vp, C.c_int]
        L.oracle3_set_state.argtypes = [vp, dp]
        L.oracle3_get_state.argtypes = [vp, dp]
        L.oracle3_get_time.argtypes = [vp, dp, dp]
        L.oracle3_step.argtypes = [vp, C.c_int, C.c_double]
        L.oracle3_rhs.argtypes = [vp, dp]
        L.oracle3_wavespeeds.argtypes = [vp, dp]
        L.oracle3_get_padded.argtypes = [vp, C.c_int, dp]
        _lib3 = L
    return _lib3


class Oracle3D:
    """One context of the 3-D oracle (smaug3d_oracle.cpp).  State: numpy float64 [8, nz, ny, nx] =
    (rho, mx, my, mz, e, bx, by, bz); bc = (x_lo, x_hi, y_lo, y_hi, z_lo, z_hi); zero background."""

    _KEYS = dict(lx=P_LX, ly=P_LY, lz=P_LZ, hd_on=P_HD_ON, c_rho=P_C_RHO, c_mom=P_C_MOM, c_e=P_C_E, c_b=P_C_B,
                 rk_order=P_RK_ORDER, fixed_dt=P_FIXED_DT, gx=P_GX, gy=P_GY, gz=P_GZ)

    def __init__(self, nx, ny, nz, gamma, bc, threads=1, **params):
        L = lib3()
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        h = C.c_void_p()
        self._chk(L.oracle3_create(self.nx, self.ny, self.nz, float(gamma), (C.c_int * 6)(*[int(b) for b in bc]), C.byref(h)))
        self._h = h
        if threads != 1:
            self._chk(L.oracle3_set_threads(self._h, int(threads)))
        for k, v in params.items():
            self.set_param(k, v)

    @staticmethod
    def _chk(rc):
        if rc != 0:
            raise RuntimeError(f"oracle3 error {rc}: {lib3().oracle3_last_error().decode()}")

    @property
    def shape(self):
        return (8, self.nz, self.ny, self.nx)

    def set_param(self, key, value):
        k = self._KEYS[key] if isinstance(key, str) else int(key)
        self._chk(lib3().oracle3_set_param(self._h, k, float(value)))

    def set_state(self, w):
        w = np.ascontiguousarray(w, dtype=np.float64)
        assert w.shape == self.shape
        self._chk(lib3().oracle3_set_state(self._h, _dp(w)))

    def get_state(self):
        w = np.empty(self.shape)
        self._chk(lib3().oracle3_get_state(self._h, _dp(w)))
        return w

    def step(self, n_steps, cfl=0.3):
        self._chk(lib3().oracle3_step(self._h, int(n_steps), float(cfl)))

    def time(self):
        t, dt = C.c_double(), C.c_double()
        self._chk(lib3().oracle3_get_time(self._h, C.byref(t), C.byref(dt)))
        return t.value, dt.value

    def rhs(self):
        r = np.empty(self.shape)
        self._chk(lib3().oracle3_rhs(self._h, _dp(r)))
        return r

    def wavespeeds(self):
        o = np.empty(5)
        self._chk(lib3().oracle3_wavespeeds(self._h, _dp(o)))
        return o

    def padded(self, f):
        o = np.empty((self.nz + 6, self.ny + 6, self.nx + 6))
        self._chk(lib3().oracle3_get_padded(self._h, int(f), _dp(o)))
        return o

    def close(self):
        if getattr(self, "_h", None):
            lib3().oracle3_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
