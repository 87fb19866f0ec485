"""paper_1710_06423_b200 -- B200-native SMAUG+ hot path (one full 2-D MHD time step), Python binding.

Thin ctypes layer over ``libsmaug.so`` (C ABI in include/smaug.h, CUDA sources in csrc/).  Argument
marshalling only: every step of the path runs in the library's kernels.  PyTorch supplies device memory
(the workspace tensor, state tensors) and the stream; nothing here computes.  There is no CPU fallback:
``lib()`` raises if the extension is missing, and every call fails loudly without a CUDA device.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
_CSRC = os.path.join(_HERE, "csrc")
LIB_PATH = os.path.join(_HERE, "libsmaug.so")
INCLUDE = os.path.join(os.path.dirname(_HERE), "include")

BC_PERIODIC, BC_OPEN, BC_FIXED = 0, 1, 2
OK, EINVAL, ENOMEM, ECUDA, ENONFINITE = 0, -1, -2, -3, -4
PARAMS = dict(lx=0, ly=1, hd_on=2, c_rho=3, c_mom=4, c_e=5, c_b=6, rk_order=7, fixed_dt=8, kernel=9, gx=10, gy=11, graph=12)

NVCC_FLAGS = ["-O3", "-std=c++17", "-fmad=false", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-shared"]

_lib = None


def _sources():
    return sorted(os.path.join(_CSRC, f) for f in os.listdir(_CSRC))


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile csrc/smaug.cu, csrc/smaug3d.cu and csrc/smaug_static.cu for sm_100a into libsmaug.so (in-tree) if missing or stale."""
    newest = max(os.path.getmtime(p) for p in _sources() + [os.path.join(INCLUDE, "smaug.h"), os.path.join(INCLUDE, "smaug3d.h")])
    if force or not os.path.exists(LIB_PATH) or os.path.getmtime(LIB_PATH) < newest:
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + \
              ["-o", LIB_PATH, os.path.join(_CSRC, "smaug.cu"), os.path.join(_CSRC, "smaug3d.cu"),
               os.path.join(_CSRC, "smaug_static.cu")]
        subprocess.run(cmd, check=True)
    return LIB_PATH


def lib() -> C.CDLL:
    """Load libsmaug.so (never builds implicitly on a box without nvcc: fails loudly instead)."""
    global _lib
    if _lib is None:
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        if os.path.exists(nvcc):
            try:
                build()                     # no-op unless the library is missing or older than csrc/ or smaug.h
            except Exception as e:  # noqa: BLE001
                raise RuntimeError(f"libsmaug.so is missing or stale and could not be built ({e}); "
                                   "there is no CPU fallback") from e
        elif not os.path.exists(LIB_PATH):
            raise RuntimeError("libsmaug.so is missing and there is no nvcc to build it; there is no CPU fallback")
        L = C.CDLL(LIB_PATH)
        dp, vp = C.POINTER(C.c_double), C.c_void_p
        L.smaug_last_error.restype = C.c_char_p
        L.smaug_workspace_bytes.restype = C.c_size_t
        L.smaug_workspace_bytes.argtypes = [C.c_int, C.c_int, C.c_int]
        L.smaug_create.argtypes = [C.c_int, C.c_int, C.c_double, C.POINTER(C.c_int), vp, C.POINTER(vp)]
        L.smaug_create_in_workspace.argtypes = [C.c_int, C.c_int, C.c_double, C.POINTER(C.c_int), vp, vp,
                                                C.c_size_t, vp, C.POINTER(vp)]
        L.smaug_set_stream.argtypes = [vp, vp]
        L.smaug_set_param.argtypes = [vp, C.c_int, C.c_double]
        L.smaug_set_state.argtypes = [vp, vp]
        L.smaug_step.argtypes = [vp, C.c_int, C.c_double]
        L.smaug_step_async.argtypes = [vp, C.c_int, C.c_double]
        L.smaug_get_state.argtypes = [vp, vp]
        L.smaug_get_time.argtypes = [vp, dp, dp]
        L.smaug_get_wavespeeds.argtypes = [vp, dp]
        L.smaug_get_launch_count.argtypes = [vp, C.POINTER(C.c_longlong)]
        L.smaug_get_kernel_info.argtypes = [vp, C.POINTER(C.c_int)]
        L.smaug_get_kernel_name.argtypes = [vp]
        L.smaug_get_kernel_name.restype = C.c_char_p
        L.smaug_set_kernel_timing.argtypes = [vp, C.c_int]
        L.smaug_get_kernel_timing.argtypes = [vp, dp, C.POINTER(C.c_longlong)]
        L.smaug_selftest_division.argtypes = [C.c_int, C.c_int, C.c_ulonglong, C.c_longlong,
                                              C.POINTER(C.c_ulonglong)]
        L.smaug_selftest_fp64_pipe.argtypes = [C.c_int, C.c_int, C.c_int, dp]
        L.smaug_destroy.argtypes = [vp]
        L.smaug_destroy.restype = None
        L.smaug_wavespeeds_static.argtypes = [C.c_int, C.c_int, C.c_double, vp, vp, vp, vp]
        ip = C.POINTER(C.c_int)
        L.smaug_group_create.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, ip, vp, ip, C.POINTER(vp)]
        L.smaug_group_size.argtypes = [vp, ip, ip]
        L.smaug_group_set_param.argtypes = [vp, C.c_int, C.c_double]
        L.smaug_group_set_state.argtypes = [vp, vp]
        L.smaug_group_step.argtypes = [vp, C.c_int, C.c_double]
        L.smaug_group_get_state.argtypes = [vp, vp]
        L.smaug_group_get_time.argtypes = [vp, dp, dp]
        L.smaug_group_get_wavespeeds.argtypes = [vp, dp]
        L.smaug_group_get_launch_count.argtypes = [vp, C.POINTER(C.c_longlong), C.POINTER(C.c_longlong)]
        L.smaug_group_set_timing.argtypes = [vp, C.c_int]
        L.smaug_group_get_tau.argtypes = [vp, dp]
        L.smaug_group_destroy.argtypes = [vp]
        L.smaug_group_destroy.restype = None
        L.smaug_group_map_cell.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, ip, C.c_int, C.c_int, C.c_int, C.c_int, ip]
        L.smaug3_last_error.restype = C.c_char_p
        L.smaug3_workspace_bytes.restype = C.c_size_t
        L.smaug3_workspace_bytes.argtypes = [C.c_int, C.c_int, C.c_int]
        L.smaug3_create.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, ip, vp, C.POINTER(vp)]
        L.smaug3_destroy.argtypes = [vp]
        L.smaug3_destroy.restype = None
        L.smaug3_set_param.argtypes = [vp, C.c_int, C.c_double]
        L.smaug3_set_state.argtypes = [vp, vp]
        L.smaug3_step.argtypes = [vp, C.c_int, C.c_double]
        L.smaug3_get_state.argtypes = [vp, vp]
        L.smaug3_get_time.argtypes = [vp, dp, dp]
        L.smaug3_get_wavespeeds.argtypes = [vp, dp]
        L.smaug3_get_launch_count.argtypes = [vp, C.POINTER(C.c_longlong)]
        L.smaug3_set_kernel_timing.argtypes = [vp, C.c_int]
        L.smaug3_get_kernel_timing.argtypes = [vp, dp, C.POINTER(C.c_longlong)]
        _lib = L
    return _lib


class SmaugError(RuntimeError):
    def __init__(self, code: int):
        self.code = code
        super().__init__(f"smaug error {code}: {lib().smaug_last_error().decode()}")


def _check(rc: int) -> None:
    if rc != 0:
        raise SmaugError(rc)


def _ptr(x):
    """Raw address of a torch tensor or numpy array (must be contiguous float64), or None."""
    if x is None:
        return None
    if hasattr(x, "data_ptr"):
        assert x.is_contiguous() and str(x.dtype) == "torch.float64"
        return C.c_void_p(x.data_ptr())
    assert x.flags["C_CONTIGUOUS"] and x.dtype.name == "float64"
    return C.c_void_p(x.ctypes.data)


def selftest_division(exp_lo: int, exp_hi: int, seed: int = 1, draws: int = 1 << 26) -> dict:
    """smaug_selftest_division: mismatch counts of the division helpers against `/` on the current device."""
    o = (C.c_ulonglong * 5)()
    _check(lib().smaug_selftest_division(int(exp_lo), int(exp_hi), int(seed), int(draws), o))
    return dict(ddiv=o[0], drcp=o[1], ratio_div=o[2], kappa_ratio=o[3], draws=o[4])


def selftest_fp64_pipe(ilp: int, warps_per_subpartition: int, iters: int = 2048):
    """smaug_selftest_fp64_pipe: (cycles per fp64 warp instruction and sub-partition, cycles per trip of the chains)."""
    o = (C.c_double * 2)()
    _check(lib().smaug_selftest_fp64_pipe(int(ilp), int(warps_per_subpartition), int(iters), o))
    return o[0], o[1]


WAVESPEEDS_STATIC_MAX_CELLS = 16384 * 4096     # SMAUG_WAVESPEEDS_STATIC_MAX_CELLS of include/smaug.h


def wavespeeds_static(w, gamma, bg=None, out=None):
    """smaug_wavespeeds_static: the four wave-speed maxima (c-4) of a cuda state tensor ``w[6, ny, nx]`` (and optional
    background ``bg[4, ny, nx]``) without a context and without any device allocation by the library -- for callers
    whose GPU memory is owned by another allocator or who must avoid cudaMalloc's synchronisation.  The library's
    scratch is a fixed array inside libsmaug.so, shared by all calls: do not let two calls overlap on the GPU.

    ``out`` is a 4-element float64 cuda tensor that receives the maxima; pass one you already own to keep torch from
    allocating either (default: a new one).  Enqueued on torch's current stream of ``w``'s device; read ``out`` after
    that stream has caught up (``out.cpu()`` does).  At most WAVESPEEDS_STATIC_MAX_CELLS cells."""
    import torch
    assert w.is_cuda and w.dim() == 3 and w.shape[0] == 6
    ny, nx = int(w.shape[1]), int(w.shape[2])
    if bg is not None:
        assert bg.is_cuda and tuple(bg.shape) == (4, ny, nx)
    with torch.cuda.device(w.device):
        if out is None:
            out = torch.empty(4, dtype=torch.float64, device=w.device)
        assert out.is_cuda and out.numel() == 4
        stream = torch.cuda.current_stream(w.device).cuda_stream
        _check(lib().smaug_wavespeeds_static(nx, ny, float(gamma), _ptr(w), _ptr(bg), _ptr(out), C.c_void_p(stream)))
    return out


class Smaug:
    """One simulation context: smaug_create / set_state / step / get_state / destroy (include/smaug.h).

    State and background are float64, ``[6, ny, nx]`` / ``[4, ny, nx]``, torch (cuda or cpu) tensors or
    numpy arrays.  Device memory is a torch uint8 workspace tensor; work is enqueued on torch's current
    stream of ``device`` at construction time.
    """

    def __init__(self, nx, ny, gamma, bc, bg=None, device="cuda:0", **params):
        import torch
        L = lib()
        self.nx, self.ny = int(nx), int(ny)
        self.device = torch.device(device)
        nbytes = L.smaug_workspace_bytes(self.nx, self.ny, int(bg is not None))
        with torch.cuda.device(self.device):
            self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            base = (self._ws.data_ptr() + 255) // 256 * 256
            stream = torch.cuda.current_stream(self.device).cuda_stream
            h = C.c_void_p()
            bc_arr = (C.c_int * 4)(*[int(b) for b in bc])
            if bg is not None:
                assert tuple(bg.shape) == (4, ny, nx)
            _check(L.smaug_create_in_workspace(self.nx, self.ny, float(gamma), bc_arr, _ptr(bg),
                                               C.c_void_p(base), nbytes, C.c_void_p(stream), C.byref(h)))
        self._h = h
        for k, v in params.items():
            self.set_param(k, v)

    def set_param(self, key, value):
        k = PARAMS[key] if isinstance(key, str) else int(key)
        _check(lib().smaug_set_param(self._h, k, float(value)))

    def set_state(self, w):
        assert tuple(w.shape) == (6, self.ny, self.nx)
        _check(lib().smaug_set_state(self._h, _ptr(w)))

    def step(self, n_steps, cfl=0.3):
        _check(lib().smaug_step(self._h, int(n_steps), float(cfl)))

    def step_async(self, n_steps, cfl=0.3):
        _check(lib().smaug_step_async(self._h, int(n_steps), float(cfl)))

    def get_state(self, out=None):
        """Copy the state into `out` (torch tensor on any device / numpy array); default: new cuda tensor."""
        import torch
        if out is None:
            out = torch.empty((6, self.ny, self.nx), dtype=torch.float64, device=self.device)
        assert tuple(out.shape) == (6, self.ny, self.nx)
        _check(lib().smaug_get_state(self._h, _ptr(out)))
        return out

    def time(self):
        t, dt = C.c_double(), C.c_double()
        _check(lib().smaug_get_time(self._h, C.byref(t), C.byref(dt)))
        return t.value, dt.value

    def wavespeeds(self):
        o = (C.c_double * 4)()
        _check(lib().smaug_get_wavespeeds(self._h, o))
        return list(o)

    def launch_count(self):
        n = C.c_longlong()
        _check(lib().smaug_get_launch_count(self._h, C.byref(n)))
        return n.value

    def kernel_info(self):
        o = (C.c_int * 5)()
        _check(lib().smaug_get_kernel_info(self._h, o))
        return dict(tile_w=o[0], tile_h=o[1], threads=o[2], smem_bytes=o[3], ctas=o[4])

    def kernel_name(self):
        return lib().smaug_get_kernel_name(self._h).decode()

    def set_kernel_timing(self, on=True):
        _check(lib().smaug_set_kernel_timing(self._h, int(on)))

    def kernel_timing(self):
        ms, n = C.c_double(), C.c_longlong()
        _check(lib().smaug_get_kernel_timing(self._h, C.byref(ms), C.byref(n)))
        return ms.value, n.value

    def close(self):
        if getattr(self, "_h", None):
            lib().smaug_destroy(self._h)
            self._h = None
            self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:  # noqa: BLE001
            pass


def group_map_cell(px, py, nx, ny, bc, member, i, j, freeze=0):
    """smaug_group_map_cell (host only): ((x0, y0, nx_m, ny_m), (source member or -1, si, sj))."""
    o = (C.c_int * 7)()
    _check(lib().smaug_group_map_cell(px, py, nx, ny, (C.c_int * 4)(*[int(b) for b in bc]), member, i, j, int(freeze), o))
    return (o[0], o[1], o[2], o[3]), (o[4], o[5], o[6])


class SmaugGroup:
    """A px x py decomposition of one nx-by-ny problem into contexts that exchange halos through peer pointers and share
    one wave-speed reduction (smaug_group_* in include/smaug.h).  Arrays are the GLOBAL state / background."""

    def __init__(self, px, py, nx, ny, gamma, bc, bg=None, devices=None, **params):
        L = lib()
        self.px, self.py, self.nx, self.ny = int(px), int(py), int(nx), int(ny)
        h = C.c_void_p()
        bc_arr = (C.c_int * 4)(*[int(b) for b in bc])
        dev_arr = None if devices is None else (C.c_int * (self.px * self.py))(*[int(d) for d in devices])
        if bg is not None:
            assert tuple(bg.shape) == (4, ny, nx)
        _check(L.smaug_group_create(self.px, self.py, self.nx, self.ny, float(gamma), bc_arr, _ptr(bg), dev_arr, C.byref(h)))
        self._h = h
        for k, v in params.items():
            self.set_param(k, v)

    def set_param(self, key, value):
        k = PARAMS[key] if isinstance(key, str) else int(key)
        _check(lib().smaug_group_set_param(self._h, k, float(value)))

    def set_state(self, w):
        assert tuple(w.shape) == (6, self.ny, self.nx)
        _check(lib().smaug_group_set_state(self._h, _ptr(w)))

    def step(self, n_steps, cfl=0.3):
        _check(lib().smaug_group_step(self._h, int(n_steps), float(cfl)))

    def get_state(self, out=None):
        import torch
        if out is None:
            out = torch.empty((6, self.ny, self.nx), dtype=torch.float64, device="cuda")
        assert tuple(out.shape) == (6, self.ny, self.nx)
        _check(lib().smaug_group_get_state(self._h, _ptr(out)))
        return out

    def time(self):
        t, dt = C.c_double(), C.c_double()
        _check(lib().smaug_group_get_time(self._h, C.byref(t), C.byref(dt)))
        return t.value, dt.value

    def wavespeeds(self):
        o = (C.c_double * 4)()
        _check(lib().smaug_group_get_wavespeeds(self._h, o))
        return list(o)

    def launch_count(self):
        a, b = C.c_longlong(), C.c_longlong()
        _check(lib().smaug_group_get_launch_count(self._h, C.byref(a), C.byref(b)))
        return a.value, b.value

    def set_timing(self, on=True):
        """smaug_group_set_timing: start (and clear) the event record behind tau()."""
        _check(lib().smaug_group_set_timing(self._h, int(on)))

    def tau(self):
        """smaug_group_get_tau: dict(t_comp, t_comm, t_idle in ms -- mean over the members, all steps since
        set_timing(True) -- and tau = ln(t_comp / (t_comm + t_idle)))."""
        o = (C.c_double * 4)()
        _check(lib().smaug_group_get_tau(self._h, o))
        return dict(t_comp=o[0], t_comm=o[1], t_idle=o[2], tau=o[3])

    def close(self):
        if getattr(self, "_h", None):
            lib().smaug_group_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:  # noqa: BLE001
            pass


PARAMS3 = dict(lx=0, ly=1, hd_on=2, c_rho=3, c_mom=4, c_e=5, c_b=6, rk_order=7, fixed_dt=8, gx=10, gy=11, lz=13, gz=14, kernel=15)
KERNEL_KINDS3 = ("ghost fill + dt", "derived quantities", "kappa / interface fluxes", "cell-centred fluxes", "assembly")


class Smaug3DError(RuntimeError):
    def __init__(self, code: int):
        self.code = code
        super().__init__(f"smaug3 error {code}: {lib().smaug3_last_error().decode()}")


def _check3(rc: int) -> None:
    if rc != 0:
        raise Smaug3DError(rc)


class Smaug3D:
    """One 3-D context: smaug3_create / set_state / step / get_state / destroy (include/smaug3d.h).  State: float64
    ``[8, nz, ny, nx]`` = (rho, mx, my, mz, e, bx, by, bz), torch (cuda or cpu) tensors or numpy arrays; the library owns
    its device memory; work is enqueued on torch's current stream of ``device`` at construction time."""

    def __init__(self, nx, ny, nz, gamma, bc, device="cuda:0", **params):
        import torch
        L = lib()
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.device = torch.device(device)
        with torch.cuda.device(self.device):
            stream = torch.cuda.current_stream(self.device).cuda_stream
            h = C.c_void_p()
            _check3(L.smaug3_create(self.nx, self.ny, self.nz, float(gamma), (C.c_int * 6)(*[int(b) for b in bc]),
                                    C.c_void_p(stream), C.byref(h)))
        self._h = h
        for k, v in params.items():
            self.set_param(k, v)

    @property
    def shape(self):
        return (8, self.nz, self.ny, self.nx)

    def set_param(self, key, value):
        k = PARAMS3[key] if isinstance(key, str) else int(key)
        _check3(lib().smaug3_set_param(self._h, k, float(value)))

    def set_state(self, w):
        assert tuple(w.shape) == self.shape
        _check3(lib().smaug3_set_state(self._h, _ptr(w)))

    def step(self, n_steps, cfl=0.3):
        _check3(lib().smaug3_step(self._h, int(n_steps), float(cfl)))

    def get_state(self, out=None):
        import torch
        if out is None:
            out = torch.empty(self.shape, dtype=torch.float64, device=self.device)
        assert tuple(out.shape) == self.shape
        _check3(lib().smaug3_get_state(self._h, _ptr(out)))
        return out

    def time(self):
        t, dt = C.c_double(), C.c_double()
        _check3(lib().smaug3_get_time(self._h, C.byref(t), C.byref(dt)))
        return t.value, dt.value

    def wavespeeds(self):
        o = (C.c_double * 5)()
        _check3(lib().smaug3_get_wavespeeds(self._h, o))
        return list(o)

    def launch_count(self):
        n = C.c_longlong()
        _check3(lib().smaug3_get_launch_count(self._h, C.byref(n)))
        return n.value

    def set_kernel_timing(self, on=True):
        _check3(lib().smaug3_set_kernel_timing(self._h, int(on)))

    def kernel_timing(self):
        """{kind: (milliseconds, launches)} accumulated since set_kernel_timing(True)."""
        ms, n = (C.c_double * 5)(), (C.c_longlong * 5)()
        _check3(lib().smaug3_get_kernel_timing(self._h, ms, n))
        return {k: (ms[i], n[i]) for i, k in enumerate(KERNEL_KINDS3)}

    def close(self):
        if getattr(self, "_h", None):
            lib().smaug3_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:  # noqa: BLE001
            pass
