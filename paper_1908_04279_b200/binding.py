"""Thin ctypes binding of libmm (include/mm.h).  Argument marshalling only: every step of the hot path
runs in the library's CUDA kernels.  PyTorch supplies device memory and the stream, nothing else.

There is no CPU fallback: if libmm.so cannot be loaded, or no CUDA device is present, calls raise.
"""
from __future__ import annotations

import ctypes
import os

from . import build as _build

MM_F32, MM_F64 = 0, 1
MM_OK, MM_ERR_INVALID_ARG, MM_ERR_CUDA, MM_ERR_NOMEM, MM_ERR_STATE, MM_ERR_UNSTABLE = 0, -1, -2, -3, -4, -5
MM_FLAG_S_PERIODIC, MM_FLAG_OFFSET_PERIODIC_NOMASK, MM_FLAG_CHECK_DT = 1, 2, 4
MM_OPT_KERNEL, MM_OPT_FUSE_T, MM_OPT_FUSE_MOMENTS, MM_OPT_INPLACE, MM_OPT_FREE_COUPLING, MM_OPT_FREE_REFRESH = 0, 1, 2, 3, 4, 5
MM_OPT_SPREAD_ATOMIC = 6
MM_MAX_FUSE_T = 12
MM_LOCAL_FUSE_T = 4

EXPORTS = ["mm_create", "mm_set_density", "mm_get_density", "mm_set_density_range", "mm_get_density_range",
           "mm_set_filament_velocity", "mm_substep", "mm_moments", "mm_set_option", "mm_get_option", "mm_launch_count",
           "mm_kernel_name", "mm_destroy", "mm_status_string", "mm_last_error", "mm_advance_local", "mm_local_steps", "mm_set_psi",
           "mm_spread_force", "mm_update_free_motors", "mm_measure_fma_peak", "mm_measure_fma_rate", "mm_free_motors_noalloc"]
MM_NOALLOC_MAX_NODES = 16384


class mm_grid(ctypes.Structure):
    _fields_ = [(n, ctypes.c_int32) for n in ("nx", "ny", "ntheta", "ns", "nxi", "neta")]


class mm_params(ctypes.Structure):
    _fields_ = [(n, ctypes.c_double) for n in
                ("v0", "f_stall", "k_spring", "k_on", "k_off0", "f_detach", "end_detach_mult", "m_free", "R",
                 "s_lo", "s_hi")] + [("n_end_cells", ctypes.c_int32), ("flags", ctypes.c_uint32)]


class MMError(RuntimeError):
    def __init__(self, status: int, name: str, msg: str):
        super().__init__(f"{name} ({status}): {msg}")
        self.status = status


_lib = None


def lib():
    """Load libmm.so (building it in-tree first if the sources are newer).  Raises if impossible."""
    global _lib
    if _lib is None:
        so = _build.SO
        if not _build.up_to_date():
            so = _build.build()
        L = ctypes.CDLL(so)
        vp, i32, i64, dbl = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_double
        L.mm_create.argtypes = [ctypes.POINTER(mm_grid), ctypes.POINTER(mm_params), ctypes.c_int, vp, vp, vp,
                                ctypes.POINTER(vp)]
        L.mm_set_density.argtypes = [vp, vp, ctypes.c_int]
        L.mm_get_density.argtypes = [vp, vp, ctypes.c_int]
        L.mm_set_density_range.argtypes = [vp, i64, i64, vp, ctypes.c_int]
        L.mm_get_density_range.argtypes = [vp, i64, i64, vp, ctypes.c_int]
        L.mm_set_filament_velocity.argtypes = [vp, vp, vp, vp, ctypes.c_int]
        L.mm_substep.argtypes = [vp, i32, dbl]
        L.mm_moments.argtypes = [vp, vp, vp, ctypes.c_int]
        L.mm_advance_local.argtypes = [vp, dbl, dbl]
        L.mm_local_steps.argtypes = [vp, vp, vp, ctypes.c_int]
        L.mm_set_psi.argtypes = [vp, vp, ctypes.c_int]
        L.mm_spread_force.argtypes = [vp, vp, ctypes.c_int]
        L.mm_update_free_motors.argtypes = [vp, vp, vp, ctypes.c_int]
        L.mm_free_motors_noalloc.argtypes = [ctypes.POINTER(mm_grid), ctypes.POINTER(mm_params), ctypes.c_int, vp, vp, vp, vp, vp]
        L.mm_set_option.argtypes = [vp, ctypes.c_int, i64]
        L.mm_get_option.argtypes = [vp, ctypes.c_int, ctypes.POINTER(i64)]
        L.mm_launch_count.argtypes = [vp]
        L.mm_launch_count.restype = i64
        L.mm_kernel_name.argtypes = [vp]
        L.mm_kernel_name.restype = ctypes.c_char_p
        L.mm_destroy.argtypes = [vp]
        L.mm_status_string.argtypes = [ctypes.c_int]
        L.mm_status_string.restype = ctypes.c_char_p
        L.mm_last_error.argtypes = [vp]
        L.mm_last_error.restype = ctypes.c_char_p
        L.mm_measure_fma_peak.argtypes = [ctypes.c_int, vp, ctypes.POINTER(dbl)]
        L.mm_measure_fma_rate.argtypes = [ctypes.c_int, ctypes.c_int32, vp, ctypes.POINTER(dbl)]
        _lib = L
    return _lib


def _grid_struct(grid) -> mm_grid:
    return mm_grid(*(int(getattr(grid, n)) for n in ("nx", "ny", "ntheta", "ns", "nxi", "neta")))


def _params_struct(p) -> mm_params:
    return mm_params(*(float(getattr(p, n)) for n in
                       ("v0", "f_stall", "k_spring", "k_on", "k_off0", "f_detach", "end_detach_mult", "m_free", "R",
                        "s_lo", "s_hi")), int(p.n_end_cells), int(p.flags))


_DTYPES = {"f32": ("float32", 4), "f64": ("float64", 8), "i32": ("int32", 4)}


def _ptr(x, dtype: str | None = None, numel: int | None = None, what: str = "argument"):
    """(address, on_device) of a torch tensor / numpy array / None.  With dtype ("f32", "f64", "i32") and numel the
    element type and the element count are checked first: the C ABI takes plain pointers and would otherwise
    reinterpret a wrong dtype or run past the end of a short array."""
    if x is None:
        return None, 0
    torch_like = hasattr(x, "data_ptr")
    if not (x.is_contiguous() if torch_like else x.flags.c_contiguous):
        raise ValueError(f"{what}: must be contiguous")
    if dtype is not None:
        name = str(x.dtype).replace("torch.", "")
        if name != _DTYPES[dtype][0]:
            raise TypeError(f"{what}: expected {_DTYPES[dtype][0]}, got {name}")
    if numel is not None:
        n = int(x.numel()) if torch_like else int(x.size)
        if n < numel:
            raise ValueError(f"{what}: needs {numel} elements, got {n}")
    if torch_like:
        return ctypes.c_void_p(x.data_ptr()), int(x.is_cuda)
    return ctypes.c_void_p(x.ctypes.data), 0


def _same_side(*pairs):
    """All non-NULL pointer arguments of one call must live on the same side (host or device): one flag goes to C."""
    sides = {dev for p, dev in pairs if p is not None}
    if len(sides) > 1:
        raise ValueError("mixing host arrays and device tensors in one call")
    return sides.pop() if sides else 0


def measure_fma_peak(dtype: str, stream: int | None = None) -> float:
    """TFLOP/s of a register-only FMA probe of the given dtype on the current device (mm_measure_fma_peak)."""
    L = lib()
    if stream is None:
        import torch
        stream = torch.cuda.current_stream().cuda_stream
    out = ctypes.c_double()
    st = L.mm_measure_fma_peak(MM_F64 if dtype == "f64" else MM_F32, ctypes.c_void_p(stream), ctypes.byref(out))
    if st != MM_OK:
        raise MMError(st, L.mm_status_string(st).decode(), L.mm_last_error(None).decode())
    return float(out.value)


def measure_fma_rate(dtype: str, fresh_operands: int, stream: int | None = None) -> float:
    """TFLOP/s of the FMA probe with 1 or 3 fresh register operands per FMA (mm_measure_fma_rate)."""
    L = lib()
    if stream is None:
        import torch
        stream = torch.cuda.current_stream().cuda_stream
    out = ctypes.c_double()
    st = L.mm_measure_fma_rate(MM_F64 if dtype == "f64" else MM_F32, int(fresh_operands), ctypes.c_void_p(stream), ctypes.byref(out))
    if st != MM_OK:
        raise MMError(st, L.mm_status_string(st).decode(), L.mm_last_error(None).decode())
    return float(out.value)


def free_motors_noalloc(grid, params, dtype: str, density, psi, Mb_coarse, M_free, stream: int | None = None):
    """mm_free_motors_noalloc: the free-motor update without a context and without any allocation (fixed device
    scratch, nx * ny <= MM_NOALLOC_MAX_NODES).  Every array is a DEVICE tensor; `density` is rescaled in place where a
    node is capped; Mb_coarse and M_free are outputs.  Calls that overlap on the GPU race (one shared scratch array)."""
    L = lib()
    if stream is None:
        import torch
        stream = torch.cuda.current_stream().cuda_stream
    nn, nc = grid.nx * grid.ny, grid.nx * grid.ny * grid.ntheta
    args = (_ptr(density, dtype, nc * grid.ns * grid.nxi * grid.neta, "density"), _ptr(psi, "f64", nc, "psi"),
            _ptr(Mb_coarse, "f64", nn, "Mb_coarse"), _ptr(M_free, "f64", nn, "M_free"))
    if any(p is None or not dev for p, dev in args):
        raise ValueError("free_motors_noalloc: density, psi, Mb_coarse and M_free must all be device tensors")
    g, p = _grid_struct(grid), _params_struct(params)
    st = L.mm_free_motors_noalloc(ctypes.byref(g), ctypes.byref(p), MM_F64 if dtype == "f64" else MM_F32, args[0][0],
                                  args[1][0], args[2][0], args[3][0], ctypes.c_void_p(stream))
    if st != MM_OK:
        raise MMError(st, L.mm_status_string(st).decode(), L.mm_last_error(None).decode())
    return Mb_coarse, M_free


class MM:
    """One libmm context.  Method names follow include/mm.h (mm_create -> MM(...), mm_substep -> .substep)."""

    def __init__(self, grid, params, dtype: str, buf0=None, buf1=None, stream: int | None = None):
        self._L = lib()
        self._h = ctypes.c_void_p()
        self.grid, self.params, self.dtype = grid, params, dtype
        self.nc = grid.nx * grid.ny * grid.ntheta
        self.inner = grid.ns * grid.nxi * grid.neta
        self._keep = (buf0, buf1)  # borrowed buffers must outlive the context
        if stream is None:
            import torch
            stream = torch.cuda.current_stream().cuda_stream
        p0, _ = _ptr(buf0)
        p1, _ = _ptr(buf1)
        g, p = _grid_struct(grid), _params_struct(params)
        st = self._L.mm_create(ctypes.byref(g), ctypes.byref(p), MM_F64 if dtype == "f64" else MM_F32, p0, p1,
                               ctypes.c_void_p(stream), ctypes.byref(self._h))
        if st != MM_OK:
            raise MMError(st, self._L.mm_status_string(st).decode(), self._L.mm_last_error(None).decode())

    def _check(self, st: int):
        if st != MM_OK:
            raise MMError(st, self._L.mm_status_string(st).decode(), self._L.mm_last_error(self._h).decode())

    def set_density(self, src):
        p, dev = _ptr(src, self.dtype, self.nc * self.inner, "density")
        self._check(self._L.mm_set_density(self._h, p, dev))

    def get_density(self, dst):
        p, dev = _ptr(dst, self.dtype, self.nc * self.inner, "density")
        self._check(self._L.mm_get_density(self._h, p, dev))
        return dst

    def set_density_range(self, c_begin: int, n_configs: int, src):
        p, dev = _ptr(src, self.dtype, int(n_configs) * self.inner, "density range")
        self._check(self._L.mm_set_density_range(self._h, c_begin, n_configs, p, dev))

    def get_density_range(self, c_begin: int, n_configs: int, dst):
        p, dev = _ptr(dst, self.dtype, int(n_configs) * self.inner, "density range")
        self._check(self._L.mm_get_density_range(self._h, c_begin, n_configs, p, dev))
        return dst

    def set_filament_velocity(self, U, V, Om):
        a = [_ptr(x, self.dtype, self.nc, n) for x, n in ((U, "U"), (V, "V"), (Om, "Omega"))]
        if any(p is None for p, _ in a):
            raise ValueError("U, V, Omega must all be given")
        self._check(self._L.mm_set_filament_velocity(self._h, a[0][0], a[1][0], a[2][0], _same_side(*a)))

    def substep(self, n_sub: int, dt: float):
        self._check(self._L.mm_substep(self._h, int(n_sub), float(dt)))

    def advance_local(self, dt: float, cfl: float):
        self._check(self._L.mm_advance_local(self._h, float(dt), float(cfl)))

    def local_steps(self, n_steps, lam):
        a, b = _ptr(n_steps, "i32", self.nc, "n_steps"), _ptr(lam, "f64", self.nc, "lambda")
        self._check(self._L.mm_local_steps(self._h, a[0], b[0], _same_side(a, b)))
        return n_steps, lam

    def set_psi(self, psi):
        pp, dev = _ptr(psi, "f64", self.nc, "psi")
        self._check(self._L.mm_set_psi(self._h, pp, dev))

    def spread_force(self, F2):
        pf, dev = _ptr(F2, "f64", self.grid.nx * self.grid.ny * 2, "F2")
        self._check(self._L.mm_spread_force(self._h, pf, dev))
        return F2

    def update_free_motors(self, Mb_coarse=None, M_free=None):
        nn = self.grid.nx * self.grid.ny
        a, b = _ptr(Mb_coarse, "f64", nn, "Mb_coarse"), _ptr(M_free, "f64", nn, "M_free")
        self._check(self._L.mm_update_free_motors(self._h, a[0], b[0], _same_side(a, b)))
        return Mb_coarse, M_free

    def moments(self, force, torque):
        a, b = _ptr(force, "f64", 2 * self.nc, "force"), _ptr(torque, "f64", self.nc, "torque")
        self._check(self._L.mm_moments(self._h, a[0], b[0], _same_side(a, b)))
        return force, torque

    def set_option(self, opt: int, value: int):
        self._check(self._L.mm_set_option(self._h, opt, value))

    def get_option(self, opt: int) -> int:
        v = ctypes.c_int64()
        self._check(self._L.mm_get_option(self._h, opt, ctypes.byref(v)))
        return int(v.value)

    @property
    def launch_count(self) -> int:
        return int(self._L.mm_launch_count(self._h))

    @property
    def kernel_name(self) -> str:
        return self._L.mm_kernel_name(self._h).decode()

    def destroy(self):
        if self._h:
            self._L.mm_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass
