"""Seeded synthetic inputs for the bound-motor microscale step (input recipe only).

SURVEY.md 8(c) S10/S11 and BASELINE.json ``configs``: grids, parameters, the benchmark
``dt`` and the mt19937_64 draw order.  This package holds NO method arithmetic (no fluxes,
rates or moments); it is the only code that both the oracle-side tests and the CUDA-side
harness call.  Neither ``oracle/`` nor ``paper_1908_04279_b200/`` imports it.
"""
from __future__ import annotations

import ctypes
import math
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libmm_inputs.so")
_SRC = os.path.join(_HERE, "gen.c")
_lib = None


def build(force: bool = False) -> str:
    """Compile gen.c -> libmm_inputs.so (in-tree) with gcc."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-fPIC", "-shared", "-std=c99", "-o", _SO, _SRC, "-lm"])
    return _SO


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_SO)
        lib.mmi_open.restype = ctypes.c_void_p
        lib.mmi_open.argtypes = [ctypes.c_uint64]
        lib.mmi_close.argtypes = [ctypes.c_void_p]
        lib.mmi_raw.restype = ctypes.c_uint64
        lib.mmi_raw.argtypes = [ctypes.c_void_p]
        lib.mmi_skip.argtypes = [ctypes.c_void_p, ctypes.c_uint64]
        lib.mmi_draw_velocities.argtypes = [ctypes.c_void_p, ctypes.c_int64, ctypes.c_double] + [ctypes.c_void_p] * 3
        lib.mmi_inside.restype = ctypes.c_int
        lib.mmi_inside.argtypes = [ctypes.c_int] * 4
        lib.mmi_draw_density.restype = ctypes.c_int
        lib.mmi_draw_density.argtypes = [ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                         ctypes.c_double, ctypes.c_int, ctypes.c_int, ctypes.c_void_p]
        _lib = lib
    return _lib


# ----------------------------------------------------------------------------------------
# workload definitions (BASELINE.json configs[0..4])
# ----------------------------------------------------------------------------------------
FLAG_S_PERIODIC = 1
FLAG_OFFSET_PERIODIC_NOMASK = 2
FLAG_CHECK_DT = 4
FLAG_RK2_SUPERBEE = 8   # the paper's RK2 + Superbee-in-s scheme instead of forward Euler + upwind


@dataclass(frozen=True)
class Grid:
    nx: int
    ny: int
    ntheta: int
    ns: int
    nxi: int
    neta: int

    @property
    def nc(self) -> int:
        return self.nx * self.ny * self.ntheta

    @property
    def inner(self) -> int:
        return self.ns * self.nxi * self.neta

    @property
    def cells(self) -> int:
        return self.nc * self.inner


@dataclass(frozen=True)
class Params:
    """Model parameters; defaults are BASELINE.json configs[0] ("params v0=1, f_stall=6, ...")."""
    v0: float = 1.0
    f_stall: float = 6.0
    k_spring: float = 50.0
    k_on: float = 5.0
    k_off0: float = 1.0
    f_detach: float = 2.0
    end_detach_mult: float = 10.0
    m_free: float = 1.0
    R: float = 0.1
    s_lo: float = -0.5
    s_hi: float = 0.5
    n_end_cells: int = 1
    flags: int = 0


@dataclass(frozen=True)
class Workload:
    name: str
    grid: Grid
    dtype: str  # "f64" | "f32"
    n_sub: int
    moments_every: int  # moments after every this many substeps (== n_sub: once at end)
    omega_max: float = 1.0
    seed: int = 1
    params: Params = field(default_factory=Params)

    @property
    def dt(self) -> float:
        return benchmark_dt(self.grid, self.params, self.omega_max)


def benchmark_dt(g: Grid, p: Params, omega_max: float, cfl: float = 0.4,
                 u_max: float = 0.5, v_max: float = 0.5) -> float:
    """SURVEY.md S10 ("dt at CFL 0.4", BASELINE.json configs[0]): dt = CFL / lambda with the
    sum-of-directions advective Courant rate built from the DISTRIBUTION BOUNDS of (U,V,Omega)."""
    ds = (p.s_hi - p.s_lo) / g.ns
    dxi = 2.0 * p.R / g.nxi
    deta = 2.0 * p.R / g.neta
    w_max = p.v0 * (1.0 + p.k_spring * p.R * math.sqrt(2.0) / p.f_stall)
    s_max = 0.5 * (p.s_hi - p.s_lo) - 0.5 * ds
    lam = 0.0
    for k in range(g.ntheta):
        th = 2.0 * math.pi * k / g.ntheta
        c, s = abs(math.cos(th)), abs(math.sin(th))
        lam = max(lam, w_max / ds + (u_max + w_max * c + s_max * omega_max * s) / dxi
                  + (v_max + w_max * s + s_max * omega_max * c) / deta)
    return cfl / lam


CONFIGS = [
    Workload("fp64_tiny", Grid(16, 16, 16, 32, 8, 8), "f64", 100, 100),
    Workload("fp64_medium", Grid(32, 32, 32, 64, 16, 16), "f64", 200, 200),
    Workload("fp32_medium", Grid(32, 32, 32, 64, 16, 16), "f32", 200, 200),
    Workload("fp64_large", Grid(64, 64, 32, 64, 16, 16), "f64", 50, 10),
    Workload("fp32_large", Grid(128, 128, 32, 64, 16, 16), "f32", 50, 10, omega_max=2.0),
]


def inside_mask(nxi: int, neta: int) -> np.ndarray:
    """bool [nxi][neta]: cell centre inside the capture disc xi^2+eta^2 <= R^2 (exact integer test)."""
    a = 2 * np.arange(nxi, dtype=np.int64)[:, None] + 1 - nxi
    b = 2 * np.arange(neta, dtype=np.int64)[None, :] + 1 - neta
    return a * a * neta * neta + b * b * nxi * nxi <= nxi * nxi * neta * neta


class Stream:
    """One mt19937_64 engine walked in the S11 draw order.

    >>> st = Stream(grid, R, seed=1, omega_max=1.0)
    >>> U, V, Om = st.velocities()                 # must be called first, exactly once
    >>> m0 = st.density(n_configs, dtype)          # consecutive configurations, c-major
    """

    def __init__(self, grid: Grid, R: float, seed: int = 1, omega_max: float = 1.0, mask_disc: bool = True):
        self.grid, self.R, self.omega_max, self.mask_disc = grid, R, omega_max, mask_disc
        self._lib = _load()
        self._h = ctypes.c_void_p(self._lib.mmi_open(seed))
        self._vel_done = False
        self.next_config = 0

    def close(self):
        if self._h:
            self._lib.mmi_close(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def velocities(self, dtype=np.float64):
        assert not self._vel_done, "velocities are the first 3*Nc draws"
        nc = self.grid.nc
        U, V, Om = (np.empty(nc, np.float64) for _ in range(3))
        self._lib.mmi_draw_velocities(self._h, nc, self.omega_max, U.ctypes.data, V.ctypes.data, Om.ctypes.data)
        self._vel_done = True
        if np.dtype(dtype) != np.float64:  # fp32 configs: round to nearest (S11)
            U, V, Om = (x.astype(dtype) for x in (U, V, Om))
        return U, V, Om

    def skip_configs(self, n: int):
        assert self._vel_done
        self._lib.mmi_skip(self._h, n * self.grid.inner)
        self.next_config += n

    def density(self, n_configs: int, dtype=np.float64, out: np.ndarray | None = None) -> np.ndarray:
        assert self._vel_done, "call velocities() first (draw order)"
        g = self.grid
        dtype = np.dtype(dtype)
        assert dtype in (np.dtype(np.float64), np.dtype(np.float32))
        if out is None:
            out = np.empty((n_configs, g.ns, g.nxi, g.neta), dtype)
        assert out.dtype == dtype and out.size == n_configs * g.inner and out.flags.c_contiguous
        rc = self._lib.mmi_draw_density(self._h, n_configs, g.ns, g.nxi, g.neta, self.R,
                                        int(self.mask_disc), int(dtype == np.float32), out.ctypes.data)
        assert rc == 0
        self.next_config += n_configs
        return out


def generate(w: Workload, c_begin: int = 0, c_end: int | None = None):
    """(U, V, Om, m0[c_begin:c_end]) for a workload, in its dtype; velocities are for ALL configs."""
    dt = np.float64 if w.dtype == "f64" else np.float32
    c_end = w.grid.nc if c_end is None else c_end
    st = Stream(w.grid, w.params.R, w.seed, w.omega_max,
                mask_disc=not (w.params.flags & FLAG_OFFSET_PERIODIC_NOMASK))
    U, V, Om = st.velocities(dt)
    st.skip_configs(c_begin)
    m0 = st.density(c_end - c_begin, dt)
    st.close()
    return U, V, Om, m0


def raw_outputs(seed: int, n: int) -> list[int]:
    lib = _load()
    h = ctypes.c_void_p(lib.mmi_open(seed))
    out = [lib.mmi_raw(h) for _ in range(n)]
    lib.mmi_close(h)
    return out
