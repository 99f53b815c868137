"""ctypes wrapper of oracle/mm_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It imports nothing from paper_1908_04279_b200/ or mm_inputs/.
See mm_oracle.c's header for the passages followed (Eq. 4, PAPER.md:43,
PAPER.md:80-81 Eq. 10, Alg. 2; BASELINE.json north_star (1)-(3)).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mm_oracle.c")
_SO = os.path.join(_HERE, "libmm_oracle.so")
_lib = None

S_PERIODIC = 1
OFFSET_PERIODIC_NOMASK = 2
RK2_SUPERBEE = 8


class OGrid(ctypes.Structure):
    _fields_ = [(n, ctypes.c_int32) for n in ("nx", "ny", "ntheta", "ns", "nxi", "neta")]


class OParams(ctypes.Structure):
    _fields_ = [(n, ctypes.c_double) for n in
                ("v0", "f_stall", "k_spring", "k_on", "k_off0", "f_detach", "end_detach_mult", "m_free", "R",
                 "s_lo", "s_hi")] + [("n_end_cells", ctypes.c_int32), ("flags", ctypes.c_uint32)]


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp, no -ffast-math."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c99", "-ffp-contract=off",
                               "-o", _SO, _SRC, "-lm"])
    return _SO


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_SO)
        vp, i64, i32, dbl = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32, ctypes.c_double
        lib.mmo_run.restype = ctypes.c_int
        lib.mmo_run.argtypes = [vp, vp, i64, i64, vp, vp, vp, vp, i32, dbl]
        lib.mmo_moments.restype = ctypes.c_int
        lib.mmo_moments.argtypes = [vp, vp, i64, i64, vp, vp, vp, vp, vp, vp]
        lib.mmo_rate_bound.restype = ctypes.c_int
        lib.mmo_rate_bound.argtypes = [vp, vp, i64, i64, vp, vp, vp, vp]
        lib.mmo_advance_local.restype = ctypes.c_int
        lib.mmo_advance_local.argtypes = [vp, vp, i64, i64, vp, vp, vp, vp, dbl, dbl, vp]
        lib.mmo_spread_force.restype = ctypes.c_int
        lib.mmo_spread_force.argtypes = [vp, vp, i64, i64, vp, vp, vp]
        lib.mmo_free_motors.restype = ctypes.c_int
        lib.mmo_free_motors.argtypes = [vp, vp, vp, vp, vp, vp]
        lib.mmo_run_coupled.restype = ctypes.c_int
        lib.mmo_run_coupled.argtypes = [vp, vp, i64, i64, vp, vp, vp, vp, i32, dbl, vp]
        lib.mmo_run_alg2.restype = ctypes.c_int
        lib.mmo_run_alg2.argtypes = [vp, vp, vp, vp, vp, vp, vp, i32, dbl, i32, vp, vp]
        lib.mmo_advance_local_coupled.restype = ctypes.c_int
        lib.mmo_advance_local_coupled.argtypes = [vp, vp, i64, i64, vp, vp, vp, vp, dbl, dbl, vp, vp]
        lib.mmo_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def _grid(grid) -> OGrid:
    return OGrid(*(int(getattr(grid, n)) for n in ("nx", "ny", "ntheta", "ns", "nxi", "neta")))


def _params(p) -> OParams:
    return OParams(*(float(getattr(p, n)) for n in
                     ("v0", "f_stall", "k_spring", "k_on", "k_off0", "f_detach", "end_detach_mult", "m_free", "R",
                      "s_lo", "s_hi")), int(p.n_end_cells), int(p.flags))


def _f64(x, n=None):
    x = np.ascontiguousarray(x, dtype=np.float64)
    if n is not None:
        assert x.size == n, (x.size, n)
    return x


def threads() -> int:
    return _load().mmo_threads()


def run(grid, params, U, V, Om, m, n_sub: int, dt: float, c_first: int = 0) -> np.ndarray:
    """n_sub explicit substeps (S2-S7) of the configurations held in ``m``.

    m: [n][ns][nxi][neta] (any float dtype; promoted to fp64, Q18); U,V,Om: [n], the velocities of
    exactly these configurations; c_first = global index of the first one (fixes theta).  Returns a
    new fp64 array."""
    lib = _load()
    g, p = _grid(grid), _params(params)
    inner = grid.ns * grid.nxi * grid.neta
    out = np.array(m, dtype=np.float64, order="C", copy=True)
    n = out.size // inner
    assert out.size == n * inner
    U, V, Om = _f64(U, n), _f64(V, n), _f64(Om, n)
    rc = lib.mmo_run(ctypes.byref(g), ctypes.byref(p), c_first, n, U.ctypes.data, V.ctypes.data, Om.ctypes.data,
                     out.ctypes.data, n_sub, dt)
    if rc != 0:
        raise MemoryError("oracle scratch allocation failed")
    return out.reshape(n, grid.ns, grid.nxi, grid.neta)


def rate_bound(grid, params, U, V, Om, c_first: int = 0) -> np.ndarray:
    """lambda_c of SURVEY.md 8(f) NEXT-3 (reading Q32): the S8 positivity rate maximised over the disc cells."""
    lib = _load()
    g, p = _grid(grid), _params(params)
    U, V, Om = _f64(U), _f64(V, U.size if hasattr(U, "size") else None), _f64(Om)
    lam = np.empty(U.size)
    lib.mmo_rate_bound(ctypes.byref(g), ctypes.byref(p), c_first, U.size, U.ctypes.data, V.ctypes.data,
                       Om.ctypes.data, lam.ctypes.data)
    return lam


def run_alg2(grid, params, U, V, Om, m, psi, n_sub: int, dt: float, refresh: int):
    """Alg. 2 with the paper's cadence: before every `refresh`-th substep the coarse reduction, the
    cap and M_f are redone on the whole state.  m: ALL configurations.  Returns (density, M_b,coarse, M_f of the last
    update)."""
    lib = _load()
    g, p = _grid(grid), _params(params)
    nc = grid.nx * grid.ny * grid.ntheta
    out = np.array(m, dtype=np.float64, order="C", copy=True)
    assert out.size == nc * grid.ns * grid.nxi * grid.neta
    U, V, Om, psi = _f64(U, nc), _f64(V, nc), _f64(Om, nc), _f64(psi, nc)
    Mbc, Mf = np.empty((grid.nx, grid.ny)), np.empty((grid.nx, grid.ny))
    rc = lib.mmo_run_alg2(ctypes.byref(g), ctypes.byref(p), U.ctypes.data, V.ctypes.data, Om.ctypes.data, out.ctypes.data,
                          psi.ctypes.data, n_sub, dt, refresh, Mbc.ctypes.data, Mf.ctypes.data)
    if rc != 0:
        raise RuntimeError(f"mmo_run_alg2 failed ({rc})")
    return out.reshape(nc, grid.ns, grid.nxi, grid.neta), Mbc, Mf


def advance_local(grid, params, U, V, Om, m, dt: float, cfl: float, c_first: int = 0, Mf=None):
    """Every configuration from t to t + dt with its own n_c = max(1, ceil(dt lambda_c / cfl)) equal local steps
    (Alg. 2 l.2-5; readings Q31-Q33); with Mf [nx][ny] the source is k_on M_f(r0) (reading Q42).
    Returns (new fp64 density, n_c int32 array)."""
    lib = _load()
    if Mf is not None:
        g, p = _grid(grid), _params(params)
        inner = grid.ns * grid.nxi * grid.neta
        out = np.array(m, dtype=np.float64, order="C", copy=True)
        n = out.size // inner
        U, V, Om = _f64(U, n), _f64(V, n), _f64(Om, n)
        Mf = _f64(Mf, grid.nx * grid.ny)
        nst = np.empty(n, np.int32)
        rc = lib.mmo_advance_local_coupled(ctypes.byref(g), ctypes.byref(p), c_first, n, U.ctypes.data, V.ctypes.data,
                                           Om.ctypes.data, out.ctypes.data, dt, cfl, nst.ctypes.data, Mf.ctypes.data)
        if rc != 0:
            raise MemoryError("oracle scratch allocation failed")
        return out.reshape(n, grid.ns, grid.nxi, grid.neta), nst
    g, p = _grid(grid), _params(params)
    inner = grid.ns * grid.nxi * grid.neta
    out = np.array(m, dtype=np.float64, order="C", copy=True)
    n = out.size // inner
    U, V, Om = _f64(U, n), _f64(V, n), _f64(Om, n)
    nst = np.empty(n, np.int32)
    rc = lib.mmo_advance_local(ctypes.byref(g), ctypes.byref(p), c_first, n, U.ctypes.data, V.ctypes.data,
                               Om.ctypes.data, out.ctypes.data, dt, cfl, nst.ctypes.data)
    if rc != 0:
        raise MemoryError("oracle scratch allocation failed")
    return out.reshape(n, grid.ns, grid.nxi, grid.neta), nst


def spread_force(grid, params, m, psi, c_first: int = 0, F2=None) -> np.ndarray:
    """Motor-force spreading (Eq. 10; readings Q34-Q37): F2[nx][ny][2] += contributions of the
    configurations held in ``m`` (Psi-weighted plane forces spread with Peskin's 4-point delta at x_c + s_j p_c)."""
    lib = _load()
    g, p = _grid(grid), _params(params)
    inner = grid.ns * grid.nxi * grid.neta
    m = _f64(m)
    n = m.size // inner
    psi = _f64(psi, n)
    if F2 is None:
        F2 = np.zeros((grid.nx, grid.ny, 2))
    assert F2.dtype == np.float64 and F2.flags.c_contiguous and F2.shape == (grid.nx, grid.ny, 2)
    lib.mmo_spread_force(ctypes.byref(g), ctypes.byref(p), c_first, n, m.ctypes.data, psi.ctypes.data, F2.ctypes.data)
    return F2


def free_motors(grid, params, m, psi):
    """Free-motor coupling (Eq. 5-6, Alg. 2 l.14-20; readings Q38-Q42).  m: ALL configurations.  Returns
    (m after the cap rescale [fp64 copy], M_b,coarse [nx][ny] after the cap, M_f [nx][ny])."""
    lib = _load()
    g, p = _grid(grid), _params(params)
    out = np.array(m, dtype=np.float64, order="C", copy=True)
    nc = grid.nx * grid.ny * grid.ntheta
    assert out.size == nc * grid.ns * grid.nxi * grid.neta
    psi = _f64(psi, nc)
    Mbc, Mf = np.empty((grid.nx, grid.ny)), np.empty((grid.nx, grid.ny))
    rc = lib.mmo_free_motors(ctypes.byref(g), ctypes.byref(p), out.ctypes.data, psi.ctypes.data, Mbc.ctypes.data, Mf.ctypes.data)
    if rc != 0:
        raise MemoryError("oracle scratch allocation failed")
    return out.reshape(nc, grid.ns, grid.nxi, grid.neta), Mbc, Mf


def run_coupled(grid, params, U, V, Om, m, n_sub: int, dt: float, Mf, c_first: int = 0) -> np.ndarray:
    """`run` with the source k_on M_f(r0) of the free-motor table Mf [nx][ny] (reading Q42)."""
    lib = _load()
    g, p = _grid(grid), _params(params)
    inner = grid.ns * grid.nxi * grid.neta
    out = np.array(m, dtype=np.float64, order="C", copy=True)
    n = out.size // inner
    U, V, Om = _f64(U, n), _f64(V, n), _f64(Om, n)
    Mf = _f64(Mf, grid.nx * grid.ny)
    rc = lib.mmo_run_coupled(ctypes.byref(g), ctypes.byref(p), c_first, n, U.ctypes.data, V.ctypes.data, Om.ctypes.data,
                             out.ctypes.data, n_sub, dt, Mf.ctypes.data)
    if rc != 0:
        raise MemoryError("oracle scratch allocation failed")
    return out.reshape(n, grid.ns, grid.nxi, grid.neta)


def moments(grid, params, m, c_first: int = 0):
    """S9.  Returns dict(force[n,2], torque[n], N0[n], SF[n], Stau[n])."""
    lib = _load()
    g, p = _grid(grid), _params(params)
    inner = grid.ns * grid.nxi * grid.neta
    m = _f64(m)
    n = m.size // inner
    force = np.empty((n, 2)); torque = np.empty(n); N0 = np.empty(n); SF = np.empty(n); St = np.empty(n)
    lib.mmo_moments(ctypes.byref(g), ctypes.byref(p), c_first, n, m.ctypes.data, force.ctypes.data,
                    torque.ctypes.data, N0.ctypes.data, SF.ctypes.data, St.ctypes.data)
    return dict(force=force, torque=torque, N0=N0, SF=SF, Stau=St)
