"""Shared helpers for the parity tests: run the CUDA path through the C ABI, run the oracle, compare.

Parity metrics (BASELINE.json north_star: "max relative
error <= 1e-11 (fp64) / <= 2e-4 (fp32) on density and moments"):
  P1 density: max |g - o| / max(|o|, 1e-6 max|o|); cells outside the disc must be exactly 0.
  P2 moments: max_c |F_g - F_o| / SF_o(c), max_c |tau_g - tau_o| / Stau_o(c)  (cancellation-free scales).
"""
from __future__ import annotations

import numpy as np

import mm_inputs as mi
from oracle import mm_oracle as orc

TOL = {"f64": 1e-11, "f32": 2e-4}
NPDT = {"f64": np.float64, "f32": np.float32}


def p1_density(g: np.ndarray, o: np.ndarray) -> float:
    o = np.asarray(o, np.float64)
    g = np.asarray(g, np.float64)
    scale = np.maximum(np.abs(o), 1e-6 * np.max(np.abs(o)))
    return float(np.max(np.abs(g - o) / scale)) if o.size else 0.0


def p2_moments(force_g, torque_g, om: dict) -> tuple[float, float]:
    sf = np.where(om["SF"] > 0, om["SF"], 1.0)        # SF == 0 only when every offset is 0: force must be 0 too
    stau = np.where(om["Stau"] > 0, om["Stau"], 1.0)
    ef = np.max(np.abs(np.asarray(force_g) - om["force"]) / sf[:, None])
    et = np.max(np.abs(np.asarray(torque_g) - om["torque"]) / stau)
    return float(ef), float(et)


def gpu_run(grid, params, dtype, U, V, Om, m0, schedule, dt, kernel=0, fuse_t=None, fuse_mom=None,
            own_buffers=False, get=True):
    """Run the CUDA path.  schedule: list of n_sub; moments are taken after each entry.
    Returns (density ndarray or None, [(force, torque), ...], MM-info dict)."""
    import torch
    from paper_1908_04279_b200 import MM, binding as b

    tdt = torch.float64 if dtype == "f64" else torch.float32
    cells = grid.cells
    dev = torch.device("cuda:0")
    if own_buffers:
        mm = MM(grid, params, dtype)
    else:
        b0 = torch.empty(cells, dtype=tdt, device=dev)
        b1 = torch.empty(cells, dtype=tdt, device=dev)
        mm = MM(grid, params, dtype, b0, b1)
    mm.set_option(b.MM_OPT_KERNEL, kernel)
    if fuse_t is not None:
        mm.set_option(b.MM_OPT_FUSE_T, fuse_t)
    if fuse_mom is not None:
        mm.set_option(b.MM_OPT_FUSE_MOMENTS, fuse_mom)
    npdt = NPDT[dtype]
    mm.set_density(np.ascontiguousarray(m0, npdt))
    mm.set_filament_velocity(*(np.ascontiguousarray(x, npdt) for x in (U, V, Om)))
    moms = []
    for n in schedule:
        mm.substep(n, dt)
        f = torch.empty((grid.nc, 2), dtype=torch.float64, device=dev)
        t = torch.empty(grid.nc, dtype=torch.float64, device=dev)
        mm.moments(f, t)
        moms.append((f.cpu().numpy(), t.cpu().numpy()))
    out = None
    if get:
        out = np.empty((grid.nc, grid.ns, grid.nxi, grid.neta), npdt)
        mm.get_density(out)
    torch.cuda.synchronize()
    info = dict(kernel=mm.kernel_name, launches=mm.launch_count)
    mm.destroy()
    return out, moms, info


def oracle_run(grid, params, U, V, Om, m0, schedule, dt, c_first=0):
    """Oracle on the same (already dtype-rounded) inputs, promoted to fp64 (Q18)."""
    m = np.asarray(m0, np.float64)
    moms = []
    for n in schedule:
        m = orc.run(grid, params, U, V, Om, m, n, dt, c_first=c_first)
        moms.append(orc.moments(grid, params, m, c_first=c_first))
    return m, moms


def random_inputs(grid, params, dtype, seed=0, omega_max=1.0):
    st = mi.Stream(grid, params.R, seed=seed + 1, omega_max=omega_max,
                   mask_disc=not (params.flags & mi.FLAG_OFFSET_PERIODIC_NOMASK))
    U, V, Om = st.velocities(NPDT[dtype])
    m0 = st.density(grid.nc, NPDT[dtype])
    return U, V, Om, m0


def check_parity(grid, params, dtype, schedule, dt, seed=0, omega_max=1.0, **kw):
    U, V, Om, m0 = random_inputs(grid, params, dtype, seed, omega_max)
    g, gm, info = gpu_run(grid, params, dtype, U, V, Om, m0, schedule, dt, **kw)
    o, om = oracle_run(grid, params, U, V, Om, m0, schedule, dt)
    tol = TOL[dtype]
    e1 = p1_density(g, o)
    assert e1 <= tol, f"density P1 {e1:.3e} > {tol} ({info})"
    if not (params.flags & mi.FLAG_OFFSET_PERIODIC_NOMASK):
        mask = mi.inside_mask(grid.nxi, grid.neta)
        assert (g[:, :, ~mask] == 0).all(), "cells outside the disc must be exactly 0"
    for (f, t), ref in zip(gm, om):
        ef, et = p2_moments(f, t, ref)
        assert ef <= tol and et <= tol, f"moments P2 {ef:.3e} {et:.3e} > {tol} ({info})"
    return e1, info
