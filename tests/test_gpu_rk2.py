"""GPU parity of the second scheme (MM_FLAG_RK2_SUPERBEE: RK2 through the half step + Superbee in s; SURVEY.md 8(f)
NEXT-1) against the oracle's RK2 mode, element by element, through the C ABI."""
import dataclasses

import numpy as np
import pytest

import mm_inputs as mi
from mm_inputs import Grid, Params
from util import check_parity, gpu_run, oracle_run, random_inputs, p1_density, TOL

pytestmark = pytest.mark.gpu
RK2 = mi.FLAG_RK2_SUPERBEE


def _dt(g, p, om=1.0, cfl=0.4):
    return mi.benchmark_dt(g, p, om, cfl=cfl)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("shape", [(2, 2, 2, 4, 3, 3), (1, 3, 5, 5, 3, 7), (2, 1, 4, 9, 16, 16), (1, 1, 3, 2, 1, 1)])
def test_rk2_generic_small_grids(dtype, shape):
    g = Grid(*shape)
    p = Params(flags=RK2)
    e, info = check_parity(g, p, dtype, [3, 4], _dt(g, p), kernel=1)
    assert info["kernel"].startswith("rk2_"), info


@pytest.mark.parametrize("flags", [mi.FLAG_S_PERIODIC, mi.FLAG_OFFSET_PERIODIC_NOMASK,
                                   mi.FLAG_S_PERIODIC | mi.FLAG_OFFSET_PERIODIC_NOMASK])
def test_rk2_generic_periodic_flags(flags):
    g = Grid(2, 2, 4, 6, 5, 4)
    p = Params(flags=flags | RK2)
    check_parity(g, p, "f64", [5, 5], _dt(g, p), kernel=1)


def test_rk2_generic_stall_clamp_and_wide_ends():
    g = Grid(1, 2, 8, 12, 8, 8)
    p = Params(k_spring=200.0, n_end_cells=3, end_detach_mult=4.0, flags=RK2)
    check_parity(g, p, "f64", [6], 0.3 * _dt(g, p), kernel=1)


def test_rk2_differs_from_euler_and_buffers_stay_put():
    """The flag really switches the scheme, and after a substep the current buffer is the one it was (stage 2 writes
    in place), so mm_get_density / mm_moments read the right one for odd and even substep counts."""
    g = Grid(1, 2, 4, 8, 8, 8)
    p = Params(flags=RK2)
    dt = _dt(g, p)
    U, V, Om, m0 = random_inputs(g, p, "f64")
    for n in (1, 2, 3):
        out, _, _ = gpu_run(g, p, "f64", U, V, Om, m0, [n], dt)
        ref, _ = oracle_run(g, p, U, V, Om, m0, [n], dt)
        assert p1_density(out, ref) < TOL["f64"]
    eul, _ = oracle_run(g, dataclasses.replace(p, flags=0), U, V, Om, m0, [3], dt)
    assert p1_density(out, eul) > 1e-4


# ------------------------------------------------------------------ fused one-pass kernel (rk2_fused_kernel)
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("nxi", [16, 8])
@pytest.mark.parametrize("ns", [7, 6, 2, 1])
def test_rk2_fused_parity(dtype, nxi, ns):
    # 700 configurations: several per warp; Ns = 7: ragged last chunk; Ns = 2, 1: shorter than the stage skew
    g = Grid(5, 7, 20, ns, nxi, nxi)
    p = Params(flags=RK2, n_end_cells=1 if ns >= 2 else 0)
    e, info = check_parity(g, p, dtype, [3, 2], _dt(g, p))
    assert info["kernel"].startswith("rk2_fused<"), info


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_rk2_fused_baseline_shape_and_omega2(dtype):
    g = Grid(2, 2, 8, 64, 16, 16)
    p = Params(flags=RK2)
    check_parity(g, p, dtype, [6], _dt(g, p, 2.0), omega_max=2.0)


def test_rk2_fused_equals_generic_and_stall_clamp():
    g = Grid(2, 2, 8, 9, 16, 16)
    p = Params(k_spring=200.0, n_end_cells=2, end_detach_mult=3.0, flags=RK2)
    dt = 0.25 * _dt(g, p, 2.0)
    U, V, Om, m0 = random_inputs(g, p, "f64", omega_max=2.0)
    a, ma, ia = gpu_run(g, p, "f64", U, V, Om, m0, [5], dt)
    b, mb, ib = gpu_run(g, p, "f64", U, V, Om, m0, [5], dt, kernel=1)
    assert ia["kernel"].startswith("rk2_fused<") and ib["kernel"].startswith("rk2_generic<")
    e = p1_density(a, b)
    assert e < 1e-12, e   # same method, different order of operations (coefficient form vs flux form)
    ref, _ = oracle_run(g, p, U, V, Om, m0, [5], dt)
    assert p1_density(a, ref) < TOL["f64"]


def test_rk2_fused_dirty_masked_input_and_zero_rates():
    g = Grid(1, 2, 4, 6, 16, 16)
    p = Params(flags=RK2)
    dt = _dt(g, p)
    U, V, Om, m0 = random_inputs(g, p, "f64")
    m0 = m0.copy(); m0[:, :, ~mi.inside_mask(16, 16)] = 3.0
    out, _, _ = gpu_run(g, p, "f64", U, V, Om, m0, [2], dt)
    ref, _ = oracle_run(g, p, U, V, Om, m0, [2], dt)
    assert p1_density(out, ref) < TOL["f64"]
    p0 = Params(k_on=0.0, v0=0.0, k_spring=0.0, flags=RK2)
    check_parity(g, p0, "f64", [4], dt)
