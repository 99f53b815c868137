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
