"""Seeded input generator (mm_inputs): engine pin, draw order, chunking, workload table."""
import numpy as np
import pytest

import mm_inputs as mi


def test_engine_pin_cxx_standard():
    # C++ standard [rand.predef]: the 10000th output of a default-seeded (5489) mt19937_64.
    assert mi.raw_outputs(5489, 10000)[-1] == 9981545732273789042


def test_unit_real_from_raw_and_draw_order():
    g = mi.Grid(2, 1, 2, 3, 3, 3)
    raw = mi.raw_outputs(1, 3 * g.nc + 5)
    u = [(r >> 11) * 2.0 ** -53 for r in raw]
    st = mi.Stream(g, 0.1, seed=1, omega_max=2.0)
    U, V, Om = st.velocities()
    for c in range(g.nc):
        assert U[c] == u[3 * c] - 0.5 and V[c] == u[3 * c + 1] - 0.5
        assert Om[c] == 2.0 * (2.0 * u[3 * c + 2] - 1.0)
    m = st.density(1)
    # first cell (j=0,a=0,b=0) of a 3x3 offset grid is inside (all 9 are); envelope at its centre
    xi = -0.1 + 0.5 * (0.2 / 3)
    env = np.exp(-(2 * xi * xi) / (2 * 0.05 ** 2))
    assert m[0, 0, 0, 0] == u[3 * g.nc] * env
    assert m[0, 0, 0, 1] == u[3 * g.nc + 1] * np.exp(-(xi * xi) / (2 * 0.05 ** 2))


def test_mask_counts():
    assert mi.inside_mask(8, 8).sum() == 52       # 52 of 64
    assert mi.inside_mask(16, 16).sum() == 208    # 208 of 256
    assert mi.inside_mask(3, 3).all()


def test_masked_cells_zero_and_stream_position_layout_independent():
    w = mi.CONFIGS[0]
    g = mi.Grid(2, 2, 2, w.grid.ns, 8, 8)
    st = mi.Stream(g, 0.1); st.velocities()
    m = st.density(g.nc)
    mask = mi.inside_mask(8, 8)
    assert (m[:, :, ~mask] == 0).all() and (m[:, :, mask] > 0).all()
    st2 = mi.Stream(g, 0.1, mask_disc=False); st2.velocities()
    m2 = st2.density(g.nc)
    assert np.array_equal(m2[:, :, mask], m[:, :, mask])


def test_chunked_equals_one_shot_and_skip():
    g = mi.Grid(2, 2, 3, 4, 3, 5)
    st = mi.Stream(g, 0.1); st.velocities()
    full = st.density(g.nc)
    st = mi.Stream(g, 0.1); st.velocities()
    parts = [st.density(5), st.density(g.nc - 5)]
    assert np.array_equal(np.concatenate(parts), full)
    st = mi.Stream(g, 0.1); st.velocities(); st.skip_configs(7)
    assert np.array_equal(st.density(2), full[7:9])


def test_fp32_rounding():
    g = mi.Grid(1, 1, 2, 4, 3, 3)
    a = mi.Stream(g, 0.1); Ua = a.velocities()[0]; ma = a.density(2)
    b = mi.Stream(g, 0.1); Ub = b.velocities(np.float32)[0]; mb = b.density(2, np.float32)
    assert mb.dtype == np.float32 and np.array_equal(mb, ma.astype(np.float32))
    assert np.array_equal(Ub, Ua.astype(np.float32))


def test_workload_table_and_dt():
    cells = [w.grid.cells for w in mi.CONFIGS]
    assert cells == [8388608, 536870912, 536870912, 2 ** 31, 2 ** 33]
    # SURVEY.md S10 survey-computed values
    assert mi.CONFIGS[0].dt == pytest.approx(1.536405363642338e-3, rel=1e-14)
    assert mi.CONFIGS[1].dt == pytest.approx(7.669008644268185e-4, rel=1e-14)
    assert mi.CONFIGS[3].dt == mi.CONFIGS[1].dt == mi.CONFIGS[2].dt
    assert mi.CONFIGS[4].dt == pytest.approx(6.92923309737695e-4, rel=1e-14)
