"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element.

Sizes here are small enough for the oracle to finish in seconds while still spanning several warps,
several TMA ring wraps, ragged chunk tails (Ns odd) and more configurations than resident warps.
Full BASELINE.json sizes live in test_gpu_baseline_configs.py.
"""
import dataclasses

import numpy as np
import pytest

import mm_inputs as mi
from mm_inputs import Grid, Params
from util import check_parity, gpu_run, oracle_run, random_inputs, p1_density, TOL
from oracle import mm_oracle as orc

pytestmark = pytest.mark.gpu


def _dt(g, p, om=1.0, cfl=0.4):
    return mi.benchmark_dt(g, p, om, cfl=cfl)


# ------------------------------------------------------------------ generic kernels: any size, all flags
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("shape", [(2, 2, 2, 4, 3, 3), (1, 3, 5, 5, 3, 7), (2, 1, 4, 9, 16, 16), (1, 1, 3, 2, 1, 1)])
def test_generic_small_grids(dtype, shape):
    g = Grid(*shape)
    p = Params()
    check_parity(g, p, dtype, [3, 4], _dt(g, p), kernel=1)


@pytest.mark.parametrize("flags", [mi.FLAG_S_PERIODIC, mi.FLAG_OFFSET_PERIODIC_NOMASK,
                                   mi.FLAG_S_PERIODIC | mi.FLAG_OFFSET_PERIODIC_NOMASK])
def test_generic_periodic_flags(flags):
    g = Grid(2, 2, 4, 6, 5, 4)
    p = Params(flags=flags)
    check_parity(g, p, "f64", [5, 5], _dt(g, p), kernel=1)


def test_generic_stall_clamp_and_wide_ends():
    g = Grid(1, 2, 8, 12, 8, 8)
    p = Params(k_spring=200.0, n_end_cells=3, end_detach_mult=4.0)
    check_parity(g, p, "f64", [6], 0.3 * _dt(g, p), kernel=1)


# ------------------------------------------------------------------ streamed kernels
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("T", [1, 2, 3, 4])
@pytest.mark.parametrize("nxi", [16, 8])
def test_stream_kernel_parity(dtype, T, nxi):
    # 700 configurations > resident warps on 148 SMs? no (that needs ~2000); still several per warp when
    # the grid is capped to ceil(Nc/4) blocks; Ns=7 gives a ragged last chunk (P=2).
    g = Grid(5, 7, 20, 7, nxi, nxi)
    p = Params()
    e, info = check_parity(g, p, dtype, [5, 3], _dt(g, p), kernel=2, fuse_t=T)
    assert info["kernel"].startswith("stream<"), info


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_stream_many_configs_per_warp(dtype):
    """More configurations than the launch has warps: exercises the ring running across configuration
    boundaries and per-configuration re-initialisation."""
    g = Grid(16, 16, 16, 6, 8, 8)   # 4096 configs of 384 cells
    p = Params()
    check_parity(g, p, dtype, [4], _dt(g, p), kernel=2, fuse_t=2)


def test_stream_equals_generic_and_fusion_invariance():
    """C8 on the GPU: T-fused passes == T=1 passes == generic kernel, and substep(a);substep(b) == substep(a+b)."""
    g = Grid(3, 3, 8, 10, 16, 16)
    p = Params()
    dt = _dt(g, p)
    U, V, Om, m0 = random_inputs(g, p, "f64")
    ref, _, _ = gpu_run(g, p, "f64", U, V, Om, m0, [7], dt, kernel=1)
    for T in (1, 2, 3, 4):
        out, _, info = gpu_run(g, p, "f64", U, V, Om, m0, [7], dt, kernel=2, fuse_t=T)
        assert p1_density(out, ref) < 1e-13, (T, info)
    a, _, _ = gpu_run(g, p, "f64", U, V, Om, m0, [3, 4], dt, kernel=2, fuse_t=2)
    b, _, _ = gpu_run(g, p, "f64", U, V, Om, m0, [7], dt, kernel=2, fuse_t=2)
    assert p1_density(a, b) < 1e-13


def test_stream_moments_fused_equals_standalone():
    g = Grid(2, 3, 8, 12, 16, 16)
    p = Params()
    dt = _dt(g, p)
    U, V, Om, m0 = random_inputs(g, p, "f64")
    _, mf, _ = gpu_run(g, p, "f64", U, V, Om, m0, [4, 4], dt, kernel=2, fuse_t=2, fuse_mom=1)
    _, ms, _ = gpu_run(g, p, "f64", U, V, Om, m0, [4, 4], dt, kernel=2, fuse_t=2, fuse_mom=0)
    for (f1, t1), (f2, t2) in zip(mf, ms):
        assert np.allclose(f1, f2, rtol=0, atol=1e-15) and np.allclose(t1, t2, rtol=0, atol=1e-15)


def test_stream_stall_clamp_wide_ends_and_omega2():
    g = Grid(2, 2, 8, 9, 16, 16)
    p = Params(k_spring=200.0, n_end_cells=2, end_detach_mult=3.0)
    check_parity(g, p, "f64", [6], 0.25 * _dt(g, p, 2.0), omega_max=2.0, kernel=2, fuse_t=3)


def test_library_owned_buffers_and_permutation_invariance():
    """NULL,NULL buffers (library allocates) and C8: same-theta configurations swapped -> outputs swapped bitwise."""
    g = Grid(2, 2, 4, 8, 8, 8)
    p = Params()
    dt = _dt(g, p)
    U, V, Om, m0 = random_inputs(g, p, "f64")
    out, _, _ = gpu_run(g, p, "f64", U, V, Om, m0, [5], dt, own_buffers=True)
    perm = np.arange(g.nc); perm[[1, 1 + g.ntheta]] = perm[[1 + g.ntheta, 1]]
    out2, _, _ = gpu_run(g, p, "f64", U[perm], V[perm], Om[perm], m0[perm], [5], dt, own_buffers=True)
    assert np.array_equal(out2, out[perm])


def test_positivity_and_mask_on_gpu():
    g = Grid(2, 2, 8, 16, 16, 16)
    p = Params()
    U, V, Om, m0 = random_inputs(g, p, "f32")
    out, _, _ = gpu_run(g, p, "f32", U, V, Om, m0, [50], _dt(g, p))
    mask = mi.inside_mask(16, 16)
    assert (out >= 0).all() and (out[:, :, ~mask] == 0).all() and (out[:, :, mask] > 0).all()


def test_dirty_masked_input_is_dropped():
    g = Grid(1, 2, 4, 6, 16, 16)
    p = Params()
    dt = _dt(g, p)
    U, V, Om, m0 = random_inputs(g, p, "f64")
    m0 = m0.copy(); m0[:, :, ~mi.inside_mask(16, 16)] = 3.0
    out, _, _ = gpu_run(g, p, "f64", U, V, Om, m0, [2], dt, kernel=2, fuse_t=2)
    ref, _ = oracle_run(g, p, U, V, Om, m0, [2], dt)
    assert p1_density(out, ref) < TOL["f64"]


# ------------------------------------------------------------------ tile kernels (tiled TMA + shared-memory level exchange)
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("T", [1, 2, 3, 4])
@pytest.mark.parametrize("nxi", [16, 8])
def test_tile_kernel_parity(dtype, T, nxi):
    # Ns=7: ragged last chunk (P=2); 700 configurations: several per warp, and for 8x8 a ragged last group of 4
    g = Grid(5, 7, 20, 7, nxi, nxi) if nxi == 16 else Grid(5, 7, 19, 7, nxi, nxi)
    p = Params()
    e, info = check_parity(g, p, dtype, [5, 3], _dt(g, p), kernel=3, fuse_t=T)
    assert info["kernel"].startswith("tile<"), info


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_tile_many_configs_per_warp(dtype):
    g = Grid(16, 16, 16, 6, 8, 8)   # 4096 configs of 384 cells: 1024 groups of 4
    p = Params()
    check_parity(g, p, dtype, [4], _dt(g, p), kernel=3, fuse_t=2)


def test_tile_equals_generic_and_fusion_invariance():
    g = Grid(3, 3, 8, 10, 16, 16)
    p = Params()
    dt = _dt(g, p)
    U, V, Om, m0 = random_inputs(g, p, "f64")
    ref, _, _ = gpu_run(g, p, "f64", U, V, Om, m0, [7], dt, kernel=1)
    for T in (1, 2, 3, 4):
        out, _, info = gpu_run(g, p, "f64", U, V, Om, m0, [7], dt, kernel=3, fuse_t=T)
        assert p1_density(out, ref) < 1e-13, (T, info)
    a, _, _ = gpu_run(g, p, "f64", U, V, Om, m0, [3, 4], dt, kernel=3, fuse_t=2)
    b, _, _ = gpu_run(g, p, "f64", U, V, Om, m0, [7], dt, kernel=3, fuse_t=2)
    assert p1_density(a, b) < 1e-13


def test_tile_moments_fused_equals_standalone():
    g = Grid(2, 3, 8, 12, 16, 16)
    p = Params()
    dt = _dt(g, p)
    U, V, Om, m0 = random_inputs(g, p, "f64")
    _, mf, _ = gpu_run(g, p, "f64", U, V, Om, m0, [4, 4], dt, kernel=3, fuse_t=2, fuse_mom=1)
    _, ms, _ = gpu_run(g, p, "f64", U, V, Om, m0, [4, 4], dt, kernel=3, fuse_t=2, fuse_mom=0)
    for (f1, t1), (f2, t2) in zip(mf, ms):
        assert np.allclose(f1, f2, rtol=0, atol=1e-14) and np.allclose(t1, t2, rtol=0, atol=1e-14)


def test_tile_stall_clamp_wide_ends_and_omega2():
    g = Grid(2, 2, 8, 9, 16, 16)
    p = Params(k_spring=200.0, n_end_cells=2, end_detach_mult=3.0)
    check_parity(g, p, "f64", [6], 0.25 * _dt(g, p, 2.0), omega_max=2.0, kernel=3, fuse_t=3)


def test_tile_dirty_masked_input_is_dropped():
    g = Grid(1, 2, 4, 6, 16, 16)
    p = Params()
    dt = _dt(g, p)
    U, V, Om, m0 = random_inputs(g, p, "f64")
    m0 = m0.copy(); m0[:, :, ~mi.inside_mask(16, 16)] = 3.0
    out, _, _ = gpu_run(g, p, "f64", U, V, Om, m0, [2], dt, kernel=3, fuse_t=2)
    ref, _ = oracle_run(g, p, U, V, Om, m0, [2], dt)
    assert p1_density(out, ref) < TOL["f64"]


# ------------------------------------------------------------------ coefficient-form kernels (mm_coef.cuh)
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("T", [1, 2, 3, 4, 5, 6])
@pytest.mark.parametrize("nxi", [16, 8])
def test_coef_kernel_parity(dtype, T, nxi):
    # Ns=7: ragged last chunk (P=2); 700 configurations: several per warp
    g = Grid(5, 7, 20, 7, nxi, nxi)
    p = Params()
    e, info = check_parity(g, p, dtype, [11, 7] if T > 4 else [5, 3], _dt(g, p), kernel=4, fuse_t=T)
    assert info["kernel"].startswith("coef<"), info


@pytest.mark.parametrize("T", [7, 8, 9, 10])
def test_coef_deep_fusion_fp32(T):
    """Depth 7-10 (fp32, 16x16 only): the upwind planes of the levels beyond 6 live in shared memory."""
    g = Grid(5, 7, 20, 7, 16, 16)
    p = Params()
    e, info = check_parity(g, p, "f32", [2 * T + 3, T], _dt(g, p), kernel=4, fuse_t=T)
    assert info["kernel"].startswith("coef<f32"), info
    # other dtypes / planes clamp the depth to 6 and still match
    check_parity(Grid(3, 3, 8, 7, 8, 8), p, "f32", [13], _dt(Grid(3, 3, 8, 7, 8, 8), p), kernel=4, fuse_t=T)
    check_parity(g, p, "f64", [13], _dt(g, p), kernel=4, fuse_t=T)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_coef_many_configs_per_warp(dtype):
    g = Grid(16, 16, 16, 6, 8, 8)   # 4096 configs of 384 cells
    p = Params()
    check_parity(g, p, dtype, [4], _dt(g, p), kernel=4, fuse_t=2)


def test_coef_equals_generic_and_fusion_invariance():
    g = Grid(3, 3, 8, 10, 16, 16)
    p = Params()
    dt = _dt(g, p)
    U, V, Om, m0 = random_inputs(g, p, "f64")
    ref, _, _ = gpu_run(g, p, "f64", U, V, Om, m0, [7], dt, kernel=1)
    for T in (1, 2, 3, 4):
        out, _, info = gpu_run(g, p, "f64", U, V, Om, m0, [7], dt, kernel=4, fuse_t=T)
        assert p1_density(out, ref) < 1e-13, (T, info)
    a, _, _ = gpu_run(g, p, "f64", U, V, Om, m0, [3, 4], dt, kernel=4, fuse_t=2)
    b, _, _ = gpu_run(g, p, "f64", U, V, Om, m0, [7], dt, kernel=4, fuse_t=2)
    assert p1_density(a, b) < 1e-13


def test_coef_moments_fused_equals_standalone():
    g = Grid(2, 3, 8, 12, 16, 16)
    p = Params()
    dt = _dt(g, p)
    U, V, Om, m0 = random_inputs(g, p, "f64")
    _, mf, _ = gpu_run(g, p, "f64", U, V, Om, m0, [4, 4], dt, kernel=4, fuse_t=2, fuse_mom=1)
    _, ms, _ = gpu_run(g, p, "f64", U, V, Om, m0, [4, 4], dt, kernel=4, fuse_t=2, fuse_mom=0)
    for (f1, t1), (f2, t2) in zip(mf, ms):
        assert np.allclose(f1, f2, rtol=0, atol=1e-14) and np.allclose(t1, t2, rtol=0, atol=1e-14)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_coef_stall_clamp_wide_ends_and_omega2(dtype):
    g = Grid(2, 2, 8, 9, 16, 16)
    p = Params(k_spring=200.0, n_end_cells=2, end_detach_mult=3.0)
    check_parity(g, p, dtype, [6], 0.25 * _dt(g, p, 2.0), omega_max=2.0, kernel=4, fuse_t=3)


def test_coef_zero_rates_and_zero_speed():
    """Degenerate parameters: no source, no walking (v0 = 0), no springs -- the coefficient folding must not
    divide by or depend on any of them."""
    g = Grid(1, 2, 8, 8, 16, 16)
    p = Params(k_on=0.0, v0=0.0, k_spring=0.0)
    check_parity(g, p, "f64", [5], _dt(g, Params()), kernel=4, fuse_t=2)


def test_coef_dirty_masked_input_is_dropped():
    g = Grid(1, 2, 4, 6, 16, 16)
    p = Params()
    dt = _dt(g, p)
    U, V, Om, m0 = random_inputs(g, p, "f64")
    m0 = m0.copy(); m0[:, :, ~mi.inside_mask(16, 16)] = 3.0
    out, _, _ = gpu_run(g, p, "f64", U, V, Om, m0, [2], dt, kernel=4, fuse_t=2)
    ref, _ = oracle_run(g, p, U, V, Om, m0, [2], dt)
    assert p1_density(out, ref) < TOL["f64"]


# ------------------------------------------------------------------ upwind-sparse tensor-memory kernel (mm_tm.cuh)
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("T", [1, 2, 3, 4, 5, 6, 7, 9, 10, 12])
@pytest.mark.parametrize("nxi", [16, 8])
def test_tm_kernel_parity(dtype, T, nxi):
    # Ns=7: ragged last chunk; 700 configurations: several per warp; odd and even depths (the level loop is rolled by two)
    g = Grid(5, 7, 20, 7, nxi, nxi)
    p = Params()
    e, info = check_parity(g, p, dtype, [2 * T + 3, T] if T > 4 else [5, 3], _dt(g, p), kernel=5, fuse_t=T)
    assert info["kernel"].startswith("tm<"), info


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_tm_every_upwind_variant(dtype):
    """The 9 straight-line variants of the level loop: per configuration (U, V) is chosen so that the xi (eta) face
    velocities are all positive, all negative or of mixed sign over the whole plane; Omega = 0 keeps the choice the
    same on every plane, Omega != 0 lets it change from plane to plane."""
    g = Grid(6, 6, 8, 9, 16, 16)
    p = Params()
    dt = 0.12 * _dt(g, p)
    U, V, Om, m0 = random_inputs(g, p, dtype)
    sel = np.arange(g.nc)
    big = np.array([-2.5, 0.0, 2.5])
    U = np.where((sel % 3) == 1, U, big[sel % 3]).astype(U.dtype)
    V = np.where(((sel // 3) % 3) == 1, V, big[(sel // 3) % 3]).astype(V.dtype)
    Om = np.where((sel // 9) % 2 == 0, 0.0, Om).astype(Om.dtype)
    out, moms, info = gpu_run(g, p, dtype, U, V, Om, m0, [6, 5], dt, kernel=5, fuse_t=6)
    ref, om = oracle_run(g, p, U, V, Om, m0, [6, 5], dt)
    assert info["kernel"].startswith("tm<"), info
    assert p1_density(out, ref) <= TOL[dtype]
    from util import p2_moments
    for (f, t), r in zip(moms, om):
        ef, et = p2_moments(f, t, r)
        assert ef <= TOL[dtype] and et <= TOL[dtype]
    # and the skipping is exact: the coefficient-form kernel, which multiplies by the zeros, agrees to rounding
    out4, _, _ = gpu_run(g, p, dtype, U, V, Om, m0, [6, 5], dt, kernel=4, fuse_t=6)
    assert p1_density(out, out4) <= (1e-13 if dtype == "f64" else 5e-5)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_tm_many_configs_per_warp(dtype):
    g = Grid(16, 16, 16, 6, 8, 8)   # 4096 configs of 384 cells
    p = Params()
    check_parity(g, p, dtype, [4], _dt(g, p), kernel=5, fuse_t=2)
    g = Grid(16, 16, 24, 5, 16, 16)   # 6144 configurations: more than the 2368 resident warps of the fp32 launch
    check_parity(g, p, dtype, [7], _dt(g, p), kernel=5, fuse_t=7)


def test_tm_equals_generic_and_fusion_invariance():
    g = Grid(3, 3, 8, 10, 16, 16)
    p = Params()
    dt = _dt(g, p)
    U, V, Om, m0 = random_inputs(g, p, "f64")
    ref, _, _ = gpu_run(g, p, "f64", U, V, Om, m0, [7], dt, kernel=1)
    for T in (1, 2, 3, 4, 7):
        out, _, info = gpu_run(g, p, "f64", U, V, Om, m0, [7], dt, kernel=5, fuse_t=T)
        assert p1_density(out, ref) < 1e-13, (T, info)
    a, _, _ = gpu_run(g, p, "f64", U, V, Om, m0, [3, 4], dt, kernel=5, fuse_t=2)
    b, _, _ = gpu_run(g, p, "f64", U, V, Om, m0, [7], dt, kernel=5, fuse_t=2)
    assert p1_density(a, b) < 1e-13


def test_tm_moments_fused_equals_standalone():
    g = Grid(2, 3, 8, 12, 16, 16)
    p = Params()
    dt = _dt(g, p)
    U, V, Om, m0 = random_inputs(g, p, "f64")
    _, mf, _ = gpu_run(g, p, "f64", U, V, Om, m0, [4, 4], dt, kernel=5, fuse_t=2, fuse_mom=1)
    _, ms, _ = gpu_run(g, p, "f64", U, V, Om, m0, [4, 4], dt, kernel=5, fuse_t=2, fuse_mom=0)
    for (f1, t1), (f2, t2) in zip(mf, ms):
        assert np.allclose(f1, f2, rtol=0, atol=1e-14) and np.allclose(t1, t2, rtol=0, atol=1e-14)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_tm_stall_clamp_wide_ends_and_omega2(dtype):
    g = Grid(2, 2, 8, 9, 16, 16)
    p = Params(k_spring=200.0, n_end_cells=2, end_detach_mult=3.0)
    check_parity(g, p, dtype, [6], 0.25 * _dt(g, p, 2.0), omega_max=2.0, kernel=5, fuse_t=3)


def test_tm_zero_rates_and_zero_speed():
    g = Grid(1, 2, 8, 8, 16, 16)
    p = Params(k_on=0.0, v0=0.0, k_spring=0.0)
    check_parity(g, p, "f64", [5], _dt(g, Params()), kernel=5, fuse_t=2)


def test_tm_dirty_masked_input_is_dropped():
    g = Grid(1, 2, 4, 6, 16, 16)
    p = Params()
    dt = _dt(g, p)
    U, V, Om, m0 = random_inputs(g, p, "f64")
    m0 = m0.copy(); m0[:, :, ~mi.inside_mask(16, 16)] = 3.0
    out, _, _ = gpu_run(g, p, "f64", U, V, Om, m0, [2], dt, kernel=5, fuse_t=2)
    ref, _ = oracle_run(g, p, U, V, Om, m0, [2], dt)
    assert p1_density(out, ref) < TOL["f64"]


def test_two_contexts_back_to_back_share_no_launch_state():
    """Launch shapes are cached per context (no process-wide statics): contexts of different dtype and offset plane,
    alive at the same time and used alternately, each run their own kernels."""
    from paper_1908_04279_b200 import MM
    ga, gb = Grid(2, 2, 8, 6, 16, 16), Grid(3, 2, 8, 5, 8, 8)
    p = Params()
    runs = []
    for g, dtype in ((ga, "f32"), (gb, "f64")):
        U, V, Om, m0 = random_inputs(g, p, dtype)
        mm = MM(g, p, dtype)
        mm.set_density(m0); mm.set_filament_velocity(U, V, Om)
        runs.append((g, dtype, mm, U, V, Om, m0))
    for rep in range(2):
        for g, dtype, mm, *_ in runs:
            mm.substep(3, _dt(g, p))
    for g, dtype, mm, U, V, Om, m0 in runs:
        from util import NPDT
        out = np.empty((g.nc, g.ns, g.nxi, g.neta), NPDT[dtype])
        mm.get_density(out)
        mm.destroy()
        ref, _ = oracle_run(g, p, U, V, Om, m0, [6], _dt(g, p))
        assert p1_density(out, ref) <= TOL[dtype]


# ------------------------------------------------------------------ in-place passes / single-buffer contexts
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("mode", ["option", "single"])
def test_inplace_passes_match_the_oracle(dtype, mode):
    """MM_OPT_INPLACE and a context created with ONE density buffer: Euler (T = 3, ragged Ns), RK2 + Superbee and the
    local step all update the buffer in place and still match the oracle; the second buffer is never touched."""
    import torch
    from paper_1908_04279_b200 import MM, binding as b
    from util import NPDT, TOL, p2_moments
    g = Grid(5, 7, 20, 7, 16, 16)
    npdt = NPDT[dtype]
    tdt = torch.float64 if dtype == "f64" else torch.float32
    for flags, what in ((0, "euler"), (mi.FLAG_RK2_SUPERBEE, "rk2"), (0, "local")):
        p = Params(flags=flags)
        dt = _dt(g, p)
        U, V, Om, m0 = random_inputs(g, p, dtype)
        b0 = torch.empty(g.cells, dtype=tdt, device="cuda")
        b1 = torch.full((g.cells,), 777.0, dtype=tdt, device="cuda") if mode == "option" else None
        mm = MM(g, p, dtype, b0, b1)
        if mode == "option":
            mm.set_option(b.MM_OPT_INPLACE, 1)
        assert mm.get_option(b.MM_OPT_INPLACE) == 1
        mm.set_option(b.MM_OPT_FUSE_T, 3)
        mm.set_density(np.ascontiguousarray(m0, npdt))
        mm.set_filament_velocity(U, V, Om)
        if what == "local":
            mm.advance_local(6.5 * dt, 0.4)
            ref, _ = orc.advance_local(g, p, U, V, Om, m0, 6.5 * dt, 0.4)
        else:
            mm.substep(7, dt)
            ref = orc.run(g, p, U, V, Om, m0, 7, dt)
        f, t = np.empty((g.nc, 2)), np.empty(g.nc)
        mm.moments(f, t)
        out = np.empty((g.nc, g.ns, g.nxi, g.neta), npdt)
        mm.get_density(out)
        name = mm.kernel_name
        mm.destroy()
        assert p1_density(out, ref) <= TOL[dtype], (what, name)
        ef, et = p2_moments(f, t, orc.moments(g, p, ref))
        assert ef <= TOL[dtype] and et <= TOL[dtype], (what, name)
        assert np.array_equal(out.reshape(-1), b0.cpu().numpy()), "the result lives in the one buffer"
        if b1 is not None:
            assert bool((b1 == 777.0).all()), "the second buffer must not be touched"


def test_single_buffer_context_refuses_two_buffer_kernels():
    import torch
    from paper_1908_04279_b200 import MM, MMError, binding as b
    g = Grid(1, 2, 4, 5, 3, 7)            # odd offset plane: generic kernels only
    p = Params()
    U, V, Om, m0 = random_inputs(g, p, "f64")
    mm = MM(g, p, "f64", torch.empty(g.cells, dtype=torch.float64, device="cuda"), None)
    mm.set_density(m0); mm.set_filament_velocity(U, V, Om)
    with pytest.raises(MMError):
        mm.substep(1, _dt(g, p))
    with pytest.raises(MMError):
        mm.advance_local(0.01, 0.4)
    with pytest.raises(MMError):
        mm.set_option(b.MM_OPT_INPLACE, 0)
    mm.destroy()
