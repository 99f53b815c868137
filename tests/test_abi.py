"""C-ABI: exported symbols, argument validation, error behaviour (CPU part needs no GPU)."""
import ctypes
import dataclasses
import os
import re

import numpy as np
import pytest

import mm_inputs as mi
from mm_inputs import Grid, Params
from paper_1908_04279_b200 import binding as b

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "mm.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(mm_[a-z_]+)\s*\(", hdr))
    assert declared == set(b.EXPORTS), declared ^ set(b.EXPORTS)
    L = b.lib()
    for name in declared:
        assert hasattr(L, name), name
    # ... and nothing else: launchers and kernel stubs stay local (csrc/libmm.map)
    import subprocess
    from paper_1908_04279_b200 import build as mm_build
    out = subprocess.run(["nm", "-D", "--defined-only", mm_build.SO], capture_output=True, text=True).stdout
    exported = {l.split()[-1] for l in out.splitlines() if len(l.split()) == 3 and l.split()[1] in "TDBR"}
    assert exported == declared, exported ^ declared


def test_struct_layout_matches_header():
    assert ctypes.sizeof(b.mm_grid) == 24
    assert ctypes.sizeof(b.mm_params) == 11 * 8 + 8


@pytest.mark.parametrize("bad", [
    dict(grid=Grid(0, 1, 1, 4, 3, 3)), dict(grid=Grid(1, 1, 1, 4, 3, 0)), dict(grid=Grid(1, 1, 1, 0, 3, 3)),
    dict(params=Params(R=0.0)), dict(params=Params(f_stall=0.0)), dict(params=Params(f_detach=-1.0)),
    dict(params=Params(k_on=-1.0)), dict(params=Params(v0=float("nan"))), dict(params=Params(n_end_cells=3)),
    dict(params=Params(s_lo=0.5, s_hi=0.5)), dict(params=Params(flags=64)), dict(params=Params(k_off0=float("inf"))),
])
def test_create_rejects_invalid_arguments_before_touching_cuda(bad):
    grid = bad.get("grid", Grid(1, 1, 2, 4, 3, 3))
    params = bad.get("params", Params())
    with pytest.raises(b.MMError) as e:
        b.MM(grid, params, "f64", stream=0)
    assert e.value.status == b.MM_ERR_INVALID_ARG


def test_status_strings_and_null_handles():
    L = b.lib()
    assert L.mm_status_string(0) == b"MM_OK" and L.mm_status_string(-5) == b"MM_ERR_UNSTABLE"
    assert L.mm_destroy(None) == b.MM_OK            # NULL is a no-op
    assert L.mm_substep(None, 1, 0.1) == b.MM_ERR_INVALID_ARG
    assert L.mm_launch_count(None) == 0


def test_no_cpu_fallback_without_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(b.MMError) as e:
        b.MM(Grid(1, 1, 2, 4, 3, 3), Params(), "f64", stream=0)
    assert e.value.status == b.MM_ERR_CUDA


# ---------------------------------------------------------------------------------- GPU part
@pytest.mark.gpu
def test_state_and_argument_errors_on_gpu():
    import torch
    g = Grid(1, 1, 2, 4, 3, 3)
    mm = b.MM(g, Params(), "f64")
    with pytest.raises(b.MMError) as e:
        mm.substep(1, 0.01)
    assert e.value.status == b.MM_ERR_STATE
    out = np.empty(g.cells)
    with pytest.raises(b.MMError) as e:
        mm.get_density(out)
    assert e.value.status == b.MM_ERR_STATE
    mm.set_density_range(0, 1, np.zeros(g.inner))
    with pytest.raises(b.MMError):
        mm.get_density(out)                      # only half of the configurations uploaded
    mm.set_density_range(1, 1, np.ones(g.inner))
    z = np.zeros(g.nc)
    mm.set_filament_velocity(z, z, z)
    mm.substep(0, -1.0)                          # n_sub == 0: no-op, dt not inspected
    for bad_dt in (0.0, -1.0, float("nan")):
        with pytest.raises(b.MMError) as e:
            mm.substep(1, bad_dt)
        assert e.value.status == b.MM_ERR_INVALID_ARG
    with pytest.raises(b.MMError):
        mm.substep(-1, 0.1)
    with pytest.raises(b.MMError):
        mm.set_density_range(1, 2, np.zeros(2 * g.inner))
    with pytest.raises(b.MMError):
        mm.set_option(b.MM_OPT_FUSE_T, b.MM_MAX_FUSE_T + 1)
    mm.set_option(b.MM_OPT_KERNEL, 2)
    with pytest.raises(b.MMError) as e:          # 3x3 offsets: streamed kernel unsupported -> loud error
        mm.substep(1, 0.01)
    assert e.value.status == b.MM_ERR_INVALID_ARG
    mm.set_option(b.MM_OPT_KERNEL, 0)
    mm.substep(2, 0.01)
    mm.get_density(out)
    assert np.isfinite(out).all()
    mm.destroy(); mm.destroy()                   # double destroy through the binding is safe


@pytest.mark.gpu
def test_check_dt_flag():
    g = Grid(1, 1, 4, 8, 8, 8)
    p = Params(flags=mi.FLAG_CHECK_DT)
    st = mi.Stream(g, p.R); U, V, Om = st.velocities(); m0 = st.density(g.nc)
    mm = b.MM(g, p, "f64")
    mm.set_density(m0); mm.set_filament_velocity(U, V, Om)
    mm.substep(2, mi.benchmark_dt(g, p, 1.0))    # CFL 0.4: fine
    with pytest.raises(b.MMError) as e:
        mm.substep(1, 10 * mi.benchmark_dt(g, p, 1.0))
    assert e.value.status == b.MM_ERR_UNSTABLE
    mm.destroy()


@pytest.mark.gpu
def test_fma_rate_probes():
    """mm_measure_fma_rate: the register file delivers two 32-bit operands per cycle and scheduler, so FMAs with three
    fresh operands run at about 2/3 of the unit's rate; fresh_operands = 1 is mm_measure_fma_peak."""
    for dtype, lo, hi in (("f32", 0.55, 0.80), ("f64", 0.55, 0.90)):
        peak = b.measure_fma_peak(dtype)
        one = b.measure_fma_rate(dtype, 1)
        three = b.measure_fma_rate(dtype, 3)
        assert abs(one / peak - 1.0) < 0.05
        assert lo < three / peak < hi, (dtype, peak, three)
    with pytest.raises(b.MMError):
        b.measure_fma_rate("f32", 2)
