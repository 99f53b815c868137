"""GPU parity of the local adaptive time step (mm_advance_local) against the oracle:
the integer step counts n_c bit-exactly, the rate bound lambda_c to rounding, the density and moments at the
usual tolerances."""
import numpy as np
import pytest

import mm_inputs as mi
from mm_inputs import Grid, Params
from oracle import mm_oracle as orc
from util import NPDT, TOL, p1_density, p2_moments, random_inputs

pytestmark = pytest.mark.gpu


def run_local(g, p, dtype, U, V, Om, m0, dt, cfl, kernel=0):
    import torch
    from paper_1908_04279_b200 import MM, binding as b
    mm = MM(g, p, dtype)
    mm.set_option(b.MM_OPT_KERNEL, kernel)
    npdt = NPDT[dtype]
    mm.set_density(np.ascontiguousarray(m0, npdt))
    mm.set_filament_velocity(*(np.ascontiguousarray(x, npdt) for x in (U, V, Om)))
    mm.advance_local(dt, cfl)
    n, lam = np.empty(g.nc, np.int32), np.empty(g.nc)
    mm.local_steps(n, lam)
    f, t = np.empty((g.nc, 2)), np.empty(g.nc)
    mm.moments(f, t)
    out = np.empty((g.nc, g.ns, g.nxi, g.neta), npdt)
    mm.get_density(out)
    name = mm.kernel_name
    mm.destroy()
    return out, n, lam, f, t, name


def check_local(g, p, dtype, dt_mult, cfl=0.4, omega_max=1.0, kernel=0):
    U, V, Om, m0 = random_inputs(g, p, dtype, omega_max=omega_max)
    lam_o = orc.rate_bound(g, p, U, V, Om)          # from the velocities as stored (fp32 contexts: rounded, Q18)
    dt = dt_mult / lam_o.mean()
    out, n, lam, f, t, name = run_local(g, p, dtype, U, V, Om, m0, dt, cfl, kernel)
    ref, n_o = orc.advance_local(g, p, U, V, Om, m0, dt, cfl)
    assert np.max(np.abs(lam - lam_o) / lam_o) < 1e-14, name
    assert np.array_equal(n, n_o), name                                  # integer work: bit-exact
    tol = TOL[dtype]
    e1 = p1_density(out, ref)
    assert e1 <= tol, (e1, name)
    rm = orc.moments(g, p, ref)
    ef, et = p2_moments(f, t, rm)
    assert ef <= tol and et <= tol, (ef, et, name)
    return n, name


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("shape", [(2, 2, 4, 6, 5, 4), (1, 3, 5, 7, 16, 16), (3, 3, 8, 9, 8, 8)])
def test_local_generic_parity(dtype, shape):
    g = Grid(*shape)
    p = Params()
    n, name = check_local(g, p, dtype, 6.3, kernel=1)
    assert name.startswith("local_generic<") and len(set(n.tolist())) > 1


def test_local_single_step_and_wide_ends():
    g = Grid(1, 2, 8, 12, 8, 8)
    p = Params(k_spring=200.0, n_end_cells=3, end_detach_mult=4.0)
    n, _ = check_local(g, p, "f64", 0.2, kernel=1)
    assert (n == 1).all()
    check_local(g, p, "f64", 9.0, omega_max=2.0, kernel=1)


def test_local_errors():
    from paper_1908_04279_b200 import MM, MMError
    g = Grid(1, 1, 2, 4, 4, 4)
    mm = MM(g, Params(), "f64")
    with pytest.raises(MMError):
        mm.advance_local(0.1, 0.4)            # nothing set yet
    with pytest.raises(MMError):
        mm.local_steps(np.empty(g.nc, np.int32), None)
    mm.destroy()
    import torch
    one = torch.zeros(g.cells, dtype=torch.float64, device="cuda:0")
    mm = MM(g, Params(flags=mi.FLAG_RK2_SUPERBEE), "f64", buf0=one)      # single-buffer context
    U, V, Om, m0 = random_inputs(g, Params(), "f64")
    mm.set_density(m0); mm.set_filament_velocity(U, V, Om)
    with pytest.raises(MMError):
        mm.advance_local(0.1, 0.4)            # local RK2 steps need the second density buffer
    with pytest.raises(MMError):
        MM(g, Params(), "f64").advance_local(-1.0, 0.4)
    mm.destroy()


# ------------------------------------------------------------------ coefficient-form local-step kernel
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("nxi", [16, 8])
@pytest.mark.parametrize("dt_mult", [0.3, 2.9, 11.0])
def test_local_coef_parity(dtype, nxi, dt_mult):
    # 700 configurations, ragged Ns = 7; dt_mult 0.3: one step everywhere, 2.9: fewer than T levels in the only pass,
    # 11: several passes with configurations finishing in different passes (copy-through)
    g = Grid(5, 7, 20, 7, nxi, nxi)
    p = Params()
    n, name = check_local(g, p, dtype, dt_mult, omega_max=2.0)
    assert name.startswith("tm_local<"), name
    if dt_mult > 1:
        assert len(set(n.tolist())) > 1


def test_local_coef_equals_generic_and_moments_standalone():
    from paper_1908_04279_b200 import binding as b
    g = Grid(2, 3, 8, 12, 16, 16)
    p = Params(k_spring=120.0, n_end_cells=2, end_detach_mult=3.0)
    U, V, Om, m0 = random_inputs(g, p, "f64", omega_max=2.0)
    dt = 7.7 / orc.rate_bound(g, p, U, V, Om).mean()
    a = run_local(g, p, "f64", U, V, Om, m0, dt, 0.4, kernel=0)
    c = run_local(g, p, "f64", U, V, Om, m0, dt, 0.4, kernel=1)
    assert a[5].startswith("tm_local<") and c[5].startswith("local_generic<")
    assert np.array_equal(a[1], c[1]) and p1_density(a[0], c[0]) < 1e-12
    assert np.allclose(a[3], c[3], rtol=0, atol=1e-13) and np.allclose(a[4], c[4], rtol=0, atol=1e-13)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("nxi", [16, 8])
def test_local_steps_with_the_coupled_source(dtype, nxi):
    """Alg. 2 as one loop: local steps whose source is k_on M_f(r0) from the free-motor table (kernel 5, tm_mf_local)."""
    import dataclasses
    from paper_1908_04279_b200 import MM, binding as b
    from util import NPDT, TOL, p1_density, p2_moments
    g = Grid(5, 7, 12, 7, nxi, nxi)
    big = Params(m_free=1e9)
    U, V, Om, m0 = random_inputs(g, big, dtype, omega_max=2.0)
    rng = np.random.default_rng(5)
    psi = rng.random(g.nc) * 30.0
    _, raw, _ = orc.free_motors(g, big, m0, psi)
    p = dataclasses.replace(big, m_free=float(np.median(raw)))
    dt = 9.5 / orc.rate_bound(g, p, U, V, Om).mean()            # several passes at depth 4, one at the default depth
    for fuse_t in (4, None):
        mm = MM(g, p, dtype)
        if fuse_t:
            mm.set_option(b.MM_OPT_FUSE_T, fuse_t)
        mm.set_density(np.ascontiguousarray(m0, NPDT[dtype]))
        mm.set_filament_velocity(U, V, Om)
        mm.set_psi(psi)
        Mf = np.empty((g.nx, g.ny))
        mm.update_free_motors(None, Mf)
        mm.advance_local(dt, 0.4)
        n = np.empty(g.nc, np.int32)
        mm.local_steps(n, None)
        f, t = np.empty((g.nc, 2)), np.empty(g.nc)
        mm.moments(f, t)
        out = np.empty((g.nc, g.ns, g.nxi, g.neta), NPDT[dtype])
        mm.get_density(out)
        name = mm.kernel_name
        mm.destroy()
        capped, _, Mf_ref = orc.free_motors(g, p, m0, psi)
        ref, n_ref = orc.advance_local(g, p, U, V, Om, capped, dt, 0.4, Mf=Mf_ref)
        assert name.startswith("tm_mf_local<"), name
        assert np.array_equal(n, n_ref) and len(set(n.tolist())) > 1
        assert p1_density(out, ref) <= TOL[dtype], name
        ef, et = p2_moments(f, t, orc.moments(g, p, ref))
        assert ef <= TOL[dtype] and et <= TOL[dtype], name


# ------------------------------------------------------------------ local steps of the paper's own scheme (NEXT-3 x NEXT-1)
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("shape", [(2, 2, 4, 6, 5, 4), (2, 3, 6, 9, 16, 16)])
def test_local_rk2_parity(dtype, shape):
    """Alg. 2 l.5 (dt_c from the CFL bound) driving l.9-10 (RK2 + Superbee): every unit takes its own n_c two-stage steps."""
    g = Grid(*shape)
    p = Params(flags=mi.FLAG_RK2_SUPERBEE)
    n, name = check_local(g, p, dtype, 5.3, omega_max=2.0)
    assert name.startswith("rk2_local_generic<") and len(set(n.tolist())) > 1


def test_local_rk2_with_the_coupled_source():
    import dataclasses
    from paper_1908_04279_b200 import MM
    g = Grid(4, 5, 6, 7, 8, 8)
    big = Params(m_free=1e9, flags=mi.FLAG_RK2_SUPERBEE)
    U, V, Om, m0 = random_inputs(g, big, "f64", omega_max=2.0)
    psi = np.random.default_rng(6).random(g.nc) * 30.0
    _, raw, _ = orc.free_motors(g, big, m0, psi)
    p = dataclasses.replace(big, m_free=float(np.median(raw)))
    dt = 4.5 / orc.rate_bound(g, p, U, V, Om).mean()
    mm = MM(g, p, "f64")
    mm.set_density(m0); mm.set_filament_velocity(U, V, Om); mm.set_psi(psi)
    mm.update_free_motors(None, None)
    mm.advance_local(dt, 0.4)
    n = np.empty(g.nc, np.int32)
    mm.local_steps(n, None)
    f, t = np.empty((g.nc, 2)), np.empty(g.nc)
    mm.moments(f, t)
    out = np.empty_like(m0)
    mm.get_density(out)
    mm.destroy()
    capped, _, Mf_ref = orc.free_motors(g, p, m0, psi)
    ref, n_ref = orc.advance_local(g, p, U, V, Om, capped, dt, 0.4, Mf=Mf_ref)
    assert np.array_equal(n, n_ref) and len(set(n.tolist())) > 1
    assert p1_density(out, ref) <= TOL["f64"]
    ef, et = p2_moments(f, t, orc.moments(g, p, ref))
    assert ef <= TOL["f64"] and et <= TOL["f64"]
