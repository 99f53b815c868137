"""GPU parity of the free-motor coupling (mm_update_free_motors + coupled source) against the
oracle: coarse bound density, cap rescale, free density, and substeps driven by k_on M_f(r0)."""
import dataclasses

import numpy as np
import pytest

import mm_inputs as mi
from mm_inputs import Grid, Params
from oracle import mm_oracle as orc
from util import NPDT, TOL, p1_density, random_inputs

pytestmark = pytest.mark.gpu
RNG = np.random.default_rng(2024)


def gpu_coupled(g, p, dtype, U, V, Om, m0, psi, n_sub, dt, kernel=0):
    from paper_1908_04279_b200 import MM, binding as b
    mm = MM(g, p, dtype)
    mm.set_option(b.MM_OPT_KERNEL, kernel)
    mm.set_density(np.ascontiguousarray(m0, NPDT[dtype]))
    mm.set_filament_velocity(*(np.ascontiguousarray(x, NPDT[dtype]) for x in (U, V, Om)))
    mm.set_psi(np.ascontiguousarray(psi, np.float64))
    Mbc, Mf = np.empty((g.nx, g.ny)), np.empty((g.nx, g.ny))
    mm.update_free_motors(Mbc, Mf)
    assert mm.get_option(b.MM_OPT_FREE_COUPLING) == 1
    capped = np.empty((g.nc, g.ns, g.nxi, g.neta), NPDT[dtype])
    mm.get_density(capped)
    mm.substep(n_sub, dt)
    out = np.empty_like(capped)
    mm.get_density(out)
    name = mm.kernel_name
    mm.destroy()
    return Mbc, Mf, capped, out, name


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("flags", [0, mi.FLAG_RK2_SUPERBEE])
@pytest.mark.parametrize("kernel", [0, 1, 4, 5])
@pytest.mark.parametrize("shape", [(6, 6, 8, 7, 16, 16), (5, 4, 4, 5, 6, 6), (8, 8, 4, 6, 8, 8)])
def test_free_motor_coupling_parity(dtype, flags, shape, kernel):
    if kernel in (4, 5) and (flags or shape[4] not in (8, 16)):
        pytest.skip("kernels 4 and 5 are forced only where the coefficient-form kernels apply")
    g = Grid(*shape)
    big = Params(flags=flags, m_free=1e9)
    U, V, Om, m0 = random_inputs(g, big, dtype)
    psi = RNG.random(g.nc) * 30.0
    _, raw, _ = orc.free_motors(g, big, m0, psi)
    p = dataclasses.replace(big, m_free=float(np.median(raw)))      # half of the nodes get capped
    dt = mi.benchmark_dt(g, p, 1.0)
    Mbc, Mf, capped, out, name = gpu_coupled(g, p, dtype, U, V, Om, m0, psi, 7, dt, kernel)
    m_ref, Mbc_ref, Mf_ref = orc.free_motors(g, p, m0, psi)
    tol = TOL[dtype]
    assert np.max(np.abs(Mbc - Mbc_ref)) / p.m_free <= tol and np.max(np.abs(Mf - Mf_ref)) / p.m_free <= tol
    assert (Mf >= 0).all() and (Mbc <= p.m_free).all()
    assert p1_density(capped, m_ref) <= tol
    # substeps with the coupled source, from the oracle's own capped state and table
    ref = orc.run_coupled(g, p, U, V, Om, m_ref, 7, dt, Mf_ref)
    assert p1_density(out, ref) <= tol, name
    fast = kernel != 1 and flags == 0 and shape[4] in (8, 16)
    fam = {0: ("tm_mf<", "coef_mf<"), 4: ("coef_mf<",), 5: ("tm_mf<",)}   # auto picks by pass depth
    assert name.startswith(fam[kernel] if fast else ("rk2_generic<" if flags else "generic<")), name


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_free_motor_deposits_of_every_magnitude(dtype):
    """The fixed-point deposit of the vectorised pass has two routes: |deposit| < 2^19 units of the table (the limbs come
    from round-down additions) and the rest (conversions, `fx_deposit`).  A density whose cells span 7 decades, with
    M_total chosen so that the largest node sum is 2^29 units, sends cells down both."""
    g = Grid(6, 6, 8, 7, 16, 16)
    big = Params(m_free=1e30)
    U, V, Om, m0 = random_inputs(g, big, dtype)
    rng = np.random.default_rng(31)
    m0 = np.ascontiguousarray(m0 * np.where(rng.random(m0.shape) < 0.003, 1e7, 1.0), NPDT[dtype])
    psi = rng.random(g.nc) * 30.0
    _, raw, _ = orc.free_motors(g, big, m0, psi)
    p = dataclasses.replace(big, m_free=float(raw.max()) / 2.0 ** 29)
    Mbc, Mf, capped, _, _ = gpu_coupled(g, p, dtype, U, V, Om, m0, psi, 0, 1e-3)
    m_ref, Mbc_ref, Mf_ref = orc.free_motors(g, p, m0, psi)
    tol = TOL[dtype]
    assert np.max(np.abs(Mbc - Mbc_ref)) / p.m_free <= tol and np.max(np.abs(Mf - Mf_ref)) / p.m_free <= tol
    assert p1_density(capped, m_ref) <= tol
    # the cap factor of a node is M_total / (its raw sum): the rescaled cells carry the sums to rounding
    nz = np.abs(m_ref) > 0
    assert np.max(np.abs(capped[nz] / m_ref[nz] - 1.0)) <= (1e-11 if dtype == "f64" else 3e-7)


def test_free_motor_option_and_errors():
    from paper_1908_04279_b200 import MM, MMError, binding as b
    g = Grid(4, 4, 4, 6, 8, 8)
    p = Params()
    U, V, Om, m0 = random_inputs(g, p, "f64")
    mm = MM(g, p, "f64")
    mm.set_density(m0); mm.set_filament_velocity(U, V, Om)
    with pytest.raises(MMError):
        mm.update_free_motors()                       # psi missing
    with pytest.raises(MMError):
        mm.set_option(b.MM_OPT_FREE_COUPLING, 1)     # no table yet
    mm.set_psi(np.zeros(g.nc))                        # nothing bound counts: M_f = M_total everywhere
    Mf = np.empty((4, 4))
    mm.update_free_motors(None, Mf)
    assert np.array_equal(Mf, np.full((4, 4), p.m_free))
    dt = mi.benchmark_dt(g, p, 1.0)
    mm.substep(3, dt)
    a = np.empty_like(m0); mm.get_density(a)
    assert p1_density(a, orc.run(g, p, U, V, Om, m0, 3, dt)) < 1e-12      # uniform table == constant source
    assert mm.kernel_name.startswith(("tm_mf<", "coef_mf<"))
    mm.set_option(b.MM_OPT_KERNEL, 4)
    with pytest.raises(MMError):
        mm.advance_local(dt, 0.4)                     # coupled local steps: kernels 0 / 5 only
    mm.set_option(b.MM_OPT_KERNEL, 0)
    with pytest.raises(MMError):
        mm.set_option(b.MM_OPT_FREE_REFRESH, -1)
    mm.set_option(b.MM_OPT_FREE_COUPLING, 0)          # back to the fast path
    mm.substep(1, dt)
    assert mm.kernel_name.startswith(("tm<", "coef<"))
    mm.destroy()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_full_microscale_step_against_the_oracle(dtype):
    """Alg. 2 on this path, two macro steps in a row: free-motor update (coarse density, cap, M_f), substeps with the
    coupled source, moments, force spreading -- every output of every stage against the oracle run the same way."""
    from paper_1908_04279_b200 import MM
    from util import p2_moments
    g = Grid(8, 6, 8, 9, 16, 16)
    big = Params(m_free=1e9)
    U, V, Om, m0 = random_inputs(g, big, dtype)
    psi = RNG.random(g.nc) * 25.0
    _, raw, _ = orc.free_motors(g, big, m0, psi)
    p = dataclasses.replace(big, m_free=float(np.quantile(raw, 0.7)))
    dt = mi.benchmark_dt(g, p, 1.0)
    tol = TOL[dtype]
    mm = MM(g, p, dtype)
    mm.set_density(np.ascontiguousarray(m0, NPDT[dtype]))
    mm.set_psi(psi)
    ref = np.asarray(m0, np.float64)
    for step in range(2):
        Us, Vs, Os = ((1.0 - 0.3 * step) * x for x in (U, V, Om))     # new macroscale velocities every step
        mm.set_filament_velocity(*(np.ascontiguousarray(x, NPDT[dtype]) for x in (Us, Vs, Os)))
        Mbc, Mf = np.empty((g.nx, g.ny)), np.empty((g.nx, g.ny))
        mm.update_free_motors(Mbc, Mf)
        mm.substep(6, dt)
        f, t = np.empty((g.nc, 2)), np.empty(g.nc)
        mm.moments(f, t)
        F2 = np.empty((g.nx, g.ny, 2))
        mm.spread_force(F2)
        out = np.empty((g.nc, g.ns, g.nxi, g.neta), NPDT[dtype])
        mm.get_density(out)
        # oracle, same sequence (fp32: from the velocities as stored)
        Uo, Vo, Oo = (np.asarray(np.asarray(x, NPDT[dtype]), np.float64) for x in (Us, Vs, Os))
        ref, Mbc_o, Mf_o = orc.free_motors(g, p, ref, psi)
        ref = orc.run_coupled(g, p, Uo, Vo, Oo, ref, 6, dt, Mf_o)
        assert np.max(np.abs(Mbc - Mbc_o)) / p.m_free <= tol and np.max(np.abs(Mf - Mf_o)) / p.m_free <= tol, step
        assert p1_density(out, ref) <= tol, step
        ef, et = p2_moments(f, t, orc.moments(g, p, ref))
        assert ef <= tol and et <= tol, step
        F2_o = orc.spread_force(g, p, ref, psi)
        assert np.max(np.abs(F2 - F2_o)) / np.max(np.abs(F2_o)) <= tol, step
    assert mm.kernel_name.startswith(("tm_mf<", "coef_mf<"))
    mm.destroy()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("flags,kernel,shape", [(0, 0, (6, 6, 8, 7, 16, 16)), (0, 5, (8, 8, 4, 6, 8, 8)), (0, 1, (5, 4, 4, 5, 6, 6)),
                                                (mi.FLAG_RK2_SUPERBEE, 0, (6, 6, 8, 7, 16, 16))])
@pytest.mark.parametrize("refresh", [1, 3])
def test_alg2_cadence_refresh_inside_substep(dtype, flags, kernel, shape, refresh):
    """MM_OPT_FREE_REFRESH = k: mm_substep redoes the coarse reduction, the cap and M_f before every k-th substep
    (k = 1: Alg. 2 l.14-20 inside the inner loop) -- against the oracle's mmo_run_alg2."""
    from paper_1908_04279_b200 import MM, binding as b
    from util import p2_moments
    g = Grid(*shape)
    big = Params(flags=flags, m_free=1e9)
    U, V, Om, m0 = random_inputs(g, big, dtype)
    psi = RNG.random(g.nc) * 30.0
    _, raw, _ = orc.free_motors(g, big, m0, psi)
    p = dataclasses.replace(big, m_free=float(np.quantile(raw, 0.6)))
    dt = mi.benchmark_dt(g, p, 1.0)
    mm = MM(g, p, dtype)
    mm.set_option(b.MM_OPT_KERNEL, kernel)
    mm.set_density(np.ascontiguousarray(m0, NPDT[dtype]))
    mm.set_filament_velocity(*(np.ascontiguousarray(x, NPDT[dtype]) for x in (U, V, Om)))
    mm.set_psi(psi)
    mm.update_free_motors()                      # switches the coupled source on (its table is replaced at substep 0)
    mm.set_option(b.MM_OPT_FREE_REFRESH, refresh)
    assert mm.get_option(b.MM_OPT_FREE_REFRESH) == refresh
    mm.substep(7, dt)
    f, t = np.empty((g.nc, 2)), np.empty(g.nc)
    mm.moments(f, t)
    out = np.empty((g.nc, g.ns, g.nxi, g.neta), NPDT[dtype])
    mm.get_density(out)
    name = mm.kernel_name
    mm.destroy()
    ref, _, _ = orc.run_alg2(g, p, U, V, Om, m0, psi, 7, dt, refresh)
    tol = TOL[dtype]
    assert p1_density(out, ref) <= tol, name
    ef, et = p2_moments(f, t, orc.moments(g, p, ref))
    assert ef <= tol and et <= tol, name
