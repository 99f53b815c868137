"""Pins of the CPU oracle against what the equations fix.

PAPER.md prints no numerical value for this path, so every pin is a closed form, an invariant, a
special case or a brute-force sum -- none re-uses the oracle's own code.  Each test names the steps
(S1-S9) a mistake in which would make it fail.
"""
import dataclasses
import math
from fractions import Fraction

import numpy as np
import pytest

import mm_inputs as mi
from mm_inputs import Grid, Params
from oracle import mm_oracle as orc
from conftest import read_golden

RNG = np.random.default_rng(12345)


def geom(g, p):
    ds = (p.s_hi - p.s_lo) / g.ns
    dxi, deta = 2 * p.R / g.nxi, 2 * p.R / g.neta
    s = p.s_lo + (np.arange(g.ns) + 0.5) * ds
    xi = -p.R + (np.arange(g.nxi) + 0.5) * dxi
    eta = -p.R + (np.arange(g.neta) + 0.5) * deta
    return ds, dxi, deta, s, xi, eta


def rand_state(g, n=None, mask=True):
    n = g.nc if n is None else n
    m = RNG.random((n, g.ns, g.nxi, g.neta))
    if mask:
        m *= mi.inside_mask(g.nxi, g.neta)[None, None]
    return m, RNG.random(n) - 0.5, RNG.random(n) - 0.5, 2 * RNG.random(n) - 1


# ---------------------------------------------------------------- C1 mass conservation
def test_c1_mass_conserved_periodic_all_directions():
    """S4, S5, S7: conservative pairing of faces in s, xi and eta (incl. the ONE wrapped face)."""
    g = Grid(2, 2, 4, 8, 5, 6)
    p = Params(k_on=0.0, k_off0=0.0, flags=mi.FLAG_S_PERIODIC | mi.FLAG_OFFSET_PERIODIC_NOMASK)
    m, U, V, Om = rand_state(g, mask=False)
    dt = 0.5 * mi.benchmark_dt(g, p, 1.0)
    out = orc.run(g, p, U, V, Om, m, 100, dt)
    m0, m1 = m.sum(axis=(1, 2, 3)), out.sum(axis=(1, 2, 3))
    assert np.max(np.abs(m1 - m0) / m0) < 1e-13
    assert not np.allclose(out, m)  # something actually moved


def test_c1_variant_no_offset_flag():
    """k=0, U=-cos, V=-sin, Omega=0  =>  A_xi = A_eta = 0 exactly; periodic s only."""
    g = Grid(1, 1, 8, 16, 8, 8)
    p = Params(k_spring=0.0, k_on=0.0, k_off0=0.0, flags=mi.FLAG_S_PERIODIC)
    m, _, _, _ = rand_state(g)
    th = 2 * np.pi * np.arange(g.ntheta) / g.ntheta
    out = orc.run(g, p, -np.cos(th), -np.sin(th), np.zeros(g.nc), m, 100, 0.3 / g.ns)
    m0, m1 = m.sum(axis=(1, 2, 3)), out.sum(axis=(1, 2, 3))
    # the relative velocity cancels only to trig rounding (|A| ~ 1e-16): leak ~ n*dt*1e-16/dxi
    assert np.max(np.abs(m1 - m0) / m0) < 1e-12


# ---------------------------------------------------------------- C1b discrete mass budget
def test_c1b_mass_budget_default_bcs():
    """S5 boundary faces, S6: interior fluxes telescope; only boundary outflow and reactions change mass.
    3x3 offset grid: all cells inside the disc, so masking removes nothing."""
    g = Grid(1, 2, 4, 6, 3, 3)
    p = Params()
    m, U, V, Om = rand_state(g)
    dt = 0.4 * mi.benchmark_dt(g, p, 1.0)
    out = orc.run(g, p, U, V, Om, m, 1, dt)
    ds, dxi, deta, s, xi, eta = geom(g, p)
    dV = ds * dxi * deta
    for c in range(g.nc):
        th = 2 * np.pi * (c % g.ntheta) / g.ntheta
        ct, st_ = math.cos(th), math.sin(th)
        w = lambda x, e: p.v0 * np.maximum(0.0, 1 - p.k_spring * (x * ct + e * st_) / p.f_stall)
        XI, ETA = np.meshgrid(xi, eta, indexing="ij")
        # outflow through s = s_hi
        out_s = dxi * deta * np.sum(w(XI, ETA) * m[c, -1])
        # xi boundary faces at -R and +R (ghost = 0 => only outward-directed part carries mass)
        S, E = np.meshgrid(s, eta, indexing="ij")
        A_hi = U[c] + w(p.R, E) * ct - S * Om[c] * st_
        A_lo = U[c] + w(-p.R, E) * ct - S * Om[c] * st_
        out_xi = ds * deta * np.sum(np.maximum(A_hi, 0) * m[c, :, -1, :] - np.minimum(A_lo, 0) * m[c, :, 0, :])
        S, X = np.meshgrid(s, xi, indexing="ij")
        B_hi = V[c] + w(X, p.R) * st_ + S * Om[c] * ct
        B_lo = V[c] + w(X, -p.R) * st_ + S * Om[c] * ct
        out_eta = ds * dxi * np.sum(np.maximum(B_hi, 0) * m[c, :, :, -1] - np.minimum(B_lo, 0) * m[c, :, :, 0])
        r = np.sqrt(XI ** 2 + ETA ** 2)
        Ej = np.ones(g.ns); Ej[0] = Ej[-1] = p.end_detach_mult
        kappa = p.k_off0 * np.exp(p.k_spring * r / p.f_detach)[None] * Ej[:, None, None]
        react = dV * np.sum(p.k_on * p.m_free - kappa * m[c])
        expect = dV * m[c].sum() - dt * (out_s + out_xi + out_eta) + dt * react
        assert dV * out[c].sum() == pytest.approx(expect, rel=1e-13)


# ---------------------------------------------------------------- C2 pure detachment
def test_c2_pure_detachment_closed_form():
    """S6, S7: Bell factor, end multiplier on both end cells, forward Euler decay."""
    gd = read_golden("c2_pure_detachment.txt")
    g = Grid(1, 1, 3, 64, 16, 16)
    p = Params(v0=0.0, k_on=0.0)
    m, _, _, _ = rand_state(g)
    z = np.zeros(g.nc)
    n, dt = 200, gd["dt"]
    out = orc.run(g, p, z, z, z, m, n, dt)
    ds, dxi, deta, s, xi, eta = geom(g, p)
    r = np.sqrt(xi[:, None] ** 2 + eta[None, :] ** 2)
    Ej = np.ones(g.ns); Ej[0] = Ej[-1] = 10.0
    kappa = np.exp(50.0 * r / 2.0)[None] * Ej[:, None, None]
    expect = m * (1 - dt * kappa[None]) ** n * mi.inside_mask(16, 16)[None, None]
    assert np.max(np.abs(out - expect)) < 1e-13
    # golden instance: innermost cell (a=b=8), interior j
    ratio = out[0, 5, 8, 8] / m[0, 5, 8, 8]
    assert ratio == pytest.approx(gd["decay_inner"], rel=1e-12)
    assert ratio / gd["exp_inner"] - 1 == pytest.approx(-9.155e-5, rel=2e-3)
    assert kappa[5, 8, 8] == pytest.approx(gd["kappa_inner"], rel=1e-14)
    assert kappa[5, 7, 0] == pytest.approx(gd["kappa_outer"], rel=1e-14)
    # end cells decay 10x faster (both ends, Q8)
    for j in (0, g.ns - 1):
        assert out[0, j, 8, 8] / m[0, j, 8, 8] == pytest.approx((1 - dt * 10 * gd["kappa_inner"]) ** n, rel=1e-12)


# ---------------------------------------------------------------- C3 exact shift at CFL = 1
@pytest.mark.parametrize("periodic", [False, True])
def test_c3_exact_shift(periodic):
    """S5 in s: upwind side is j-1, zero-inflow ghost, walk-off face."""
    g = Grid(1, 1, 4, 8, 4, 4)
    p = Params(k_spring=0.0, k_on=0.0, k_off0=0.0, flags=mi.FLAG_S_PERIODIC if periodic else 0)
    m, _, _, _ = rand_state(g)
    # theta in {0, pi/2, pi, 3pi/2}: use exact -cos/-sin of the oracle's own theta values
    th = 2 * np.pi * np.arange(g.ntheta) / g.ntheta
    U, V, Om = -np.cos(th), -np.sin(th), np.zeros(g.nc)
    ds = 1.0 / g.ns
    out = orc.run(g, p, U, V, Om, m, 1, ds)
    expect = np.roll(m, 1, axis=1)
    if not periodic:
        expect[:, 0] = 0.0
    assert np.max(np.abs(out - expect)) < 1e-14
    if periodic:
        back = orc.run(g, p, U, V, Om, m, g.ns, ds)
        assert np.max(np.abs(back - m)) < 1e-13


# ---------------------------------------------------------------- C4 steady state
@pytest.mark.parametrize("ns", [4, 32])
def test_c4_steady_state_recursion(ns):
    """S5-S7 together: end cells, walk-off face, source; fixed point is dt independent."""
    gd = read_golden("c4_steady_state.txt")
    g = Grid(1, 1, 2, ns, 3, 3)
    p = Params(k_spring=0.0)
    th = 2 * np.pi * np.arange(g.ntheta) / g.ntheta
    U, V, Om = -np.cos(th), -np.sin(th), np.zeros(g.nc)
    m = np.zeros((g.nc, ns, 3, 3))
    dt = 0.5 / (ns + 10.0)
    out = orc.run(g, p, U, V, Om, m, 6000, dt)
    # exact rational recursion
    a, lam = Fraction(5), Fraction(ns)
    mj, prev = [], Fraction(0)
    for j in range(ns):
        kj = Fraction(10 if j in (0, ns - 1) else 1)
        prev = (a + lam * prev) / (kj + lam)
        mj.append(prev)
    expect = np.array([float(x) for x in mj])
    for ab in [(0, 0), (1, 1), (2, 0)]:
        assert np.max(np.abs(out[0, :, ab[0], ab[1]] - expect)) < 1e-11
        assert np.max(np.abs(out[1, :, ab[0], ab[1]] - expect)) < 1e-11
    if ns == 4:
        for j in range(4):
            assert float(mj[j]) == pytest.approx(gd[f"ns4_m{j}"], rel=1e-15)
        bal = Fraction(1, ns) * sum(a - Fraction(10 if j in (0, 3) else 1) * mj[j] for j in range(4))
        assert bal == mj[-1] == Fraction(459, 490)
    else:
        for j in (0, 1, 15, 30, 31):
            assert out[0, j, 1, 1] == pytest.approx(gd[f"ns32_m{j}"], rel=1e-10)


# ---------------------------------------------------------------- C5 moments
def test_c5_moments_bruteforce_and_analytic():
    """S9: weights, signs, theta dependence, index/layout conventions."""
    gd = read_golden("c5_moments.txt")
    g = Grid(2, 2, 2, 4, 3, 3)
    p = Params()
    ds, dxi, deta, s, xi, eta = geom(g, p)
    dV = ds * dxi * deta
    assert dV == pytest.approx(gd["dV"], rel=1e-15)
    m, _, _, _ = rand_state(g)
    got = orc.moments(g, p, m)
    ld = np.longdouble
    for c in range(g.nc):
        th = 2 * np.pi * (c % 2) / 2
        ct, st_ = ld(math.cos(th)), ld(math.sin(th))
        fx = fy = tq = n0 = ld(0)
        for j in range(4):
            for a in range(3):
                for b in range(3):
                    v = ld(m[c, j, a, b])
                    fx += ld(xi[a]) * v; fy += ld(eta[b]) * v
                    tq += ld(s[j]) * (ld(eta[b]) * ct - ld(xi[a]) * st_) * v
                    n0 += v
        k = ld(50.0)
        assert got["force"][c, 0] == pytest.approx(float(-k * dV * fx), rel=1e-13, abs=1e-17)
        assert got["force"][c, 1] == pytest.approx(float(-k * dV * fy), rel=1e-13, abs=1e-17)
        assert got["torque"][c] == pytest.approx(float(-k * dV * tq), rel=1e-12, abs=1e-17)
        assert got["N0"][c] == pytest.approx(float(dV * n0), rel=1e-14)
    ones = np.ones_like(m)
    r = orc.moments(g, p, ones)
    assert np.allclose(r["N0"], gd["ones_N0"], rtol=1e-14) and np.max(np.abs(r["force"])) < 1e-16
    assert np.max(np.abs(r["torque"])) < 1e-16
    mx = np.broadcast_to(xi[None, None, :, None], m.shape)
    r = orc.moments(g, p, mx)
    assert np.allclose(r["force"][:, 0], gd["xi_Fx"], rtol=1e-14) and np.max(np.abs(r["force"][:, 1])) < 1e-17
    assert np.max(np.abs(r["torque"])) < 1e-17
    mse = np.broadcast_to(s[None, :, None, None] * eta[None, None, None, :], m.shape)
    r = orc.moments(g, p, mse)
    assert np.allclose(r["torque"][0::2], gd["seta_tau_theta0"], rtol=1e-13)
    assert np.allclose(r["torque"][1::2], gd["seta_tau_thetapi"], rtol=1e-13)
    assert np.max(np.abs(r["force"])) < 1e-17
    # cancellation-free scales
    rr = np.sqrt(xi[:, None] ** 2 + eta[None, :] ** 2)
    got = orc.moments(g, p, m)
    assert got["SF"][3] == pytest.approx(50 * dV * np.sum(rr[None] * m[3]), rel=1e-13)
    assert got["Stau"][3] == pytest.approx(50 * dV * np.sum(np.abs(s)[:, None, None] * rr[None] * m[3]), rel=1e-13)


# ---------------------------------------------------------------- C6 delta column
def test_c6_single_cell_delta_column():
    """S3-S7: signs, upwind side selection, conservative pairing -- one column of the update matrix."""
    gd = read_golden("c6_delta_column.txt")
    g = Grid(1, 1, 1, 4, 3, 3)
    p = Params(k_on=0.0)
    m = np.zeros((1, 4, 3, 3)); m[0, 1, 1, 1] = 1.0
    out = orc.run(g, p, [0.3], [-0.2], [0.5], m, 1, 0.01)[0]
    assert out[1, 1, 1] == pytest.approx(gd["self"], rel=1e-14)
    assert out[2, 1, 1] == pytest.approx(gd["s_plus"], rel=1e-14)
    assert out[1, 2, 1] == pytest.approx(gd["xi_plus"], rel=1e-14)
    assert out[1, 0, 1] == gd["xi_minus"] == 0.0
    assert out[1, 1, 2] == gd["eta_plus"] == 0.0
    assert out[1, 1, 0] == pytest.approx(gd["eta_minus"], rel=1e-14)
    assert out.sum() == pytest.approx(gd["total"], rel=1e-14)
    assert np.count_nonzero(out) == 4


def test_c6b_delta_column_theta_quarter_turn():
    """Same column at theta = pi/2 (Ntheta=4, c=1): the walking term moves to eta, the rotation term to xi."""
    g = Grid(1, 1, 4, 4, 3, 3)
    p = Params(k_on=0.0)
    m = np.zeros((1, 4, 3, 3)); m[0, 1, 1, 1] = 1.0
    U, V, Om, dt = 0.3, -0.2, 0.5, 0.01
    out = orc.run(g, p, [U], [V], [Om], m, 1, dt, c_first=1)[0]
    dx = 0.2 / 3
    s1 = -0.125
    # theta = pi/2: p = (0,1), p_perp = (-1,0).  A_xi = U - s*Om = 0.3625 at both xi faces (w*cos = 0 up to 6e-17)
    # A_eta(b+1/2) = V + w(eta=+1/30) = -0.2 + (1 - 50/30/6); A_eta(b-1/2) = -0.2 + (1 + 50/30/6)
    a_xi = U - s1 * Om
    a_eta_p = V + (1 - 50 * (1 / 30) / 6)
    assert out[1, 2, 1] == pytest.approx(dt * a_xi / dx, rel=1e-13)
    assert out[1, 0, 1] == pytest.approx(0.0, abs=1e-17)
    assert out[1, 1, 2] == pytest.approx(dt * a_eta_p / dx, rel=1e-13)
    assert out[1, 1, 0] == pytest.approx(0.0, abs=1e-17)
    assert out[2, 1, 1] == pytest.approx(dt * 1.0 / 0.25, rel=1e-13)
    assert out.sum() == pytest.approx(1 - dt * 1.0, rel=1e-13)


# ---------------------------------------------------------------- C7 symmetries
def test_c7_point_symmetry():
    """S3, S4, S9 sign conventions: theta -> theta+pi, (U,V) -> -(U,V), m(s,xi,eta) -> m(s,-xi,-eta)."""
    g = Grid(1, 1, 8, 8, 6, 6)
    p = Params()
    m, U, V, Om = rand_state(g)
    half = g.ntheta // 2
    m2, U2, V2, Om2 = m.copy(), U.copy(), V.copy(), Om.copy()
    for k in range(half):
        m2[k + half] = m[k][:, ::-1, ::-1]; U2[k + half] = -U[k]; V2[k + half] = -V[k]; Om2[k + half] = Om[k]
    dt = 0.4 * mi.benchmark_dt(g, p, 1.0)
    out = orc.run(g, p, U2, V2, Om2, m2, 25, dt)
    mom = orc.moments(g, p, out)
    for k in range(half):
        assert np.max(np.abs(out[k + half] - out[k][:, ::-1, ::-1])) < 1e-13
        assert np.allclose(mom["force"][k + half], -mom["force"][k], rtol=0, atol=1e-14)
        assert mom["torque"][k + half] == pytest.approx(mom["torque"][k], abs=1e-14)
    assert np.abs(mom["force"]).max() > 1e-4 and np.abs(mom["torque"]).max() > 1e-6


def test_c7b_diagonal_reflection_swaps_xi_eta():
    """A transposed xi/eta operand anywhere fails this: reflect across xi=eta, theta -> pi/2-theta, U<->V, Om -> -Om."""
    g = Grid(1, 1, 8, 8, 6, 6)
    p = Params()
    m, U, V, Om = rand_state(g)
    pairs = {0: 2, 1: 1, 3: 7, 4: 6}
    m2, U2, V2, Om2 = m.copy(), U.copy(), V.copy(), Om.copy()
    for k, k2 in pairs.items():
        if k2 == k:
            continue
        m2[k2] = np.swapaxes(m[k], 1, 2); U2[k2] = V[k]; V2[k2] = U[k]; Om2[k2] = -Om[k]
    dt = 0.4 * mi.benchmark_dt(g, p, 1.0)
    out = orc.run(g, p, U2, V2, Om2, m2, 25, dt)
    mom = orc.moments(g, p, out)
    for k, k2 in pairs.items():
        if k2 == k:
            continue
        assert np.max(np.abs(out[k2] - np.swapaxes(out[k], 1, 2))) < 1e-13
        assert np.allclose(mom["force"][k2], mom["force"][k][::-1], rtol=0, atol=1e-14)
        assert mom["torque"][k2] == pytest.approx(-mom["torque"][k], abs=1e-14)


# ---------------------------------------------------------------- C8 independence / additivity
def test_c8_permutation_and_split():
    g = Grid(2, 3, 4, 6, 5, 7)  # odd sizes
    p = Params()
    m, U, V, Om = rand_state(g)
    dt = 0.4 * mi.benchmark_dt(g, p, 1.0)
    full = orc.run(g, p, U, V, Om, m, 7, dt)
    # configurations are independent: running a slice alone gives the same bits
    sl = slice(5, 11)
    part = orc.run(g, p, U[sl], V[sl], Om[sl], m[sl], 7, dt, c_first=5)
    assert np.array_equal(part, full[sl])
    # substep(a); substep(b) == substep(a+b)
    ab = orc.run(g, p, U, V, Om, orc.run(g, p, U, V, Om, m, 3, dt), 4, dt)
    assert np.array_equal(ab, full)
    # same theta, swapped (x,y) labels: swap whole configurations that share theta
    perm = np.arange(g.nc); perm[[1, 1 + g.ntheta]] = perm[[1 + g.ntheta, 1]]
    sw = orc.run(g, p, U[perm], V[perm], Om[perm], m[perm], 7, dt)
    assert np.array_equal(sw, full[perm])


# ---------------------------------------------------------------- C9 positivity, affinity, mask
def test_c9_positivity_mask_affinity():
    g = Grid(1, 2, 8, 16, 8, 8)
    p = Params()
    m, U, V, Om = rand_state(g)
    dt = mi.benchmark_dt(g, p, 1.0)
    out = orc.run(g, p, U, V, Om, m, 50, dt)
    mask = mi.inside_mask(8, 8)
    assert (out >= 0).all() and (out[:, :, ~mask] == 0).all() and (out[:, :, mask] > 0).all()
    # affine map: step(m1+m2) - step(m2) = step_{k_on=0}(m1)
    m1, m2 = m, rand_state(g)[0]
    lin = orc.run(g, dataclasses.replace(p, k_on=0.0), U, V, Om, m1, 3, dt)
    diff = orc.run(g, p, U, V, Om, m1 + m2, 3, dt) - orc.run(g, p, U, V, Om, m2, 3, dt)
    assert np.max(np.abs(diff - lin)) < 1e-14
    # masked input mass is dropped, not redistributed: garbage outside the disc cannot stay outside
    dirty = m.copy(); dirty[:, :, ~mask] = 7.0
    assert (orc.run(g, p, U, V, Om, dirty, 1, dt)[:, :, ~mask] == 0).all()


def test_stall_clamp_active():
    """Q5: k=200 => load k*xi/f_stall > 1 for xi > 0.03: no back-stepping, W = 0 there."""
    g = Grid(1, 1, 1, 8, 8, 8)
    p = Params(k_spring=200.0, k_on=0.0, k_off0=0.0)
    ds, dxi, deta, s, xi, eta = geom(g, p)
    m = np.zeros((1, 8, 8, 8))
    a_st, a_mv = 5, 2  # xi = +0.0375 (stalled: 1 - 200*0.0375/6 < 0), xi = -0.0375 (w = 2.25)
    m[0, 3, a_st, 4] = 1.0; m[0, 3, a_mv, 4] = 1.0
    dt = 1e-3
    out = orc.run(g, p, [0.0], [0.0], [0.0], m, 1, dt)[0]
    assert out[4, a_st, 4] == 0.0                       # stalled head does not walk
    assert out[4, a_mv, 4] == pytest.approx(dt * 2.25 / ds, rel=1e-13)
    # theta=0: A_xi = w(xi_face) >= 0, stalled faces have zero velocity
    assert out[3, a_st + 1, 4] == 0.0 and out[3, a_st, 4] == 1.0
    assert out[3, a_mv + 1, 4] == pytest.approx(dt * (1 - 200 * (xi[a_mv] + dxi / 2) / 6) / dxi, rel=1e-12)
