"""Pins of the oracle's second scheme: RK2 through the half step + Superbee flux limiter
in s (Alg. 2 l.9-10 PAPER.md:194-199; readings Q27-Q30 in DESIGN.md).

The paper prints no formula or number for it, so the pins are closed forms, invariants and a hand-derived step:
R1 conservation, R2 the RK2 amplification factor, R3 exact transport of linear data (what a second-order flux buys),
R4 one step derived by hand (golden file), R5 TVD / range preservation, R6 it beats first-order upwind on smooth and
on discontinuous data, R7 point symmetry and independence of configurations.  None re-uses the oracle's code.
"""
import dataclasses
import os

import numpy as np

import mm_inputs as mi
from mm_inputs import Grid, Params
from oracle import mm_oracle as orc
from conftest import GOLDEN

RK2 = mi.FLAG_RK2_SUPERBEE
RNG = np.random.default_rng(2468)


def s_only(g, extra_flags=0, **kw):
    """Parameters and velocities under which ONLY the s advection acts, at unit speed: k = 0 (W = v0 = 1),
    U = -cos(theta), V = -sin(theta), Omega = 0 (A_xi = A_eta = 0 up to trig rounding), no reactions, no mask."""
    p = Params(k_spring=0.0, k_on=0.0, k_off0=0.0, flags=RK2 | mi.FLAG_OFFSET_PERIODIC_NOMASK | extra_flags, **kw)
    th = 2 * np.pi * (np.arange(g.nc) % g.ntheta) / g.ntheta
    return p, -np.cos(th), -np.sin(th), np.zeros(g.nc)


def vec_golden(name):
    out = {}
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.split("#", 1)[0].strip()
            if line:
                k, v = line.split("=", 1)
                out[k.strip()] = np.array([float(t) for t in v.split()])
    return out


# ---------------------------------------------------------------- R1 conservation
def test_r1_mass_conserved_periodic():
    """Flux form of both stages, limited s faces included (the wrapped slope uses the wrapped neighbours)."""
    g = Grid(2, 1, 4, 9, 4, 5)
    p = Params(k_on=0.0, k_off0=0.0, flags=RK2 | mi.FLAG_S_PERIODIC | mi.FLAG_OFFSET_PERIODIC_NOMASK)
    m = RNG.random((g.nc, g.ns, g.nxi, g.neta))
    U, V, Om = RNG.random(g.nc) - 0.5, RNG.random(g.nc) - 0.5, 2 * RNG.random(g.nc) - 1
    out = orc.run(g, p, U, V, Om, m, 60, 0.5 * mi.benchmark_dt(g, p, 1.0))
    m0, m1 = m.sum(axis=(1, 2, 3)), out.sum(axis=(1, 2, 3))
    assert np.max(np.abs(m1 - m0) / m0) < 1e-13
    assert not np.allclose(out, m)


# ---------------------------------------------------------------- R2 RK2 amplification factor
def test_r2_pure_detachment_amplification():
    """No advection (v0 = 0, U = V = Omega = 0), no source: every cell obeys m' = -kappa m, for which midpoint RK2
    gives m^n = m^0 (1 - z + z^2/2)^n, z = dt kappa (forward Euler would give (1 - z)^n)."""
    g = Grid(1, 1, 2, 6, 4, 4)
    p = Params(v0=0.0, k_on=0.0, flags=RK2 | mi.FLAG_OFFSET_PERIODIC_NOMASK)
    m = RNG.random((g.nc, g.ns, g.nxi, g.neta)) + 0.1
    z0 = np.zeros(g.nc)
    dt, n = 0.01, 25
    out = orc.run(g, p, z0, z0, z0, m, n, dt)
    xi = -p.R + (np.arange(g.nxi) + 0.5) * 2 * p.R / g.nxi
    eta = -p.R + (np.arange(g.neta) + 0.5) * 2 * p.R / g.neta
    kap = p.k_off0 * np.exp(p.k_spring * np.hypot(xi[:, None], eta[None, :]) / p.f_detach)
    kap = np.broadcast_to(kap, (g.ns, g.nxi, g.neta)).copy()
    kap[0] *= p.end_detach_mult
    kap[-1] *= p.end_detach_mult
    z = dt * kap
    expect = m * (1 - z + 0.5 * z * z) ** n
    assert np.max(np.abs(out - expect) / expect) < 1e-13
    euler = m * (1 - z) ** n
    assert np.max(np.abs(out - euler) / expect) > 1e-4   # and it is NOT the Euler factor


# ---------------------------------------------------------------- R3 linear data move exactly
def test_r3_linear_profile_is_transported_exactly():
    """For m = alpha + beta s the Superbee slope is the exact slope (a = b, phi(1) = 1), the face value is the exact
    face-centre value and L(m) = -W beta everywhere, so after n steps m_j = alpha + beta (s_j - W n dt) for ANY dt --
    in the interior, away from the inflow ghost (travels downstream 2 cells per stage at most) and the outflow ghost
    (reaches upstream through the slope, 1 cell per stage)."""
    g = Grid(1, 1, 3, 40, 1, 1)
    p, U, V, Om = s_only(g)
    ds = 1.0 / g.ns
    s = -0.5 + (np.arange(g.ns) + 0.5) * ds
    alpha, beta = 2.0, 1.5
    m = np.broadcast_to((alpha + beta * s)[None, :, None, None], (g.nc, g.ns, 1, 1)).copy()
    n, dt = 3, 0.37 * ds
    out = orc.run(g, p, U, V, Om, m, n, dt)
    expect = alpha + beta * (s - n * dt)
    sl = slice(4 * n + 2, g.ns - 2 * n - 2)
    assert np.max(np.abs(out[:, sl, 0, 0] - expect[None, sl])) < 1e-13
    # a monotone parabola separates the scheme from first-order upwind (error O(ds) there); away from extrema the
    # limiter does not clip
    m2 = np.broadcast_to((1.0 + (s + 1.0) ** 2)[None, :, None, None], (g.nc, g.ns, 1, 1)).copy()
    hi = orc.run(g, p, U, V, Om, m2, n, dt)
    lo = orc.run(g, dataclasses.replace(p, flags=p.flags & ~RK2), U, V, Om, m2, n, dt)
    ex = 1.0 + (s - n * dt + 1.0) ** 2
    assert np.max(np.abs(hi[0, sl, 0, 0] - ex[sl])) < 0.1 * np.max(np.abs(lo[0, sl, 0, 0] - ex[sl]))


# ---------------------------------------------------------------- R4 one step by hand
def test_r4_hand_derived_step():
    """Both branches of the limiter (minmod(2a,b) and minmod(a,2b)), both signs, the zero slope at a sign change,
    the zero inflow and the zero ghost beyond the outflow end, the half step and the full step."""
    gold = vec_golden("r4_superbee_rk2_step.txt")
    g = Grid(1, 1, 4, 5, 1, 1)
    p, U, V, Om = s_only(g)
    for name in ("rising", "falling"):
        m = np.broadcast_to(gold[name + "_in"][None, :, None, None], (g.nc, 5, 1, 1)).copy()
        out = orc.run(g, p, U, V, Om, m, 1, 0.1)
        assert np.max(np.abs(out[:, :, 0, 0] - gold[name + "_out"][None])) < 1e-14, (name, out[:, :, 0, 0])


# ---------------------------------------------------------------- R5 TVD, range preservation
def test_r5_total_variation_does_not_grow():
    """Square pulse, periodic s, CFL 0.4: Superbee is TVD, so with the (SSP) midpoint RK2 no new extrema appear and
    sum |m_{j+1} - m_j| never grows."""
    g = Grid(1, 1, 1, 50, 1, 1)
    p, U, V, Om = s_only(g, extra_flags=mi.FLAG_S_PERIODIC)
    m = np.zeros((1, g.ns, 1, 1))
    m[0, 10:25] = 1.0
    tv_prev, cur = 2.0, m
    for _ in range(40):
        cur = orc.run(g, p, U, V, Om, cur, 1, 0.4 / g.ns)
        v = cur[0, :, 0, 0]
        tv = np.abs(np.diff(np.append(v, v[0]))).sum()
        assert tv <= tv_prev + 1e-12 and v.min() >= -1e-12 and v.max() <= 1 + 1e-12
        tv_prev = tv


# ---------------------------------------------------------------- R6 sharper than upwind
def test_r6_beats_first_order_upwind():
    g = Grid(1, 1, 1, 64, 1, 1)
    p, U, V, Om = s_only(g, extra_flags=mi.FLAG_S_PERIODIC)
    p1 = dataclasses.replace(p, flags=p.flags & ~RK2)
    s = -0.5 + (np.arange(g.ns) + 0.5) / g.ns
    n, dt = 160, 0.4 / g.ns          # exactly one period: 160 * 0.4/64 = 1
    for prof, factor in ((1.5 + np.sin(2 * np.pi * s), 0.2), ((np.abs(s) < 0.2).astype(float), 0.6)):
        m = prof[None, :, None, None].copy()
        e2 = np.abs(orc.run(g, p, U, V, Om, m, n, dt)[0, :, 0, 0] - prof).sum()
        e1 = np.abs(orc.run(g, p1, U, V, Om, m, n, dt)[0, :, 0, 0] - prof).sum()
        assert e2 < factor * e1, (e2, e1)


# ---------------------------------------------------------------- R7 symmetry, independence
def test_r7_point_symmetry_and_independence():
    """theta -> theta + pi, (U,V) -> -(U,V), m(s,xi,eta) -> m(s,-xi,-eta) mirrors the evolution (S3, S4 sign
    conventions, unchanged by the scheme); permuting same-theta configurations permutes outputs bitwise."""
    g = Grid(1, 2, 4, 6, 6, 6)
    p = Params(flags=RK2)
    mask = mi.inside_mask(g.nxi, g.neta)
    m = RNG.random((g.nc, g.ns, g.nxi, g.neta)) * mask
    U, V, Om = RNG.random(g.nc) - 0.5, RNG.random(g.nc) - 0.5, 2 * RNG.random(g.nc) - 1
    dt = mi.benchmark_dt(g, p, 1.0)
    out = orc.run(g, p, U, V, Om, m, 7, dt)
    half = g.ntheta // 2
    idx = np.arange(g.nc).reshape(g.nx * g.ny, g.ntheta)
    shifted = np.roll(idx, -half, axis=1).reshape(-1)          # configuration with theta + pi
    out2 = orc.run(g, p, -U[shifted], -V[shifted], Om[shifted], m[shifted][:, :, ::-1, ::-1].copy(), 7, dt)
    assert np.max(np.abs(out2[:, :, ::-1, ::-1] - out[shifted])) < 1e-13
    perm = np.arange(g.nc)
    perm[[1, 1 + g.ntheta]] = perm[[1 + g.ntheta, 1]]
    out3 = orc.run(g, p, U[perm], V[perm], Om[perm], m[perm], 7, dt)
    assert np.array_equal(out3, out[perm])
    assert (out >= 0).all() and (out[:, :, ~mask] == 0).all()
