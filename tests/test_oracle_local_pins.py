"""Pins of the oracle's local adaptive time step (Alg. 2 l.2-5 PAPER.md:184-190;
readings Q31-Q33 in DESIGN.md): lambda_c = S8 positivity rate maximised over the disc cells of configuration c,
n_c = max(1, ceil(dt lambda_c / cfl)) equal local steps dt / n_c.

L1 closed form of lambda_c where the face velocities are uniform; L2 lambda_c is the SHARP positivity bound of the
substep itself (a delta at the worst cell goes negative just above it and stays non-negative just below) -- ties
`rate_bound` to `run`, two separately written pieces of the oracle; L3 n_c and the landing on t + dt; L4 units are
independent.
"""
import math

import numpy as np

import mm_inputs as mi
from mm_inputs import Grid, Params
from oracle import mm_oracle as orc

RNG = np.random.default_rng(97531)


def kappa_table(g, p):
    xi = -p.R + (np.arange(g.nxi) + 0.5) * 2 * p.R / g.nxi
    eta = -p.R + (np.arange(g.neta) + 0.5) * 2 * p.R / g.neta
    return p.k_off0 * np.exp(p.k_spring * np.hypot(xi[:, None], eta[None, :]) / p.f_detach)


def test_l1_closed_form_uniform_velocities():
    """k = 0 and Omega = 0: W = v0 and A_xi = U + v0 cos, A_eta = V + v0 sin on every face, so
    lambda = v0/ds + |A_xi|/dxi + |A_eta|/deta + E * max_{disc} kappa (max(A,0) - min(A,0) = |A|)."""
    g = Grid(1, 3, 8, 10, 6, 8)
    p = Params(k_spring=0.0, v0=1.3, k_off0=0.7, end_detach_mult=5.0)
    U, V = RNG.random(g.nc) - 0.5, RNG.random(g.nc) - 0.5
    lam = orc.rate_bound(g, p, U, V, np.zeros(g.nc))
    th = 2 * np.pi * (np.arange(g.nc) % g.ntheta) / g.ntheta
    ds, dxi, deta = 1.0 / g.ns, 2 * p.R / g.nxi, 2 * p.R / g.neta
    kmax = kappa_table(g, p)[mi.inside_mask(g.nxi, g.neta)].max() * p.end_detach_mult
    expect = p.v0 / ds + np.abs(U + p.v0 * np.cos(th)) / dxi + np.abs(V + p.v0 * np.sin(th)) / deta + kmax
    assert np.max(np.abs(lam - expect) / expect) < 1e-14
    # with springs the Bell factor picks the disc cell farthest from the centre: the masked corners must not count
    p2 = Params(v0=0.0)
    lam2 = orc.rate_bound(g, p2, np.zeros(g.nc), np.zeros(g.nc), np.zeros(g.nc))
    k2 = kappa_table(g, p2)
    assert np.allclose(lam2, k2[mi.inside_mask(g.nxi, g.neta)].max() * p2.end_detach_mult, rtol=1e-14)
    assert k2.max() > k2[mi.inside_mask(g.nxi, g.neta)].max()


def test_l2_lambda_is_the_sharp_positivity_bound():
    """S8: the coefficient of m[cell] in its own update is 1 - dt * rate(cell).  Put a unit mass in every disc cell in
    turn... is too slow; instead use linearity: with no source, the update of the all-cells-delta family is read off
    m = 1 at one cell.  Scan all disc cells of one configuration for the most negative self-response: it must change
    sign exactly at dt = 1/lambda_c."""
    g = Grid(1, 1, 4, 5, 6, 6)
    p = Params(k_on=0.0, end_detach_mult=3.0)
    U, V, Om = RNG.random(g.nc) - 0.5, RNG.random(g.nc) - 0.5, 4 * RNG.random(g.nc) - 2
    lam = orc.rate_bound(g, p, U, V, Om)
    mask = mi.inside_mask(g.nxi, g.neta)
    cells = [(j, a, b) for j in range(g.ns) for a in range(g.nxi) for b in range(g.neta) if mask[a, b]]
    for c in range(g.nc):
        for scale, want_negative in ((1.0 + 1e-9, True), (1.0 - 1e-9, False)):
            dt = scale / lam[c]
            # one configuration replicated once per probe cell: a delta in a different cell each
            m = np.zeros((len(cells), g.ns, g.nxi, g.neta))
            for i, (j, a, b) in enumerate(cells):
                m[i, j, a, b] = 1.0
            n = len(cells)
            # c_first must keep theta: replicate by calling one at a time would be slow; theta index = c for all
            outs = np.stack([orc.run(g, p, U[c:c + 1], V[c:c + 1], Om[c:c + 1], m[i:i + 1], 1, dt, c_first=c)[0]
                             for i in range(n)])
            self_resp = np.array([outs[i][cells[i]] for i in range(n)])
            assert (self_resp.min() < 0) == want_negative, (c, scale, self_resp.min())
            # every other entry of the response is a non-negative inflow coefficient
            for i in range(n):
                outs[i][cells[i]] = 0.0
            assert outs.min() >= 0.0


def test_l3_step_count_and_landing():
    g = Grid(2, 2, 8, 12, 8, 8)
    p = Params()
    U, V, Om = RNG.random(g.nc) - 0.5, RNG.random(g.nc) - 0.5, 2 * RNG.random(g.nc) - 1
    m = RNG.random((g.nc, g.ns, g.nxi, g.neta)) * mi.inside_mask(g.nxi, g.neta)
    lam = orc.rate_bound(g, p, U, V, Om)
    dt, cfl = 7.3 / lam.mean(), 0.4
    out, n = orc.advance_local(g, p, U, V, Om, m, dt, cfl)
    expect_n = np.maximum(1, np.ceil(dt * lam / cfl)).astype(np.int32)
    assert np.array_equal(n, expect_n) and n.min() >= 1 and len(set(n.tolist())) > 1   # really local
    assert np.all(dt / n * lam <= cfl * (1 + 1e-15))
    for c in (0, 5, g.nc - 1):
        ref = orc.run(g, p, U[c:c + 1], V[c:c + 1], Om[c:c + 1], m[c:c + 1], int(n[c]), dt / n[c], c_first=c)
        assert np.array_equal(ref[0], out[c])
    # a macro step shorter than every local bound is ONE step of size dt
    out1, n1 = orc.advance_local(g, p, U, V, Om, m, 0.3 * cfl / lam.max(), cfl)
    assert (n1 == 1).all()
    assert np.array_equal(out1, orc.run(g, p, U, V, Om, m, 1, 0.3 * cfl / lam.max()))
    assert (out >= 0).all()


def test_l4_units_are_independent():
    g = Grid(1, 2, 4, 6, 8, 8)
    p = Params(flags=mi.FLAG_RK2_SUPERBEE)     # the local step drives whichever scheme the flags select
    U, V, Om = RNG.random(g.nc) - 0.5, RNG.random(g.nc) - 0.5, 2 * RNG.random(g.nc) - 1
    m = RNG.random((g.nc, g.ns, g.nxi, g.neta)) * mi.inside_mask(g.nxi, g.neta)
    dt = 5.0 / orc.rate_bound(g, p, U, V, Om).mean()
    out, n = orc.advance_local(g, p, U, V, Om, m, dt, 0.4)
    perm = np.arange(g.nc)
    perm[[1, 1 + g.ntheta]] = perm[[1 + g.ntheta, 1]]
    out2, n2 = orc.advance_local(g, p, U[perm], V[perm], Om[perm], m[perm], dt, 0.4)
    assert np.array_equal(n2, n[perm]) and np.array_equal(out2, out[perm])
    # ... and each is bitwise its own run of n_c RK2 + Superbee substeps of dt / n_c (ties the local RK2 call to `run`
    # with the flag, which pins R1-R7 fix)
    assert len(set(n.tolist())) > 1
    for c in (0, 3, g.nc - 1):
        ref = orc.run(g, p, U[c:c + 1], V[c:c + 1], Om[c:c + 1], m[c:c + 1], int(n[c]), dt / n[c], c_first=c)
        assert np.array_equal(ref[0], out[c])


def test_l5_local_steps_with_the_coupled_source():
    """Alg. 2 is one loop: local steps (l.5) with the source k_on M_f(r0) (l.20 feeding Eq. 4).  `advance_local(Mf=...)`:
    the step counts do not depend on the table; a uniform table M_f = m_free is the uncoupled call bitwise; every unit is
    bitwise its own `run_coupled` with n_c steps of dt / n_c (ties the coupled local call to the pinned coupled run, N4 /
    N6); and with a one-hot table, no transport and no detachment only the cells anchored on that node change."""
    import dataclasses
    g = Grid(4, 3, 4, 6, 6, 6)
    p = Params(m_free=0.8)
    rng = np.random.default_rng(77)
    m0 = rng.random((g.nc, g.ns, g.nxi, g.neta)) * mi.inside_mask(g.nxi, g.neta)
    U, V, Om = rng.random(g.nc) - 0.5, rng.random(g.nc) - 0.5, 4 * rng.random(g.nc) - 2
    dt = 5.3 / orc.rate_bound(g, p, U, V, Om).mean()
    plain, n_plain = orc.advance_local(g, p, U, V, Om, m0, dt, 0.4)
    same, n_same = orc.advance_local(g, p, U, V, Om, m0, dt, 0.4, Mf=np.full((g.nx, g.ny), 0.8))
    assert np.array_equal(n_plain, n_same) and np.array_equal(plain, same) and len(set(n_plain.tolist())) > 1
    Mf = rng.random((g.nx, g.ny))
    out, n_c = orc.advance_local(g, p, U, V, Om, m0, dt, 0.4, Mf=Mf)
    assert np.array_equal(n_c, n_plain) and np.max(np.abs(out - plain)) > 1e-4
    for c in (0, 5, g.nc - 1):
        ref = orc.run_coupled(g, p, U[c:c + 1], V[c:c + 1], Om[c:c + 1], m0[c:c + 1], int(n_c[c]), dt / n_c[c], Mf, c_first=c)
        assert np.array_equal(out[c:c + 1], ref)
    # a slice of configurations keeps its global indices (theta AND the anchor's node)
    part, _ = orc.advance_local(g, p, U[7:19], V[7:19], Om[7:19], m0[7:19], dt, 0.4, c_first=7, Mf=Mf)
    assert np.array_equal(part, out[7:19])
