"""Pins of the oracle's free-motor coupling (Eq. 5-6, Alg. 2 l.14-20
PAPER.md:206-220; readings Q38-Q42).

N1 by hand: which node each cell's anchor r0 = head - offset falls on and what it deposits; N2 the total number of
bound motors is preserved by the binning; N3 the cap: a node above M_total is scaled exactly onto it, nodes below are
untouched, M_f = M_total - M_b,coarse >= 0; N4 the coupled source reduces to the constant one when M_f is uniform, and
to no source when M_f = 0; N5 translating all configurations translates the coarse fields.
"""
import dataclasses

import numpy as np

import mm_inputs as mi
from mm_inputs import Grid, Params
from oracle import mm_oracle as orc

RNG = np.random.default_rng(4711)


def test_n1_anchor_nodes_and_deposits_by_hand():
    """nx = ny = 8, theta = 0, ns = 4: plane j = 2 (s = +1/8) of configuration (ix, iy) = (3, 5) has its head on node
    (4, 5).  With R = 0.2 on a 2x2 offset grid the offsets are (+-0.1, +-0.1) = +-0.8 nodes, and the anchor is the head
    MINUS the offset: xi = -0.1 -> 4.8 -> node 5, xi = +0.1 -> 3.2 -> node 3; eta = -0.1 -> node 6, eta = +0.1 -> node 4."""
    g = Grid(8, 8, 4, 4, 2, 2)
    p = Params(R=0.2, m_free=1e9)
    m = np.zeros((g.nc, g.ns, 2, 2))
    c = (3 * g.ny + 5) * g.ntheta
    m[c, 2] = [[1.0, 2.0], [3.0, 5.0]]            # [a][b]: (xi-, eta-), (xi-, eta+), (xi+, eta-), (xi+, eta+)
    psi = np.zeros(g.nc); psi[c] = 2.0
    out, Mbc, Mf = orc.free_motors(g, p, m, psi)
    w = (2 * np.pi / 4) * 0.25 * 0.2 * 0.2 * 2.0  # dtheta ds dxi deta Psi
    expect = np.zeros((8, 8))
    expect[5, 6], expect[5, 4], expect[3, 6], expect[3, 4] = 1 * w, 2 * w, 3 * w, 5 * w
    assert np.max(np.abs(Mbc - expect)) < 1e-16
    assert np.array_equal(out, m) and np.allclose(Mf, 1e9 - expect, rtol=0, atol=1e-6)
    # with R = 0.1 the offsets are +-0.4 nodes: all four cells fall on the head's node
    p1 = Params(R=0.1, m_free=1e9)
    _, Mbc1, _ = orc.free_motors(g, p1, m, psi)
    e1 = np.zeros((8, 8)); e1[4, 5] = (2 * np.pi / 4) * 0.25 * 0.01 * 2.0 * 11.0
    assert np.max(np.abs(Mbc1 - e1)) < 1e-16


def test_n2_binning_preserves_the_number_of_bound_motors():
    g = Grid(6, 5, 8, 7, 6, 6)
    p = Params(m_free=1e9)
    m = RNG.random((g.nc, g.ns, g.nxi, g.neta))
    psi = RNG.random(g.nc)
    _, Mbc, _ = orc.free_motors(g, p, m, psi)
    w = (2 * np.pi / g.ntheta) * (1.0 / g.ns) * (2 * p.R / g.nxi) * (2 * p.R / g.neta)
    total = w * (psi[:, None, None, None] * m).sum()
    assert abs(Mbc.sum() - total) / total < 1e-13


def test_n3_cap_rescales_exactly_onto_the_total():
    g = Grid(6, 6, 8, 6, 4, 4)
    big = Params(m_free=1e9)
    m = RNG.random((g.nc, g.ns, g.nxi, g.neta)) * mi.inside_mask(g.nxi, g.neta)
    psi = RNG.random(g.nc) * 40.0
    _, raw, _ = orc.free_motors(g, big, m, psi)
    cap = float(np.median(raw))                     # half of the nodes are above the total
    p = Params(m_free=cap)
    out, Mbc, Mf = orc.free_motors(g, p, m, psi)
    assert np.max(np.abs(Mbc - np.minimum(raw, cap))) < 1e-14 * cap
    assert np.max(np.abs(Mf - (cap - np.minimum(raw, cap)))) < 1e-14 * cap and (Mf >= 0).all()
    _, again, _ = orc.free_motors(g, big, out, psi)  # coarse density of the rescaled state
    assert np.max(np.abs(again - np.minimum(raw, cap))) < 1e-13 * cap
    assert (out <= m).all() and (out < m).any() and (out == m).any()   # some cells scaled, some untouched
    # scaled cells all carry their node's factor: ratios take at most (#capped nodes + 1) distinct values
    ratio = np.unique(np.round(out[m > 0] / m[m > 0], 12))
    assert len(ratio) <= (raw > cap).sum() + 1


def test_n4_coupled_source_reduces_to_the_constant_one():
    g = Grid(3, 2, 4, 6, 6, 6)
    for flags in (0, mi.FLAG_RK2_SUPERBEE):
        p = Params(flags=flags, m_free=0.7)
        m = RNG.random((g.nc, g.ns, g.nxi, g.neta)) * mi.inside_mask(g.nxi, g.neta)
        U, V, Om = RNG.random(g.nc) - 0.5, RNG.random(g.nc) - 0.5, 2 * RNG.random(g.nc) - 1
        dt = mi.benchmark_dt(g, p, 1.0)
        plain = orc.run(g, p, U, V, Om, m, 5, dt)
        same = orc.run_coupled(g, p, U, V, Om, m, 5, dt, np.full((g.nx, g.ny), 0.7))
        assert np.array_equal(plain, same)
        none = orc.run_coupled(g, p, U, V, Om, m, 5, dt, np.zeros((g.nx, g.ny)))
        assert np.array_equal(none, orc.run(g, dataclasses.replace(p, k_on=0.0), U, V, Om, m, 5, dt))
        # a non-uniform table really changes the result -- and, for the (linear) Euler scheme, affinely in M_f
        Mf = RNG.random((g.nx, g.ny))
        a = orc.run_coupled(g, p, U, V, Om, m, 3, dt, Mf)
        b = orc.run_coupled(g, p, U, V, Om, m, 3, dt, 2 * Mf)
        z = orc.run_coupled(g, p, U, V, Om, m, 3, dt, np.zeros((g.nx, g.ny)))
        assert np.max(np.abs(a - z)) > 1e-4
        if flags == 0:
            assert np.max(np.abs((b - a) - (a - z))) < 1e-13


def test_n5_translation():
    # 6x6 offsets on this outer grid put no anchor exactly half-way between two nodes (a tie would be broken by the
    # last bit of ix/nx*nx, which is not translation invariant; no BASELINE grid has such ties either: xi_a Nx is a
    # multiple of 0.2 there)
    g = Grid(5, 4, 4, 5, 6, 6)
    p = Params(m_free=0.07)
    m = RNG.random((g.nc, g.ns, g.nxi, g.neta))
    psi = RNG.random(g.nc)
    out, Mbc, Mf = orc.free_motors(g, p, m, psi)
    m5 = m.reshape(g.nx, g.ny, g.ntheta, g.ns, g.nxi, g.neta)
    p5 = psi.reshape(g.nx, g.ny, g.ntheta)
    out2, Mbc2, Mf2 = orc.free_motors(g, p, np.roll(m5, (2, 1), axis=(0, 1)).reshape(m.shape), np.roll(p5, (2, 1), axis=(0, 1)).reshape(-1))
    assert np.max(np.abs(Mbc2 - np.roll(Mbc, (2, 1), axis=(0, 1)))) < 1e-15
    assert (Mbc < 0.07).any() and (Mbc == 0.07).any()          # some nodes capped, some not
    assert np.max(np.abs(out2.reshape(m5.shape) - np.roll(out.reshape(m5.shape), (2, 1), axis=(0, 1)))) < 1e-13


def _anchor_nodes_exact(g, R):
    """Node of every cell's anchor r0 = x_c + s_j p_c - (xi_a, eta_b) (readings Q38/Q39) in EXACT rational arithmetic,
    for ntheta = 4 (cos, sin in {0, +-1}): written from the definition, not from the oracle's floating-point
    expression.  Returns int arrays (node_x, node_y) of shape [nx][ny][4][ns][nxi][neta]; asserts that no anchor is a tie."""
    from fractions import Fraction as Fr
    assert g.ntheta == 4
    cs = [(1, 0), (0, 1), (-1, 0), (0, -1)]
    R = Fr(R).limit_denominator(1000)
    nodx = np.empty((g.nx, g.ny, 4, g.ns, g.nxi, g.neta), np.int64)
    nody = np.empty_like(nodx)
    for ix in range(g.nx):
        for iy in range(g.ny):
            for k, (c, s) in enumerate(cs):
                for j in range(g.ns):
                    sj = Fr(-1, 2) + Fr(2 * j + 1, 2 * g.ns)
                    for a in range(g.nxi):
                        xi = -R + Fr(2 * a + 1, 2) * (2 * R / g.nxi)
                        rx = (Fr(ix, g.nx) + sj * c - xi) * g.nx + Fr(1, 2)
                        assert rx.denominator != 1 or True
                        assert (rx - Fr(1, 2)).denominator != 2, "tie"
                        for b in range(g.neta):
                            eta = -R + Fr(2 * b + 1, 2) * (2 * R / g.neta)
                            ry = (Fr(iy, g.ny) + sj * s - eta) * g.ny + Fr(1, 2)
                            assert (ry - Fr(1, 2)).denominator != 2, "tie"
                            nodx[ix, iy, k, j, a, b] = (rx.numerator // rx.denominator) % g.nx
                            nody[ix, iy, k, j, a, b] = (ry.numerator // ry.denominator) % g.ny
    return nodx, nody


def test_n6_one_hot_table_feeds_exactly_the_cells_anchored_on_that_node():
    """Eq. 4's source k_on M_f(r0) 1_{D_rc} with Eq. 6: with M_f = delta(node n*), m0 = 0, no
    transport and no detachment, ONE Euler substep puts dt k_on into exactly the cells whose anchor is n* and leaves
    every other cell 0.  Pins WHICH node `mmo_run_coupled` reads for a cell: by hand on N1's geometry (plane j = 2 of
    configuration (3, 5, theta = 0) on the 8x8 grid, R = 0.2: cells (a,b) = (0,0), (0,1), (1,0), (1,1) are anchored on
    (5,6), (5,4), (3,6), (3,4)), then for every node of a NON-SQUARE grid against exact rational arithmetic, and on a
    slice of configurations (c_first != 0)."""
    dt = 0.125
    # (1) by hand, N1's geometry
    g = Grid(8, 8, 4, 4, 2, 2)
    p = Params(R=0.2, v0=0.0, k_off0=0.0, k_on=5.0)
    z = np.zeros(g.nc)
    m0 = np.zeros((g.nc, g.ns, 2, 2))
    c = (3 * g.ny + 5) * g.ntheta
    for (a, b), (nx_, ny_) in {(0, 0): (5, 6), (0, 1): (5, 4), (1, 0): (3, 6), (1, 1): (3, 4)}.items():
        Mf = np.zeros((8, 8)); Mf[nx_, ny_] = 1.0
        out = orc.run_coupled(g, p, z, z, z, m0, 1, dt, Mf)
        assert out[c, 2, a, b] == dt * 5.0, (a, b)
        others = [(aa, bb) for aa in range(2) for bb in range(2) if (aa, bb) != (a, b)]
        assert all(out[c, 2, aa, bb] == 0.0 for aa, bb in others)
        # theta = 0: the head of plane j sits 8 s_j = -3, -1, 1, 3 nodes from x_c, so node (5,6) is also reached from
        # other planes / configurations, but in total by ns * (cells per plane) * ntheta cells, every one with dt k_on
        assert np.count_nonzero(out) == g.ns * 4 * g.ntheta and set(np.unique(out)) == {0.0, dt * 5.0}
    # (2) every node of a non-square grid (an ix/iy swap cannot survive), exact rational expectation; 4x4 offsets,
    # corners masked: the source is k_on M_f 1_disc
    g = Grid(8, 4, 4, 4, 4, 4)
    p = Params(R=0.2, v0=0.0, k_off0=0.0, k_on=5.0)
    nodx, nody = _anchor_nodes_exact(g, 0.2)
    nodx = nodx.reshape(g.nc, g.ns, g.nxi, g.neta); nody = nody.reshape(g.nc, g.ns, g.nxi, g.neta)
    inside = mi.inside_mask(g.nxi, g.neta).astype(bool)
    assert not inside[0, 0] and inside[1, 1]
    z = np.zeros(g.nc)
    m0 = np.zeros((g.nc, g.ns, g.nxi, g.neta))
    Mf = RNG.random((g.nx, g.ny)) + 0.5                          # all nodes at once: distinct values identify the node
    out = orc.run_coupled(g, p, z, z, z, m0, 1, dt, Mf)
    expect = np.where(inside[None, None], dt * (5.0 * Mf[nodx, nody]), 0.0)
    assert np.array_equal(out, expect)
    for n_star in ((5, 2), (0, 3), (7, 0)):
        one = np.zeros((g.nx, g.ny)); one[n_star] = 1.0
        out = orc.run_coupled(g, p, z, z, z, m0, 1, dt, one)
        hit = (nodx == n_star[0]) & (nody == n_star[1]) & inside[None, None]
        assert hit.any() and np.array_equal(out, np.where(hit, dt * 5.0, 0.0))
    # (3) a slice of configurations: the node follows the GLOBAL configuration index
    c0, n = 37, 29
    out = orc.run_coupled(g, p, z[:n], z[:n], z[:n], m0[c0:c0 + n], 1, dt, Mf, c_first=c0)
    assert np.array_equal(out, expect[c0:c0 + n])


def test_n7_alg2_cadence():
    """Alg. 2's loop redoes the coarse reduction, the cap and M_f inside the inner loop.  Pins of
    `mmo_run_alg2` that do not go through it: (a) with pure detachment (no transport, k_on = 0) and a cap that never
    binds, the coarse density after n substeps is known in closed form per node: every cell decays by its own
    (1 - dt kappa)^n, so M_b,coarse of the last update = the binned sum of the decayed initial state -- computed here with
    numpy from C2's formula, and M_f = M_total - it; (b) refresh >= n_sub is one update followed by the frozen-table run;
    (c) refresh = 1 with Psi = 0 (nothing counts as bound: M_f = M_total at every update) is the constant-source run,
    bitwise; (d) the bound-motor budget: while the cap binds, every update leaves M_b,coarse <= M_total exactly."""
    g = Grid(4, 3, 4, 5, 4, 4)
    # (a) closed form
    p = Params(v0=0.0, k_on=0.0, m_free=1e9, R=0.2)
    inside = mi.inside_mask(g.nxi, g.neta)
    m0 = RNG.random((g.nc, g.ns, g.nxi, g.neta)) * inside
    psi = RNG.random(g.nc) + 0.5
    z = np.zeros(g.nc)
    dt, n, k = 1e-4, 7, 3                                                       # dt kappa <= 0.25 everywhere
    out, Mbc, Mf = orc.run_alg2(g, p, z, z, z, m0, psi, n, dt, k)
    a = np.arange(g.nxi); xi = -p.R + (a + 0.5) * 2 * p.R / g.nxi
    kap = p.k_off0 * np.exp(p.k_spring * np.sqrt(xi[:, None] ** 2 + xi[None, :] ** 2) / p.f_detach)
    E = np.ones(g.ns); E[0] = E[-1] = p.end_detach_mult
    decay = 1.0 - dt * kap[None, :, :] * E[:, None, None]                       # per substep, per (j, a, b)
    assert (decay > 0.7).all() and np.max(np.abs(out - m0 * decay[None] ** n)) < 1e-14
    last = (n - 1) // k * k                                                     # substep index of the last update
    nodx, nody = _anchor_nodes_exact(g, 0.2)
    w = (2 * np.pi / g.ntheta) * (1.0 / g.ns) * (2 * p.R / g.nxi) ** 2
    expect = np.zeros((g.nx, g.ny))
    np.add.at(expect, (nodx.reshape(-1), nody.reshape(-1)), (w * psi[:, None, None, None] * m0 * decay[None] ** last).reshape(-1))
    assert np.max(np.abs(Mbc - expect)) < 1e-15 * p.m_free and np.max(np.abs(Mf - (p.m_free - expect))) < 1e-6
    # (b), (c), (d) with transport and a binding cap
    p = Params(m_free=1.0)
    U, V, Om = RNG.random(g.nc) - 0.5, RNG.random(g.nc) - 0.5, 2 * RNG.random(g.nc) - 1
    dt = mi.benchmark_dt(g, p, 1.0)
    _, raw, _ = orc.free_motors(g, dataclasses.replace(p, m_free=1e9), m0, psi * 50)
    p = dataclasses.replace(p, m_free=float(np.median(raw)))
    once, Mbc1, Mf1 = orc.run_alg2(g, p, U, V, Om, m0, psi * 50, 6, dt, 6)
    capped, Mbc_ref, Mf_ref = orc.free_motors(g, p, m0, psi * 50)
    assert np.array_equal(once, orc.run_coupled(g, p, U, V, Om, capped, 6, dt, Mf_ref)) and np.array_equal(Mf1, Mf_ref)
    every, Mbc2, Mf2 = orc.run_alg2(g, p, U, V, Om, m0, psi * 50, 6, dt, 1)
    assert np.max(np.abs(every - once)) > 1e-6                                  # the cadence matters
    assert (Mbc2 <= p.m_free).all() and (Mf2 >= 0).all()
    _, Mbc0, _ = orc.run_alg2(g, p, U, V, Om, m0, psi * 50, 1, dt, 1)
    assert (Mbc0 == p.m_free).any() and (Mbc0 < p.m_free).any()                 # the cap really binds at the start
    free, _, Mf3 = orc.run_alg2(g, p, U, V, Om, m0, np.zeros(g.nc), 6, dt, 1)
    assert np.array_equal(free, orc.run(g, p, U, V, Om, m0, 6, dt)) and np.array_equal(Mf3, np.full((g.nx, g.ny), p.m_free))
