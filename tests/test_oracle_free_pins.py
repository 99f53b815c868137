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
