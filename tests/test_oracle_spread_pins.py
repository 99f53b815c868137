"""Pins of the oracle's motor-force spreading (Eq. 10; readings Q34-Q37).

F1 the discrete delta's weights and the plane force, by hand (golden file): a head exactly on a node and exactly half
way between nodes; F2 total force is conserved (sum_g F2 = dtheta sum_c Psi_c Force_c with the S9 force) including
across the periodic wrap; F3 the first moment of the spread force equals that of the point forces (Peskin's first-
moment condition); F4 translating every configuration by one node translates F2; F5 linearity in Psi and m.
"""
import os

import numpy as np

import mm_inputs as mi
from mm_inputs import Grid, Params
from oracle import mm_oracle as orc
from conftest import GOLDEN

RNG = np.random.default_rng(8642)


def vec_golden(name):
    out = {}
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.split("#", 1)[0].strip()
            if line:
                k, v = line.split("=", 1)
                out[k.strip()] = np.array([float(t) for t in v.split()])
    return out


def test_f1_weights_and_plane_force_by_hand():
    gold = vec_golden("f1_peskin_weights.txt")
    p = Params()
    # (a) theta = 0, ns = 4, nx = 8: heads at ix + 8 s_j = ix - 3, -1, +1, +3 -- all on nodes
    g = Grid(8, 8, 4, 4, 2, 2)
    m = np.zeros((g.nc, g.ns, 2, 2))
    c = (3 * g.ny + 5) * g.ntheta + 0
    m[c, 2] = [[1.0, 2.0], [3.0, 5.0]]                    # plane j = 2: s = +1/8 -> node (4, 5)
    psi = np.zeros(g.nc); psi[c] = 2.0
    F = orc.spread_force(g, p, m, psi)
    scale = (2 * np.pi / 4) * 0.25 * 2.0                    # dtheta ds Psi
    w = np.outer(gold["on_node"], gold["on_node"])
    expect = np.zeros((8, 8, 2))
    expect[3:6, 4:7, 0] = scale * gold["plane_force"][0] * w
    expect[3:6, 4:7, 1] = scale * gold["plane_force"][1] * w
    assert np.max(np.abs(F - expect)) < 1e-16
    # (b) theta = pi/2, ns = 8, ny = 8: heads at iy + 8 s_j = iy +- 0.5, 1.5, ... -- half way between nodes; iy = 7 wraps
    g = Grid(8, 8, 4, 8, 2, 2)
    m = np.zeros((g.nc, g.ns, 2, 2))
    c = (2 * g.ny + 7) * g.ntheta + 1
    m[c, 4] = [[1.0, 2.0], [3.0, 5.0]]                    # s = +1/16 -> gy = 7.5: nodes 6, 7, 0 (wrapped), 1
    psi = np.zeros(g.nc); psi[c] = 1.0
    F = orc.spread_force(g, p, m, psi)
    scale = (2 * np.pi / 4) * 0.125
    # x: theta = pi/2 gives cos = 6e-17, so gx = 2 + 4e-17 rounds to the node: on-node weights in x
    expect = np.zeros((8, 8, 2))
    for u, wx in zip((1, 2, 3), gold["on_node"]):
        for v, wy in zip((6, 7, 0, 1), gold["half_way"]):
            expect[u, v] = scale * wx * wy * gold["plane_force"]
    assert np.max(np.abs(F - expect)) < 1e-15


def test_f2_total_force_is_conserved_across_the_wrap():
    g = Grid(6, 5, 8, 7, 6, 6)
    p = Params()
    m = RNG.random((g.nc, g.ns, g.nxi, g.neta)) * mi.inside_mask(g.nxi, g.neta)
    psi = RNG.random(g.nc)
    F = orc.spread_force(g, p, m, psi)
    mom = orc.moments(g, p, m)
    expect = (2 * np.pi / g.ntheta) * (psi[:, None] * mom["force"]).sum(axis=0)
    scale = (2 * np.pi / g.ntheta) * (psi * mom["SF"]).sum()
    assert np.max(np.abs(F.sum(axis=(0, 1)) - expect)) / scale < 1e-14


def test_f3_first_moment_of_the_spread_force():
    """Heads kept >= 2 nodes from the edge of the unit square (short filament, central configurations), so no wrap:
    sum_g X_g F2[g] = dtheta ds sum_{c,j} Psi_c f_j(c) X_cj  (sum_i (r - i) phi(r - i) = 0)."""
    g = Grid(16, 16, 8, 6, 4, 4)
    p = Params(s_lo=-0.1, s_hi=0.1)
    m = RNG.random((g.nc, g.ns, g.nxi, g.neta)) * mi.inside_mask(g.nxi, g.neta)
    psi = np.zeros(g.nc)
    idx = np.arange(g.nc)
    ix, iy, it = idx // (g.ny * g.ntheta), (idx // g.ntheta) % g.ny, idx % g.ntheta
    central = (ix >= 6) & (ix <= 9) & (iy >= 6) & (iy <= 9)
    psi[central] = RNG.random(central.sum())
    F = orc.spread_force(g, p, m, psi)
    X = np.arange(g.nx)[:, None] / g.nx
    Y = np.arange(g.ny)[None, :] / g.ny
    got = np.array([(X * F[:, :, 0]).sum(), (Y * F[:, :, 0]).sum(), (X * F[:, :, 1]).sum(), (Y * F[:, :, 1]).sum()])
    ds = 0.2 / g.ns
    s = -0.1 + (np.arange(g.ns) + 0.5) * ds
    xi = -p.R + (np.arange(g.nxi) + 0.5) * 2 * p.R / g.nxi
    eta = -p.R + (np.arange(g.neta) + 0.5) * 2 * p.R / g.neta
    dA = (2 * p.R / g.nxi) * (2 * p.R / g.neta)
    fx = -p.k_spring * dA * np.einsum("cjab,a->cj", m, xi)
    fy = -p.k_spring * dA * np.einsum("cjab,b->cj", m, eta)
    th = 2 * np.pi * it / g.ntheta
    Xh = (ix / g.nx)[:, None] + s[None, :] * np.cos(th)[:, None]
    Yh = (iy / g.ny)[:, None] + s[None, :] * np.sin(th)[:, None]
    w = (2 * np.pi / g.ntheta) * ds * psi[:, None]
    expect = np.array([(w * fx * Xh).sum(), (w * fx * Yh).sum(), (w * fy * Xh).sum(), (w * fy * Yh).sum()])
    assert np.max(np.abs(got - expect)) / np.abs(w * np.hypot(fx, fy)).sum() < 1e-14


def test_f4_translation_and_f5_linearity():
    g = Grid(5, 4, 4, 5, 4, 4)
    p = Params()
    m = RNG.random((g.nc, g.ns, g.nxi, g.neta))
    psi = RNG.random(g.nc)
    F = orc.spread_force(g, p, m, psi)
    m5 = m.reshape(g.nx, g.ny, g.ntheta, g.ns, g.nxi, g.neta)
    p5 = psi.reshape(g.nx, g.ny, g.ntheta)
    Fs = orc.spread_force(g, p, np.roll(m5, (1, 2), axis=(0, 1)).reshape(m.shape), np.roll(p5, (1, 2), axis=(0, 1)).reshape(-1))
    assert np.max(np.abs(Fs - np.roll(F, (1, 2), axis=(0, 1)))) < 1e-14
    m2, psi2 = RNG.random(m.shape), RNG.random(g.nc)
    Fa = orc.spread_force(g, p, 2.0 * m + m2, psi)
    assert np.max(np.abs(Fa - (2.0 * F + orc.spread_force(g, p, m2, psi)))) < 1e-13
    Fb = orc.spread_force(g, p, m, psi + 3.0 * psi2)
    assert np.max(np.abs(Fb - (F + 3.0 * orc.spread_force(g, p, m, psi2)))) < 1e-13
    # accumulating two halves of the configuration range equals one call
    h = g.nc // 2
    Fc = orc.spread_force(g, p, m[:h], psi[:h])
    orc.spread_force(g, p, m[h:], psi[h:], c_first=h, F2=Fc)
    assert np.max(np.abs(Fc - F)) < 1e-14
