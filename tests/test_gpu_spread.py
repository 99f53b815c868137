"""GPU parity of the motor-force spreading (mm_set_psi / mm_spread_force) against the oracle.

The GPU sums in another order than the oracle (a gather per fluid node in a fixed order by default; fp64 atomic adds,
whose order also differs from run to run, with MM_OPT_SPREAD_ATOMIC): the comparison is
relative to the cancellation-free scale of a node, max_g |F2| of the oracle (all terms of a node share the sign of
f_j up to the mix of configurations; the force field is O(1) everywhere on these inputs)."""
import numpy as np
import pytest

import mm_inputs as mi
from mm_inputs import Grid, Params
from oracle import mm_oracle as orc
from util import NPDT, TOL, random_inputs

pytestmark = pytest.mark.gpu
RNG = np.random.default_rng(1357)


def gpu_spread(g, p, dtype, m0, psi, n_sub=0, dt=0.0, vel=None, atomic=0, twice=False):
    from paper_1908_04279_b200 import MM, binding as b
    mm = MM(g, p, dtype)
    mm.set_option(b.MM_OPT_SPREAD_ATOMIC, atomic)
    assert mm.get_option(b.MM_OPT_SPREAD_ATOMIC) == atomic
    mm.set_density(np.ascontiguousarray(m0, NPDT[dtype]))
    if n_sub:
        mm.set_filament_velocity(*(np.ascontiguousarray(x, NPDT[dtype]) for x in vel))
        mm.substep(n_sub, dt)
    mm.set_psi(np.ascontiguousarray(psi, np.float64))
    F = np.empty((g.nx, g.ny, 2))
    mm.spread_force(F)
    if twice:               # the gather sums in a fixed order: a second call returns the same bits
        F_again = np.empty_like(F)
        mm.spread_force(F_again)
        assert np.array_equal(F, F_again)
    out = np.empty((g.nc, g.ns, g.nxi, g.neta), NPDT[dtype])
    mm.get_density(out)
    mm.destroy()
    return F, out


# the last three: a grid narrower than the stencil (it wraps onto itself), (theta, j) pairs over several ragged chunks,
# a node count that fills neither a transpose tile nor a gather block
@pytest.mark.parametrize("atomic", [0, 1])
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("shape", [(6, 5, 8, 7, 16, 16), (8, 8, 4, 6, 8, 8), (3, 4, 5, 5, 3, 7), (16, 16, 8, 12, 16, 16),
                                   (1, 2, 3, 5, 4, 4), (2, 3, 9, 11, 4, 4), (33, 7, 2, 3, 4, 4)])
def test_spread_parity(dtype, shape, atomic):
    g = Grid(*shape)
    p = Params()
    U, V, Om, m0 = random_inputs(g, p, dtype)
    psi = RNG.random(g.nc)
    F, _ = gpu_spread(g, p, dtype, m0, psi, atomic=atomic, twice=not atomic)
    ref = orc.spread_force(g, p, m0, psi)
    e = np.max(np.abs(F - ref)) / np.max(np.abs(ref))
    assert e <= TOL[dtype], e
    # total force: sum over the grid = dtheta sum_c Psi_c Force_c (F2 of the oracle pins), from the GPU's own moments
    mom = orc.moments(g, p, m0)
    tot = (2 * np.pi / g.ntheta) * (psi[:, None] * mom["force"]).sum(axis=0)
    assert np.max(np.abs(F.sum(axis=(0, 1)) - tot)) / ((2 * np.pi / g.ntheta) * (psi * mom["SF"]).sum()) <= TOL[dtype]


def test_spread_after_substeps_and_hand_weights():
    """The spreading reads the CURRENT density buffer (odd number of passes), and the on-node case of the oracle pin
    F1 comes out of the GPU too."""
    g = Grid(4, 4, 8, 8, 16, 16)
    p = Params()
    U, V, Om, m0 = random_inputs(g, p, "f64")
    psi = RNG.random(g.nc)
    dt = mi.benchmark_dt(g, p, 1.0)
    F, out = gpu_spread(g, p, "f64", m0, psi, n_sub=5, dt=dt, vel=(U, V, Om))
    ref = orc.spread_force(g, p, out, psi)
    assert np.max(np.abs(F - ref)) / np.max(np.abs(ref)) < 1e-12
    g = Grid(8, 8, 4, 4, 2, 2)
    m = np.zeros((g.nc, g.ns, 2, 2))
    c = (3 * g.ny + 5) * g.ntheta
    m[c, 2] = [[1.0, 2.0], [3.0, 5.0]]
    psi = np.zeros(g.nc); psi[c] = 2.0
    F, _ = gpu_spread(g, p, "f64", m, psi)
    w = np.outer([0.25, 0.5, 0.25], [0.25, 0.5, 0.25])
    expect = np.zeros((8, 8, 2))
    expect[3:6, 4:7, 0] = (np.pi / 4) * -0.125 * w
    expect[3:6, 4:7, 1] = (np.pi / 4) * -0.075 * w
    assert np.max(np.abs(F - expect)) < 1e-15


def test_spread_errors():
    from paper_1908_04279_b200 import MM, MMError
    g = Grid(2, 2, 2, 4, 4, 4)
    mm = MM(g, Params(), "f64")
    with pytest.raises(MMError):
        mm.spread_force(np.empty((2, 2, 2)))      # nothing set
    mm.set_density(np.zeros((g.nc, 4, 4, 4)))
    with pytest.raises(MMError):
        mm.spread_force(np.empty((2, 2, 2)))      # psi missing
    mm.set_psi(np.ones(g.nc))
    F = mm.spread_force(np.full((2, 2, 2), 7.0))
    assert (F == 0).all()                          # overwritten, zero density -> zero force
    mm.destroy()
