"""mm_free_motors_noalloc (include/mm.h): the free-motor update without a context and without any allocation, its
scratch in a file-scope device array.  Checked against the existing path (mm_update_free_motors on a context) on the
same inputs, on two calls in a row: the second call meets the first call's contents in the shared array.  Collected
last on purpose (the suite runs with pytest -x)."""
import dataclasses

import numpy as np
import pytest

from mm_inputs import Grid, Params
from util import NPDT, TOL, p1_density, random_inputs

pytestmark = pytest.mark.gpu


def existing_path(g, p, dtype, m0, psi):
    """mm_update_free_motors on a context: (M_b,coarse, M_f, the density after the cap rescale)."""
    from paper_1908_04279_b200 import MM
    mm = MM(g, p, dtype)
    mm.set_density(np.ascontiguousarray(m0, NPDT[dtype]))
    mm.set_psi(np.ascontiguousarray(psi, np.float64))
    Mbc, Mf = np.empty((g.nx, g.ny)), np.empty((g.nx, g.ny))
    mm.update_free_motors(Mbc, Mf)
    dens = np.empty((g.nc, g.ns, g.nxi, g.neta), NPDT[dtype])
    mm.get_density(dens)
    mm.destroy()
    return Mbc, Mf, dens


def case(shape, dtype, seed, cap_quantile):
    g = Grid(*shape)
    big = Params(m_free=1e9)
    _, _, _, m0 = random_inputs(g, big, dtype)
    rng = np.random.default_rng(seed)
    psi = rng.random(g.nc) * 30.0
    # M_total such that a part of the nodes is capped: from an uncapped run of the existing path
    raw, _, _ = existing_path(g, big, dtype, m0, psi)
    p = dataclasses.replace(big, m_free=float(np.quantile(raw, cap_quantile)))
    return g, p, np.ascontiguousarray(m0, NPDT[dtype]), psi


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_two_calls_in_a_row_match_the_existing_path(dtype):
    import torch
    from paper_1908_04279_b200 import binding as b
    dev = torch.device("cuda:0")
    # first a 16x16-offset grid (vector kernels, fixed-point tables), then a SMALLER grid with other offsets (generic
    # kernels, fp64 table) that finds the first call's sums, factors and flag in the array; then the first again
    cases = [case((6, 6, 8, 7, 16, 16), dtype, 11, 0.5), case((5, 4, 4, 5, 6, 6), dtype, 12, 0.3),
             case((6, 6, 8, 7, 16, 16), dtype, 13, 0.9)]
    tol = TOL[dtype]
    for k, (g, p, m0, psi) in enumerate(cases):
        Mbc_ref, Mf_ref, dens_ref = existing_path(g, p, dtype, m0, psi)
        assert (Mbc_ref >= p.m_free * (1 - 1e-15)).any() and (Mbc_ref < p.m_free).any()      # the cap binds somewhere
        dens = torch.from_numpy(m0).to(dev)
        psi_d = torch.from_numpy(psi).to(dev)
        Mbc = torch.full((g.nx, g.ny), -1.0, dtype=torch.float64, device=dev)
        Mf = torch.full((g.nx, g.ny), -1.0, dtype=torch.float64, device=dev)
        torch.cuda.synchronize()
        free_before, _ = torch.cuda.mem_get_info()
        b.free_motors_noalloc(g, p, dtype, dens, psi_d, Mbc, Mf)
        torch.cuda.synchronize()
        free_after, _ = torch.cuda.mem_get_info()
        if k == 2:          # same kernels as call 0: nothing left to load lazily, and nothing may have been allocated
            assert free_after >= free_before, (free_before, free_after)
        assert np.max(np.abs(Mbc.cpu().numpy() - Mbc_ref)) / p.m_free <= tol, k
        assert np.max(np.abs(Mf.cpu().numpy() - Mf_ref)) / p.m_free <= tol, k
        assert p1_density(dens.cpu().numpy(), dens_ref) <= tol, k


def test_same_inputs_twice_and_the_size_limit():
    import torch
    from paper_1908_04279_b200 import MMError, binding as b
    dev = torch.device("cuda:0")
    g, p, m0, psi = case((8, 8, 4, 6, 8, 8), "f64", 21, 0.5)
    Mbc_ref, Mf_ref, dens_ref = existing_path(g, p, "f64", m0, psi)
    psi_d = torch.from_numpy(psi).to(dev)
    for _ in range(2):      # back to back on one stream, same inputs: the second result equals the first
        dens = torch.from_numpy(m0).to(dev)
        Mbc = torch.empty((g.nx, g.ny), dtype=torch.float64, device=dev)
        Mf = torch.empty_like(Mbc)
        b.free_motors_noalloc(g, p, "f64", dens, psi_d, Mbc, Mf)
        assert np.max(np.abs(Mbc.cpu().numpy() - Mbc_ref)) / p.m_free <= TOL["f64"]
        assert np.max(np.abs(Mf.cpu().numpy() - Mf_ref)) / p.m_free <= TOL["f64"]
        assert p1_density(dens.cpu().numpy(), dens_ref) <= TOL["f64"]
    # beyond the fixed scratch array: refused with a clear message, nothing launched
    big = Grid(129, 128, 1, 1, 2, 2)
    assert big.nx * big.ny > b.MM_NOALLOC_MAX_NODES
    d = torch.zeros(big.cells, dtype=torch.float64, device=dev)
    ps = torch.zeros(big.nc, dtype=torch.float64, device=dev)
    out = torch.zeros((big.nx, big.ny), dtype=torch.float64, device=dev)
    with pytest.raises(MMError, match="MM_NOALLOC_MAX_NODES"):
        b.free_motors_noalloc(big, p, "f64", d, ps, out, out.clone())
    with pytest.raises(ValueError):
        b.free_motors_noalloc(g, p, "f64", m0, psi_d, Mbc, Mf)       # a host array where a device tensor is required
