"""The N>1 path on CPU: world_size-2 `gloo` process group.

What is checked: the partition of configurations over ranks is exact and contiguous; the ranks' weak-scaling input
streams differ; the only collective of the path -- MAX over ranks of the timed milliseconds -- returns the slowest
rank's time on every rank; and a grid split over two ranks, each rank advancing only its own configurations with no
exchange of any kind, reproduces the unsplit run bit for bit (configurations are independent units).
The last check runs the CPU oracle on each rank (oracle/ is test infrastructure; no GPU here).
"""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1908_04279_b200 import shard  # noqa: E402


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, tmpdir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import mm_inputs as mi
        from oracle import mm_oracle as orc

        # --- the one collective: MAX over ranks of the device-timed milliseconds
        ms = shard.max_over_ranks(10.0 + 5.0 * rank)
        assert ms == 10.0 + 5.0 * (world - 1), ms
        rate = shard.whole_job_rate(1000.0, 4, world, ms)
        assert rate == pytest.approx(1000.0 * world * 4 / (ms * 1e-3))

        # --- weak scaling: each rank draws its own grid
        g = mi.Grid(2, 3, 4, 6, 8, 8)
        p = mi.Params()
        st = mi.Stream(g, p.R, shard.rank_seed(1, rank))
        U, V, Om = st.velocities()
        st.close()
        flat = torch.from_numpy(np.concatenate([U, V, Om]))
        gathered = [torch.empty_like(flat) for _ in range(world)]
        dist.all_gather(gathered, flat)   # test-only exchange, to compare the ranks' inputs
        assert not torch.equal(gathered[0], gathered[1])

        # --- strong split of ONE grid: rank advances only its own configurations, no exchange
        st = mi.Stream(g, p.R, 1)
        U, V, Om = st.velocities()
        m0 = st.density(g.nc)
        st.close()
        dt = mi.benchmark_dt(g, p, 1.0)
        lo, hi = shard.config_range(g.nc, rank, world)
        mine = orc.run(g, p, U[lo:hi], V[lo:hi], Om[lo:hi], m0[lo:hi], 5, dt, c_first=lo)
        mom = orc.moments(g, p, mine, c_first=lo)
        np.save(os.path.join(tmpdir, f"dens{rank}.npy"), mine)
        np.save(os.path.join(tmpdir, f"force{rank}.npy"), mom["force"])
        dist.barrier()
        if rank == 0:
            full = orc.run(g, p, U, V, Om, m0, 5, dt)
            fmom = orc.moments(g, p, full)
            parts = [np.load(os.path.join(tmpdir, f"dens{r}.npy")) for r in range(world)]
            assert np.array_equal(np.concatenate(parts), full)
            fparts = [np.load(os.path.join(tmpdir, f"force{r}.npy")) for r in range(world)]
            assert np.array_equal(np.concatenate(fparts), fmom["force"])
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_config_range_partitions_exactly():
    for nc in (0, 1, 7, 32768, 524288 + 3):
        for world in (1, 2, 3, 8):
            edges = [shard.config_range(nc, r, world) for r in range(world)]
            assert edges[0][0] == 0 and edges[-1][1] == nc
            assert all(a[1] == b[0] for a, b in zip(edges, edges[1:]))
            sizes = [e - b for b, e in edges]
            assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)
    with pytest.raises(ValueError):
        shard.config_range(10, 2, 2)


def test_max_over_ranks_without_process_group_is_identity():
    assert shard.max_over_ranks(3.25) == 3.25


@pytest.mark.timeout(300)
def test_world_size_2_gloo(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
