"""Host logic: seeded workload generators, parameter recipe, replica sharding (gloo, world size 2)."""
import math
import os
import socket

import numpy as np
import pytest


def _min_gap(pos, radii, L):
    """Smallest surface gap over all pairs (brute force, minimum image)."""
    d = pos[:, None, :] - pos[None, :, :]
    d -= L * np.round(d / L)
    r = np.sqrt((d ** 2).sum(-1))
    gap = r - (radii[:, None] + radii[None, :])
    np.fill_diagonal(gap, np.inf)
    return gap.min()


@pytest.mark.parametrize("name,L,xi,rc", [("c1", 16.1199, 1.0195, 3.0), ("c2", 29.1665, 0.8031, 5.3443), ("c3", 45.3202, 1.0337, 4.1521)])
def test_configs_match_the_recipe(workloads, name, L, xi, rc):
    wl = workloads.make_workload(name)
    assert wl.L == pytest.approx(L, abs=1e-3) and wl.xi == pytest.approx(xi, abs=1e-3) and wl.rc == pytest.approx(rc, abs=1e-3)
    phi = (4 * math.pi / 3 * wl.radii ** 3).sum() / wl.L ** 3
    assert phi == pytest.approx(wl.phi, rel=1e-12)
    assert _min_gap(wl.pos, wl.radii, wl.L) >= 0.0
    assert (wl.pos >= 0).all() and (wl.pos < wl.L).all()
    assert wl.rc <= 0.5 * wl.L
    # balanced truncation: exp(-xi^2 rc^2) = exp(-kN^2/4xi^2)
    kN = math.pi * wl.M / wl.L
    assert wl.xi * wl.rc == pytest.approx(kN / (2 * wl.xi), rel=1e-12)
    # deterministic
    wl2 = workloads.make_workload(name)
    assert np.array_equal(wl.pos, wl2.pos) and np.array_equal(wl.S, wl2.S)


def test_composition_of_the_bidisperse_and_polydisperse_recipes(workloads):
    rng = np.random.default_rng(0)
    r2 = workloads.make_radii("bi_1_2", 1000, rng)
    assert (r2 == 2).sum() == 111 and (r2 == 1).sum() == 889
    r4 = workloads.make_radii("bi_1_4", 100_000, rng)
    assert (r4 == 4).sum() == 1538 and (r4 == 1).sum() == 98462
    rl = workloads.make_radii("lognormal", 20000, rng)
    assert rl.min() >= 0.5 and rl.max() <= 2.0 and np.median(rl) == pytest.approx(1.0, abs=0.02)


def test_reduced_config_keeps_the_recipe(workloads):
    wl = workloads.make_workload("c4", N=2000, M=64)
    assert wl.N == 2000 and wl.M == 64 and set(np.unique(wl.radii)) == {1.0, 4.0}
    assert _min_gap(wl.pos, wl.radii, wl.L) >= 0.0


def test_shard_range_partitions_exactly(workloads):
    for n in (0, 1, 7, 64):
        for world in (1, 2, 3, 8):
            got = [i for r in range(world) for i in workloads.shard_range(n, r, world)]
            assert got == list(range(n))
            sizes = [len(workloads.shard_range(n, r, world)) for r in range(world)]
            assert max(sizes) - min(sizes) <= 1


def _gloo_worker(rank, world, port, n_units, q):
    import torch
    import torch.distributed as dist
    import workloads
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    mine = workloads.shard_range(n_units, rank, world)
    # replicas only: no data-path collective; the only exchange is the timing max and the unit count
    t = torch.tensor([float(len(mine)), 1.0 + rank], dtype=torch.float64)
    cnt = t[:1].clone(); dist.all_reduce(cnt, op=dist.ReduceOp.SUM)
    tmax = t[1:].clone(); dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
    dist.barrier()
    q.put((rank, list(mine), cnt.item(), tmax.item()))
    dist.destroy_process_group()


def test_replica_sharding_world_size_2_gloo():
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_gloo_worker, args=(r, 2, port, 5, q)) for r in range(2)]
    for p in procs: p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs: p.join(timeout=60)
    assert res[0][1] + res[1][1] == [0, 1, 2, 3, 4]
    assert res[0][2] == 5.0 and res[1][2] == 5.0      # total units over ranks
    assert res[0][3] == 2.0 and res[1][3] == 2.0      # max-over-ranks timing
