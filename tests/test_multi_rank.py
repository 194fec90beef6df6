"""The N > 1 path of bench.py on CPU: two gloo ranks, each with its own problem (seed + rank), times combined
as the max over ranks, whole-job rate summed over ranks.  No GPU needed."""
import os

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2412_12360_b200 import sharding, workloads as wl
    w = wl.c3_mini(nx=24, ny=20, nz=20, d=4, n_steps=4, seed=sharding.problem_seed(33, rank))
    ms = sharding.max_over_ranks(10.0 * (rank + 1))
    rate = sharding.whole_job_rate(w.cells * w.n_steps, 3, ms, world)
    chk = torch.tensor([float(np.asarray(w.meta["rho"]).sum())], dtype=torch.float64)
    gathered = [torch.zeros_like(chk) for _ in range(world)]
    dist.all_gather(gathered, chk)
    out[rank] = (ms, rate, [float(g.item()) for g in gathered], w.cells * w.n_steps)
    dist.destroy_process_group()


def test_two_gloo_ranks_independent_problems_and_max_time():
    world, port = 2, 29500 + os.getpid() % 2000
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert set(res) == {0, 1}
    for rank in range(world):
        ms, rate, sums, cs = res[rank]
        assert ms == 20.0                                        # the slowest rank's time, on every rank
        assert abs(rate - world * cs * 3 / 20e-3 / 1e6) < 1e-9    # aggregate over both ranks
        assert sums[0] != sums[1]                                # different seeds: different problems
    assert res[0][2] == res[1][2]


# ------------------------------------------------------------------------------------------------------------------
# Domain decomposition along z: the host logic of sharding.py -- which planes a rank holds, how
# sources / detectors are cut, which halo planes travel where -- without a GPU.
# ------------------------------------------------------------------------------------------------------------------
def test_z_slab_plan_covers_the_grid_once_with_one_ghost_plane_per_cut():
    from paper_2412_12360_b200 import sharding
    for nz, world, d in [(44, 2, 8), (44, 3, 8), (600, 8, 16), (200, 4, 12), (17, 1, 3)]:
        slabs = sharding.z_slabs(nz, world, d)
        assert [s.k_lo for s in slabs] == [0] + [s.k_hi for s in slabs[:-1]] and slabs[-1].k_hi == nz
        for s in slabs:
            assert s.ghost_lo == (0 if s.rank == 0 else 1) and s.ghost_hi == (0 if s.rank == world - 1 else 1)
            assert s.z_offset == s.k_lo - s.ghost_lo and s.nz == s.k_hi - s.k_lo + s.ghost_lo + s.ghost_hi
            kw = s.grid_kwargs()
            assert kw["z_offset"] + kw["nz"] <= nz and kw["z_global"] == nz
            assert max(c.nz for c in slabs) - min(c.nz for c in slabs) <= 3          # balanced
    import pytest
    with pytest.raises(ValueError):
        sharding.z_slabs(44, 2, 8, cuts=[5])            # the lower slab would own no interior plane
    with pytest.raises(ValueError):
        sharding.z_slabs(44, 3, 8, cuts=[30, 20])


def test_sources_and_detectors_are_cut_to_the_slab():
    from paper_2412_12360_b200 import sharding, workloads as wl
    w = wl.c3_mini(n_steps=4)
    w.sources.append(wl.Source(2, (10, 10, 18), (30, 20, 26), w.sources[0].waveform,
                               np.arange(8 * 10 * 20, dtype=np.float32).reshape(8, 10, 20)))
    w.detectors.append(wl.Detector(0b100010, (10, 10, 18), (70, 40, 24), [0.3]))
    slabs = sharding.z_slabs(w.nz, 3, w.pml_cells, cuts=[20, 23])
    seen = np.zeros(8, dtype=int)
    for s in slabs:
        src = sharding.local_sources(w.sources, s)
        for q in src:
            assert 0 <= q.lo[2] < q.hi[2] <= s.nz
            if q.component == 2:                         # the box source: profile rows follow the planes kept
                k0 = q.lo[2] + s.z_offset
                assert q.profile.shape[0] == q.hi[2] - q.lo[2]
                assert q.profile[0, 0, 0] == (k0 - 18) * 200
        fwd = sharding.local_detectors(w.detectors, s, with_ghosts=False)
        bwd = sharding.local_detectors(w.detectors, s, with_ghosts=True)
        for idx, d, sl in fwd:
            if idx == 1:
                seen[sl] += 1                            # owned planes: every plane of the box exactly once over the slabs
                assert d.lo[2] + s.z_offset >= s.k_lo and d.hi[2] + s.z_offset <= s.k_hi
        for idx, d, sl in bwd:
            assert 0 <= d.lo[2] < d.hi[2] <= s.nz
        n_f = sum(sl.stop - sl.start for i, _, sl in fwd if i == 1)
        n_b = sum(sl.stop - sl.start for i, _, sl in bwd if i == 1)
        assert n_b >= n_f                                # the backward boxes reach into the ghost planes
    assert (seen[:6] == 1).all()


def _halo_worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2412_12360_b200 import sharding
    slab = sharding.z_slabs(30, world, 4)[rank]
    shape = (3, 5, 8)
    down = torch.full(shape, 10.0 * rank + 1)            # my lowest owned plane
    up = torch.full(shape, 10.0 * rank + 2)              # my highest owned plane
    below, above = torch.full(shape, -1.0), torch.full(shape, -1.0)
    for _ in range(3):                                    # several steps: the pairing must not drift
        sharding.exchange_halos_dist(slab, down, up, below, above)
    out[rank] = (float(below[0, 0, 0]), float(above[2, 4, 7]))
    dist.destroy_process_group()


def test_halo_exchange_over_three_gloo_ranks():
    world, port = 3, 31500 + os.getpid() % 2000
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_halo_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    # ghost below <- the lower neighbour's highest plane; ghost above <- the upper neighbour's lowest plane
    assert res[0] == (-1.0, 11.0)
    assert res[1] == (2.0, 21.0)
    assert res[2] == (12.0, -1.0)


def _token_worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2412_12360_b200 import sharding
    slab = sharding.z_slabs(30, world, 4)[rank]
    token, scratch = torch.zeros(1), torch.full((2, 1), -1.0)
    seen = []
    for step in range(4):                                  # the token of step n must meet the neighbours' token of step n
        token.fill_(100.0 * step + rank)
        sharding.neighbour_tokens(slab, token, scratch)
        seen.append((float(scratch[0, 0]), float(scratch[1, 0])))
    out[rank] = seen
    dist.destroy_process_group()


def test_neighbour_tokens_over_three_gloo_ranks():
    """What is left of the halo exchange with peer stores (include/fdtd.h "Peer stores"): one token to and from every
    neighbour per step, paired step by step."""
    world, port = 3, 33500 + os.getpid() % 2000
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_token_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    for step in range(4):
        assert res[0][step] == (-1.0, 100.0 * step + 1)       # no neighbour below
        assert res[1][step] == (100.0 * step + 0, 100.0 * step + 2)
        assert res[2][step] == (100.0 * step + 1, -1.0)
