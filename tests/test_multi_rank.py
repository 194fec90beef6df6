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
