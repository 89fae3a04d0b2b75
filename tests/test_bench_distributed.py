"""The N > 1 path of bench.py on CPU: two gloo ranks.  The stream-collide path does not exchange data between
GPUs (replicas only), so what N > 1 adds is the timing rule -- a step lasts as long as the
slowest rank -- the whole-job aggregation, and per-rank inputs."""
import os
import socket
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench
    import workloads as wl
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    try:
        ms = 10.0 + 5.0 * rank                                   # rank 1 is the slow one
        worst = bench.max_over_ranks(ms, device="cpu")
        w = wl.perturbed_equilibrium(16, 4, 4, seed=bench.rank_seed(rank))
        sums = torch.tensor([float(w.rho.astype(np.float64).sum())], dtype=torch.float64)
        gathered = [torch.zeros_like(sums) for _ in range(world)]
        dist.all_gather(gathered, sums)
        dist.barrier()
        out[rank] = (worst, bench.whole_job_mlups(world, w.n_cells, 7, worst), [float(g.item()) for g in gathered])
    finally:
        dist.destroy_process_group()


def test_two_ranks_gloo():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    world = 2
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert set(res) == {0, 1}
    for rank in (0, 1):
        worst, mlups, sums = res[rank]
        assert worst == 15.0                                      # MAX over ranks, on every rank
        assert abs(mlups - 2 * 256 * 7 / 15e-3 / 1e6) < 1e-9      # all ranks' updates / slowest rank's time
        assert sums[0] != sums[1]                                 # every rank steps its own box (seed + rank)
    assert res[0][2] == res[1][2]


def test_single_process_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.25, device="cpu") == 3.25
    assert bench.whole_job_mlups(1, 1000, 10, 1.0) == 10.0
