"""The z-slab decomposition's bookkeeping on CPU (paper_2112_08926_b200/slab.py): the halo plan,
the slicing of global fields into slabs with ghost planes, and the distributed exchange with two gloo ranks.  No kernel
runs here: the buffers are filled with a pattern that names (direction, global plane, cell), and after the exchange
every ghost plane must hold exactly what its neighbour owns, in the directions that cross the face, and nothing else
may have changed.  (The same plan with the real kernels: tests/test_gpu_slab.py.)"""
import os
import socket
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from paper_2112_08926_b200 import slab  # noqa: E402

NX, NY, NZ, Q, ES = 6, 4, 8, 19, 2


def pattern(z0, nzl):
    """buffer of a slab whose local plane l is global plane z0 - 1 + l: byte k of element (i, l, cell) names them"""
    n_loc = NX * NY * (nzl + 2)
    buf = np.zeros((Q, nzl + 2, NX * NY, ES), np.uint8)
    for i in range(Q):
        for l in range(nzl + 2):
            zg = (z0 - 1 + l) % NZ
            buf[i, l, :, 0] = (i * 11 + zg * 3) % 251
            buf[i, l, :, 1] = np.arange(NX * NY) % 253
    return buf.reshape(-1), n_loc


def test_plan_and_crossing_directions():
    up, down = slab.crossing_directions(19)
    assert up == [5, 9, 11, 16, 18] and down == [6, 10, 12, 15, 17]        # c_z of the numbering of DESIGN.md R1
    up27, down27 = slab.crossing_directions(27)
    assert len(up27) == 9 and len(down27) == 9 and set(up27).isdisjoint(down27)
    plan = slab.halo_plan(19, NX, NY, 4, ES)
    plane = NX * NY * ES
    n_loc = NX * NY * 6
    assert plan["send_up"][0] == ((5 * n_loc + 4 * NX * NY) * ES, plane)     # top owned plane of direction 5
    assert plan["recv_below"][0] == ((5 * n_loc) * ES, plane)               # ghost plane below
    assert plan["send_down"][0] == ((6 * n_loc + NX * NY) * ES, plane)
    assert plan["recv_above"][0] == ((6 * n_loc + 5 * NX * NY) * ES, plane)
    for k in plan.values():
        assert len(k) == 5


def test_slab_slice_wraps():
    f = np.arange(NZ * NY * NX)
    s = slab.slab_slice(f, NX, NY, NZ, 0, 4).reshape(6, NY * NX)
    assert np.array_equal(s[0], f.reshape(NZ, -1)[NZ - 1]) and np.array_equal(s[1], f.reshape(NZ, -1)[0])
    u = np.stack([f, 2 * f, 3 * f])
    s3 = slab.slab_slice(u, NX, NY, NZ, 4, 4)
    assert s3.shape == (3, 6 * NY * NX) and np.array_equal(s3[1].reshape(6, -1)[5], 2 * f.reshape(NZ, -1)[0])


def _worker(rank, world, port, out):
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    try:
        nzl = NZ // world
        z0 = rank * nzl
        good, _ = pattern(z0, nzl)
        stale = good.copy().reshape(Q, nzl + 2, NX * NY, ES)
        stale[:, 0] = 0xEE                                       # ghost planes hold garbage after a step
        stale[:, nzl + 1] = 0xEE
        buf = torch.from_numpy(stale.reshape(-1).copy())
        plan = slab.halo_plan(Q, NX, NY, nzl, ES)
        slab.exchange_distributed(buf, plan, rank, world, dist)
        got = buf.numpy().reshape(Q, nzl + 2, NX * NY, ES)
        want = good.reshape(Q, nzl + 2, NX * NY, ES)
        up, down = slab.crossing_directions(Q)
        ok = True
        for i in range(Q):
            ok &= np.array_equal(got[i, 1:-1], want[i, 1:-1])                          # owned planes untouched
            ok &= np.array_equal(got[i, 0], want[i, 0]) if i in up else bool((got[i, 0] == 0xEE).all())
            ok &= np.array_equal(got[i, nzl + 1], want[i, nzl + 1]) if i in down else bool((got[i, nzl + 1] == 0xEE).all())
        out[rank] = bool(ok)
    finally:
        dist.destroy_process_group()


def test_exchange_two_ranks_gloo():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
        res = dict(out)
    assert res == {0: True, 1: True}
