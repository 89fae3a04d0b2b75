"""z-slab decomposition of one box over several GPUs (the paper only cites its
multi-GPU version).

The path shards with ONE exchange per time step.  The box is cut into P slabs of nz/P planes; a rank's library handle
holds its slab plus one ghost plane below and one above (local planes 0 .. nzl+1, owned 1 .. nzl).  In the
structure-of-arrays layout a plane of one direction is one contiguous run of nx*ny elements, and after a step only the
directions that cross the face are needed on the other side: the ghost plane BELOW a slab (local z = 0) must hold the
c_z = +1 directions of the lower neighbour's top owned plane (cells at z = 1 pull them upward), the ghost plane ABOVE
(z = nzl+1) the c_z = -1 directions of the upper neighbour's bottom owned plane: 5 of 19 directions per face for D3Q19
(9 of 27, 3 of 9 -- D2Q9 has no z and is not decomposed).  The planes travel in the STORED format, so nothing is
re-encoded and every owned cell sees exactly the inputs it sees in the undecomposed box: the results are bit-identical to
the single-GPU run (tests/test_gpu_slab.py, tests/test_slab_distributed.py).  Ghost cells are computed like any cell
(with the local box's own periodic wrap, i.e. wrongly) and overwritten by the exchange; their flags and initial fields
are the neighbour's, so walls across a slab face bounce correctly.

Two communicators drive the same plan (`halo_plan`):
  * `LocalSlabs`   all P slabs in this process on one device, ghost planes filled by device copies -- the parity
                   test of the plan with the real kernels on one GPU (slabs step one after the other);
  * `DistSlab`     one slab per rank, torch.distributed point-to-point (NCCL over NVLink on GPUs; gloo in the CPU test
                   of the bookkeeping), all sends and receives of a step in one batch.
This module moves bytes between buffers; it holds none of the method's arithmetic.
"""
from __future__ import annotations

import numpy as np

# c_z of the library's direction numbering (R1): D3Q19 = the first 19 of D3Q27
_CZ27 = [0, 0, 0, 0, 0, 1, -1, 0, 0, 1, -1, 1, -1, 0, 0, -1, 1, -1, 1, 1, -1, -1, 1, 1, -1, 1, -1]
_ELEM_BYTES = {0: 4, 7: 8, 8: 4}          # storage format id -> bytes per DDF (all others: 2)


def crossing_directions(velset: int):
    """(directions with c_z = +1, directions with c_z = -1)"""
    if velset not in (19, 27):
        raise ValueError("z-slab decomposition needs a 3-D velocity set (D3Q19 or D3Q27)")
    cz = _CZ27[:velset]
    return [i for i in range(velset) if cz[i] > 0], [i for i in range(velset) if cz[i] < 0]


def halo_plan(velset: int, nx: int, ny: int, nzl: int, elem_bytes: int):
    """The byte ranges of one slab's DDF buffer ([q][nx*ny*(nzl+2)] elements) that take part in the exchange.
    Returns {"send_up": [(offset, nbytes)], "recv_below": [...], "send_down": [...], "recv_above": [...]}: send_up[k]
    of a slab goes to recv_below[k] of the slab above it, send_down[k] to recv_above[k] of the slab below."""
    up, down = crossing_directions(velset)
    plane = nx * ny * elem_bytes
    n_loc = nx * ny * (nzl + 2)

    def at(i, z):
        return ((i * n_loc) + z * nx * ny) * elem_bytes, plane
    return {"send_up": [at(i, nzl) for i in up], "recv_below": [at(i, 0) for i in up],
            "send_down": [at(i, 1) for i in down], "recv_above": [at(i, nzl + 1) for i in down]}


def slab_slice(field, nx, ny, nz, z0, nzl):
    """The planes z0-1 .. z0+nzl (periodic) of a global per-cell field [..., nz*ny*nx] -> [..., (nzl+2)*ny*nx]."""
    f = np.asarray(field)
    lead = f.shape[:-1] if f.ndim > 1 else ()
    g = f.reshape(lead + (nz, ny * nx))
    zs = np.arange(z0 - 1, z0 + nzl + 1) % nz
    return np.ascontiguousarray(g[..., zs, :]).reshape(lead + (-1,))


class _Slab:
    """One slab: a library handle on nzl + 2 planes and the views of its two DDF buffers."""

    def __init__(self, nx, ny, nz, z0, nzl, velset, ddf_format, tau, force, collision):
        import paper_2112_08926_b200 as lbm
        self.nx, self.ny, self.nz, self.z0, self.nzl, self.q = nx, ny, nz, z0, nzl, velset
        self.sim = lbm.Simulation(nx, ny, nzl + 2, velset, ddf_format, tau, force=force, collision=collision)
        self.es = _ELEM_BYTES.get(self.sim.fmt, 2)
        self.plan = halo_plan(velset, nx, ny, nzl, self.es)
        self.buffers = self.sim._keep[:2]                   # the torch uint8 tensors bound as DDF buffers A and B

    def current(self):
        """the buffer holding the current state (lbm_init leaves it in A; every step swaps)"""
        return self.buffers[self.sim.steps_done & 1]

    def set_flags(self, flags):
        self.sim.set_flags(slab_slice(flags, self.nx, self.ny, self.nz, self.z0, self.nzl))

    def init(self, rho, u):
        self.sim.init(slab_slice(rho, self.nx, self.ny, self.nz, self.z0, self.nzl),
                      slab_slice(u, self.nx, self.ny, self.nz, self.z0, self.nzl))

    def owned(self, field):
        """the owned planes of a per-cell field of the local box"""
        f = np.asarray(field)
        lead = f.shape[:-1] if f.ndim > 1 else ()
        return f.reshape(lead + (self.nzl + 2, self.ny * self.nx))[..., 1:-1, :].reshape(lead + (-1,))

    def read_rho_u(self):
        rho, u = self.sim.read_rho_u()
        return self.owned(rho), self.owned(u)

    def read_ddf(self, i):
        return self.owned(self.sim.read_ddf(i))

    def close(self):
        self.sim.close()


def _split(nz, parts):
    if nz % parts != 0:
        raise ValueError("nz must be a multiple of the number of slabs")
    return [(r * (nz // parts), nz // parts) for r in range(parts)]


class LocalSlabs:
    """All slabs in this process, on the current device; the exchange is device-to-device copies."""

    def __init__(self, nx, ny, nz, parts, velset=19, ddf_format="FP32", tau=0.6, force=None, collision=0):
        self.slabs = [_Slab(nx, ny, nz, z0, nzl, velset, ddf_format, tau, force, collision) for z0, nzl in _split(nz, parts)]
        self.nx, self.ny, self.nz, self.q = nx, ny, nz, velset

    def set_flags(self, flags):
        for s in self.slabs:
            s.set_flags(flags)

    def init(self, rho, u):
        for s in self.slabs:
            s.init(rho, u)                                  # (ghost planes come initialised: no exchange needed)

    def exchange(self):
        P = len(self.slabs)
        for r, s in enumerate(self.slabs):
            above, below = self.slabs[(r + 1) % P], self.slabs[(r - 1) % P]
            src = s.current()
            for (so, n), (do, _) in zip(s.plan["send_up"], above.plan["recv_below"]):
                above.current()[do:do + n].copy_(src[so:so + n])
            for (so, n), (do, _) in zip(s.plan["send_down"], below.plan["recv_above"]):
                below.current()[do:do + n].copy_(src[so:so + n])

    def step(self, n=1):
        for _ in range(n):
            for s in self.slabs:
                s.sim.step(1)
            self.exchange()

    def read_rho_u(self):
        parts = [s.read_rho_u() for s in self.slabs]
        return np.concatenate([p[0] for p in parts]), np.concatenate([p[1] for p in parts], axis=1)

    def read_ddf(self, i):
        return np.concatenate([s.read_ddf(i) for s in self.slabs])

    def close(self):
        for s in self.slabs:
            s.close()


def exchange_distributed(buffer, plan, rank, world, dist, group=None):
    """One step's halo exchange of this rank's current DDF buffer (a 1-D uint8 tensor): all sends and receives in one
    batch (with NCCL: one group of point-to-point operations over NVLink; the periodic wrap closes the ring)."""
    above, below = (rank + 1) % world, (rank - 1) % world
    ops = []
    for o, n in plan["send_up"]:
        ops.append(dist.P2POp(dist.isend, buffer[o:o + n], above, group))
    for o, n in plan["send_down"]:
        ops.append(dist.P2POp(dist.isend, buffer[o:o + n], below, group))
    for o, n in plan["recv_below"]:
        ops.append(dist.P2POp(dist.irecv, buffer[o:o + n], below, group))
    for o, n in plan["recv_above"]:
        ops.append(dist.P2POp(dist.irecv, buffer[o:o + n], above, group))
    for req in dist.batch_isend_irecv(ops):
        req.wait()


class DistSlab:
    """This rank's slab of a box decomposed over torch.distributed's world (one process per GPU)."""

    def __init__(self, nx, ny, nz, velset=19, ddf_format="FP32", tau=0.6, force=None, collision=0, group=None):
        import torch.distributed as dist
        self.dist, self.group = dist, group
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)
        z0, nzl = _split(nz, self.world)[self.rank]
        self.slab = _Slab(nx, ny, nz, z0, nzl, velset, ddf_format, tau, force, collision)

    def set_flags(self, flags):
        self.slab.set_flags(flags)

    def init(self, rho, u):
        self.slab.init(rho, u)

    def init_local(self, rho_loc, u_loc, flags_loc=None):
        """fields of the local box (nzl + 2 planes, ghosts included) made by the caller -- for boxes too large to build whole"""
        if flags_loc is not None:
            self.slab.sim.set_flags(flags_loc)
        self.slab.sim.init(rho_loc, u_loc)

    def step(self, n=1):
        for _ in range(n):
            self.slab.sim.step(1)
            exchange_distributed(self.slab.current(), self.slab.plan, self.rank, self.world, self.dist, self.group)

    def read_rho_u(self):
        return self.slab.read_rho_u()

    def read_ddf(self, i):
        return self.slab.read_ddf(i)

    def close(self):
        self.slab.close()
