"""GPU parity of the z-slab decomposition (paper_2112_08926_b200/slab.py): a box cut into 2 and
4 slabs, each a library handle of its own with ghost planes, exchanged after every step, must reproduce the undecomposed
run -- and therefore the oracle -- bit for bit, in every stored DDF.  All slabs live on the one GPU of the test box and
step one after the other (LocalSlabs); the distributed exchange of the same plan is tested with two gloo ranks in
tests/test_slab_distributed.py."""
import numpy as np
import pytest

import oracle
import paper_2112_08926_b200 as lbm
import workloads as wl
from paper_2112_08926_b200 import slab
from workloads import FORMATS

pytestmark = pytest.mark.gpu


def _run(w, name, parts, steps, collision=lbm.BGK):
    force = w.force if any(float(v) != 0.0 for v in w.force) else None
    s = slab.LocalSlabs(w.nx, w.ny, w.nz, parts, w.velset, name, w.tau, force, collision)
    if w.flags.any():
        s.set_flags(w.flags)
    s.init(w.rho, w.u)
    s.step(steps)
    return s


@pytest.mark.parametrize("name", ["FP32", "FP16S", "FP16C", "P16_1S", "FP64"])
@pytest.mark.parametrize("q,shape,parts", [(19, (24, 7, 8), 2), (19, (272, 5, 12), 4), (27, (32, 6, 8), 2)])
def test_slabs_equal_the_whole_box(q, shape, parts, name):
    w = wl.perturbed_equilibrium(*shape, seed=71, velset=q, tau=0.7)
    w = wl.random_walls(w, 0.1, seed=73, moving_fraction=0.5)       # walls across the slab faces too
    w.force = (1e-5, -2e-5, 3e-5)
    steps = 9
    s = _run(w, name, parts, steps)
    if name == "FP64":
        # (the C ABI takes tau and the force as floats: the FP64 oracle gets them rounded the same way, R16)
        import dataclasses
        w64 = dataclasses.replace(w, tau=float(np.float32(w.tau)), force=tuple(float(np.float32(v)) for v in w.force))
        o = oracle.from_workload(w64, oracle.FP64, oracle.ARITH_F64)
    else:
        o = oracle.from_workload(w, FORMATS[name])
    o.step(steps)
    for i in range(q):
        assert np.array_equal(s.read_ddf(i), o.read_ddf(i)), (name, i)
    if name != "FP64":
        srho, su = s.read_rho_u()
        orho, ou = o.read_rho_u()
        assert np.array_equal(srho.view(np.uint32), orho.view(np.uint32)) and np.array_equal(su.view(np.uint32), ou.view(np.uint32))
    s.close()


def test_slabs_staged_kernel_cavity():
    """slabs large enough for the staged kernel (2^20 cells each), lid and walls: against the undecomposed GPU run"""
    w = wl.lid_driven_cavity(128)
    steps = 6
    g = lbm.from_workload(w, "FP16S")
    g.step(steps)
    s = _run(w, "FP16S", 2, steps)
    assert "staged" in s.slabs[0].sim.kernel_name
    for i in range(19):
        assert np.array_equal(s.read_ddf(i), g.read_ddf(i)), i
    s.close()
    g.close()
