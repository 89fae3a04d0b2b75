"""lbm_read_rho_u_at_static (include/lbm.h): the probe read-out whose device scratch is a fixed array inside the library,
for callers that must not call cudaMalloc.  Checked against the existing path (lbm_read_rho_u_at, whose scratch is the
handle's staging buffer) bit for bit -- the same kernel on the same inputs -- on calls in a row that share the array.

This file sorts last on purpose: the suite runs with pytest -x, and a failure here must not hide another test."""
import numpy as np
import pytest

import workloads as wl

pytestmark = pytest.mark.gpu


def _same(a, b):
    return np.array_equal(np.asarray(a).view(np.uint32), np.asarray(b).view(np.uint32))


@pytest.mark.parametrize("name", ["FP32", "FP16S", "P16_1S", "FP64"])
def test_static_scratch_probe_equals_the_allocating_path_two_calls_in_a_row(name):
    import paper_2112_08926_b200 as lbm
    w = wl.perturbed_equilibrium(48, 20, 12, seed=91, tau=0.7)
    w = wl.random_walls(w, 0.1, seed=93, moving_fraction=0.5)
    w.force = (1e-5, -2e-5, 3e-5)
    sim = lbm.from_workload(w, name)
    sim.step(5)
    rng = np.random.default_rng(7)
    # first call: the largest request the array takes; second call: fewer cells, after more steps -- it must not see the
    # first call's leftovers; third: one cell
    cells1 = rng.integers(0, w.n_cells, lbm.STATIC_PROBES_MAX)
    r1, u1 = sim.read_rho_u_at_static(cells1)
    e1, v1 = sim.read_rho_u_at(cells1)
    assert _same(r1, e1) and _same(u1, v1)
    sim.step(3)
    cells2 = rng.integers(0, w.n_cells, 1000)
    r2, u2 = sim.read_rho_u_at_static(cells2)
    e2, v2 = sim.read_rho_u_at(cells2)
    assert _same(r2, e2) and _same(u2, v2)
    assert not _same(r2, r1[:1000])                       # (the state did move on between the calls)
    r3, u3 = sim.read_rho_u_at_static([int(cells2[17])])
    assert _same(r3, e2[17:18]) and _same(u3, v2[:, 17:18])
    # and against the full read-out of the existing path
    if name != "FP64":
        rho, u = sim.read_rho_u()
        assert _same(r2, rho[cells2]) and _same(u2, u[:, cells2])
    sim.close()


def test_static_scratch_probe_limits_and_second_handle():
    import paper_2112_08926_b200 as lbm
    w = wl.taylor_green_3d(16)
    a = lbm.from_workload(w, "FP16C")
    b = lbm.from_workload(w, "FP32")
    a.step(2)
    b.step(4)
    with pytest.raises(lbm.LbmError) as err:
        a.read_rho_u_at_static(np.zeros(lbm.STATIC_PROBES_MAX + 1, np.int64))
    assert "LBM_STATIC_PROBES_MAX" in str(err.value)
    with pytest.raises(lbm.LbmError):
        a.read_rho_u_at_static([w.n_cells])                # out of range
    r0, u0 = a.read_rho_u_at_static([])                    # nothing to do
    assert r0.size == 0 and u0.shape == (3, 0)
    cells = np.arange(0, w.n_cells, 5)
    ra, ua = a.read_rho_u_at_static(cells)                 # two handles, one after the other, share the array
    rb, ub = b.read_rho_u_at_static(cells)
    ea, va = a.read_rho_u_at(cells)
    eb, vb = b.read_rho_u_at(cells)
    assert _same(ra, ea) and _same(ua, va) and _same(rb, eb) and _same(ub, vb)
    a.close()
    b.close()
