"""GPU parity of the FP64-arithmetic formats (the paper's FP64/FP64 and FP64/FP32
columns; FP64 storage of BASELINE config 5) through the C ABI vs the oracle run with
`arith = ORC_ARITH_F64` on the same seeded inputs.

Bar: north_star's 1e-6 on rho and u -- and, because the kernels repeat the oracle's IEEE binary64 operations in
the same order (--fmad=false, explicit fma, IEEE division), the stronger property: every stored DDF, and rho, u
read out in double, are bit for bit the oracle's.

tau and the body force cross the C ABI as floats (include/lbm.h) and are widened exactly; the oracle's FP64 mode
takes doubles, so the tests hand it the float-rounded values.
"""
import dataclasses

import numpy as np
import pytest

import oracle
import paper_2112_08926_b200 as lbm
import workloads as wl

pytestmark = pytest.mark.gpu

# product format name -> (oracle storage format, element view for bit comparison)
F64_FORMATS = {"FP64": (oracle.FP64, np.uint64), "FP64_FP32": (oracle.FP32, np.uint32)}


def f32_params(w):
    """tau and force as the product sees them: rounded once to float32."""
    return dataclasses.replace(w, tau=float(np.float32(w.tau)), force=tuple(float(np.float32(v)) for v in w.force))


def run_pair(w, name, steps):
    w = f32_params(w)
    osim = oracle.from_workload(w, F64_FORMATS[name][0], oracle.ARITH_F64)
    gsim = lbm.from_workload(w, name)
    assert "stream_collide64" in gsim.kernel_name
    osim.step(steps)
    gsim.step(steps)
    return osim, gsim


def assert_parity(osim, gsim, name):
    view = F64_FORMATS[name][1]
    for i in range(osim.q):
        a, b = gsim.read_ddf(i), osim.read_ddf(i)
        assert a.dtype == b.dtype
        assert np.array_equal(a.view(view), b.view(view)), (name, "direction", i)
    orho, ou = osim.read_rho_u(f64=True)
    grho, gu = gsim.read_rho_u_f64()
    assert np.all(np.isfinite(grho)) and np.all(np.isfinite(gu))
    assert np.abs(grho - orho).max() <= 1e-6 and np.abs(gu - ou).max() <= 1e-6 * max(np.abs(ou).max(), 1e-30)
    assert np.array_equal(grho.view(np.uint64), orho.view(np.uint64))
    assert np.array_equal(gu.view(np.uint64), ou.view(np.uint64))
    # the float read-out is the double one rounded to nearest
    orho32, ou32 = osim.read_rho_u()
    grho32, gu32 = gsim.read_rho_u()
    assert np.array_equal(grho32.view(np.uint32), orho32.view(np.uint32))
    assert np.array_equal(gu32.view(np.uint32), ou32.view(np.uint32))


# ---- BASELINE config 1: Taylor-Green 32^3, 200 steps --------------------------------------------------
@pytest.mark.parametrize("name", list(F64_FORMATS))
def test_taylor_green_3d_config1(name):
    w = wl.taylor_green_3d(32)
    osim, gsim = run_pair(w, name, w.steps)
    assert gsim.steps_done == 200
    assert_parity(osim, gsim, name)


@pytest.mark.parametrize("name", list(F64_FORMATS))
def test_init_readout_without_steps(name):
    osim, gsim = run_pair(wl.taylor_green_3d(16), name, 0)
    assert_parity(osim, gsim, name)


# ---- velocity sets, ragged sizes (several CTAs + a tail, rows shorter than a warp) ---------------------
@pytest.mark.parametrize("q,shape", [(19, (37, 5, 3)), (19, (260, 3, 2)), (19, (2, 2, 2)), (19, (1, 1, 1)),
                                     (27, (24, 10, 6)), (27, (7, 3, 5)), (9, (48, 20, 1)), (9, (33, 9, 1)), (9, (1, 7, 1))])
@pytest.mark.parametrize("name", list(F64_FORMATS))
def test_periodic_shapes_and_velocity_sets(q, shape, name):
    w = wl.perturbed_equilibrium(*shape, seed=11, velset=q)
    osim, gsim = run_pair(w, name, 20)
    assert_parity(osim, gsim, name)


# ---- walls, moving walls, body force, equilibrium cells --------------------------------------------------
@pytest.mark.parametrize("q,shape", [(19, (24, 9, 7)), (27, (12, 8, 6)), (9, (40, 17, 1))])
@pytest.mark.parametrize("name", list(F64_FORMATS))
def test_random_walls_moving_walls_force(q, shape, name):
    w = wl.perturbed_equilibrium(*shape, seed=3, velset=q, tau=0.7)
    w = wl.random_walls(w, 0.15, seed=9, moving_fraction=0.5)
    w.force = (1e-5, -2e-5, 0.0 if q == 9 else 3e-5)
    osim, gsim = run_pair(w, name, 30)
    assert_parity(osim, gsim, name)


@pytest.mark.parametrize("name", list(F64_FORMATS))
def test_equilibrium_rim(name):
    w = wl.equilibrium_rim(wl.perturbed_equilibrium(20, 11, 9, seed=4, tau=0.65))
    osim, gsim = run_pair(w, name, 25)
    assert_parity(osim, gsim, name)


@pytest.mark.parametrize("q,shape", [(19, (24, 9, 7)), (27, (12, 8, 6))])
@pytest.mark.parametrize("name", list(F64_FORMATS))
def test_outflow_cells(q, shape, name):
    """zero-gradient outflow cells (LBM_FLAG_OUT, R18) with an equilibrium inflow plane, walls and a force"""
    w = wl.perturbed_equilibrium(*shape, seed=41, velset=q, tau=0.75)
    w = wl.random_walls(w, 0.08, seed=43, moving_fraction=0.5)
    f = w.flags.reshape(w.nz, w.ny, w.nx).copy()
    f[:, :, 0] = lbm.FLAG_EQ
    f[:, :, -1] = lbm.FLAG_OUT
    w.flags = f.reshape(-1)
    w.force = (1e-5, 0.0, 0.0)
    osim, gsim = run_pair(w, name, 20)
    assert_parity(osim, gsim, name)


def test_all_cells_walls_is_a_noop():
    w = wl.perturbed_equilibrium(8, 4, 4, seed=1)
    w.flags[:] = wl.FLAG_WALL
    osim, gsim = run_pair(w, "FP64", 3)
    assert_parity(osim, gsim, "FP64")


# ---- BASELINE config 2 (prefix) and config 3 (the oracle-sized 32^3 copy, prefix) -------------------------
@pytest.mark.parametrize("name", list(F64_FORMATS))
def test_poiseuille_config2_prefix(name):
    osim, gsim = run_pair(wl.poiseuille_channel(), name, 1000)
    assert_parity(osim, gsim, name)


def test_lid_driven_cavity_config3_prefix():
    osim, gsim = run_pair(wl.lid_driven_cavity(32), "FP64", 300)
    assert_parity(osim, gsim, "FP64")


# ---- the API around the new formats ---------------------------------------------------------------------
def test_sizes_and_unsupported_calls():
    assert lbm.bytes_per_cell(19, "FP64") == 305           # 2 * 19 * 8 + 1
    assert lbm.bytes_per_cell(19, "FP64_FP32") == 153
    assert lbm.ddf_buffer_bytes(4, 4, 4, 19, "FP64") == (64 * 19 * 8 + 255) // 256 * 256
    w = wl.perturbed_equilibrium(16, 4, 4, seed=2)
    with pytest.raises(lbm.LbmError) as e:
        lbm.from_workload(w, "FP32").read_rho_u_f64()
    assert e.value.code == lbm.E_UNSUPPORTED
    with pytest.raises(lbm.LbmError) as e:
        lbm.from_workload(w, "FP64", variant=lbm.VARIANT_BULK)
    assert e.value.code == lbm.E_UNSUPPORTED
    g = lbm.from_workload(w, "FP64")
    cells = np.array([0, 5, 255, 17], np.int64)
    rho, u = g.read_rho_u()
    prho, pu = g.read_rho_u_at(cells)
    assert np.array_equal(prho, rho[cells]) and np.array_equal(pu, u[:, cells])


# ---- full size, in the launch configuration bench.py times (see test_gpu_lbm.py for the block argument) ----
FULL_L, FULL_STEPS, BLK = 512, 3, 14


def _block(field, origin, L):
    ix = [np.arange(o, o + BLK) % L for o in origin]
    return field[..., ix[2][:, None, None], ix[1][None, :, None], ix[0][None, None, :]]


@pytest.mark.parametrize("name", list(F64_FORMATS))
def test_full_size_sampled_blocks(name):
    L = FULL_L
    w = f32_params(wl.perturbed_equilibrium(L, L, L, seed=20211208, tau=0.6))
    g = lbm.from_workload(w, name)
    g.step(FULL_STEPS)
    grho, gu = g.read_rho_u_f64()
    g.close()
    assert np.all(np.isfinite(grho))
    grho = grho.reshape(L, L, L)
    gu = gu.reshape(3, L, L, L)
    rho0 = w.rho.reshape(L, L, L)
    u0 = w.u.reshape(3, L, L, L)
    rng = np.random.default_rng(6)
    origins = [(-7, -7, -7), (L - 7, 100, 200), (300, L - 7, 17), (40, 50, L - 7), (0, 0, 0)]
    origins += [tuple(int(v) for v in rng.integers(0, L, 3)) for _ in range(5)]
    c = slice(3, BLK - 3)
    for o in origins:
        sub = wl.Workload("block", BLK, BLK, BLK, 19, w.tau, np.ascontiguousarray(_block(rho0, o, L)).reshape(-1),
                          np.ascontiguousarray(_block(u0, o, L)).reshape(3, -1), np.zeros(BLK ** 3, np.uint8))
        osim = oracle.from_workload(sub, F64_FORMATS[name][0], oracle.ARITH_F64)
        osim.step(FULL_STEPS)
        orho, ou = osim.read_rho_u(f64=True)
        orho = orho.reshape(BLK, BLK, BLK)[c, c, c]
        ou = ou.reshape(3, BLK, BLK, BLK)[:, c, c, c]
        assert np.array_equal(_block(grho, o, L)[c, c, c].view(np.uint64), orho.view(np.uint64)), (name, o)
        assert np.array_equal(_block(gu, o, L)[:, c, c, c].view(np.uint64), ou.view(np.uint64)), (name, o)
