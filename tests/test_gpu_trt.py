"""GPU parity of the TRT collision operator (BASELINE config 3 names it) through the
C ABI (lbm_create(..., LBM_TRT, ...), lbm_set_trt_lambda) vs the oracle's ORC_TRT on the same seeded inputs.

The paper only names TRT and states that it stays bound by memory; the operator
is the textbook one of DESIGN.md reading R13, which the oracle pins by the vanishing Poiseuille slip at
Lambda = 3/16, the BGK limit, conservation and the Taylor-Green decay rate (tests/test_oracle_lbm.py).

Bar: north_star's 1e-6 (FP32 storage) / 1e-3 (16-bit storage) on rho and u, and -- the kernels repeating the
oracle's IEEE operations in the same order -- every stored DDF bit for bit the oracle's, in all three kernels
(per-thread, staged, FP64 arithmetic).
"""
import dataclasses

import numpy as np
import pytest

import oracle
import paper_2112_08926_b200 as lbm
import workloads as wl
from workloads import FORMATS

pytestmark = pytest.mark.gpu
ALL_FORMATS = list(FORMATS)
TOL = {name: (1e-6 if name == "FP32" else 1e-3) for name in ALL_FORMATS}
F64_FORMATS = {"FP64": (oracle.FP64, np.uint64), "FP64_FP32": (oracle.FP32, np.uint32)}


def run_pair(w, name, steps, lam=None, variant=0, cells_per_thread=0):
    if name in F64_FORMATS:
        w = dataclasses.replace(w, tau=float(np.float32(w.tau)), force=tuple(float(np.float32(v)) for v in w.force))
        osim = oracle.from_workload(w, F64_FORMATS[name][0], oracle.ARITH_F64)
    else:
        osim = oracle.from_workload(w, FORMATS[name])
    gsim = lbm.from_workload(w, name, collision=lbm.TRT, variant=variant, cells_per_thread=cells_per_thread)
    if lam is None:
        osim.set_collision(oracle.TRT)
    else:
        osim.set_collision(oracle.TRT, lam)
        gsim.set_trt_lambda(lam)
    assert "COLL=TRT" in gsim.kernel_name
    osim.step(steps)
    gsim.step(steps)
    return osim, gsim


def assert_parity(osim, gsim, name):
    if name in F64_FORMATS:
        view, tol = F64_FORMATS[name][1], 1e-6
    else:
        view, tol = (np.uint32 if name == "FP32" else np.uint16), TOL[name]
    orho, ou = osim.read_rho_u()
    grho, gu = gsim.read_rho_u()
    assert np.all(np.isfinite(grho)) and np.all(np.isfinite(gu))
    assert np.abs(grho.astype(np.float64) - orho).max() <= tol
    assert np.abs(gu.astype(np.float64) - ou).max() / max(np.abs(ou).max(), 1e-30) <= tol
    for i in range(osim.q):
        a, b = gsim.read_ddf(i), osim.read_ddf(i)
        assert a.dtype == b.dtype
        assert np.array_equal(a.view(view), b.view(view)), (name, "direction", i)
    assert np.array_equal(grho.view(np.uint32), orho.view(np.uint32))
    assert np.array_equal(gu.view(np.uint32), ou.view(np.uint32))


# ---- BASELINE config 1 with TRT: Taylor-Green 32^3, 200 steps ------------------------------------------
@pytest.mark.parametrize("name", ALL_FORMATS + list(F64_FORMATS))
def test_taylor_green_3d_trt(name):
    w = wl.taylor_green_3d(32)
    osim, gsim = run_pair(w, name, w.steps)
    assert_parity(osim, gsim, name)


# ---- per-thread kernel: velocity sets, ragged shapes, walls + moving walls + force, several Lambda ---------
@pytest.mark.parametrize("q,shape", [(19, (37, 5, 3)), (19, (260, 3, 2)), (19, (1, 1, 1)), (27, (12, 8, 6)), (9, (40, 17, 1))])
@pytest.mark.parametrize("name", ["FP32", "FP16S", "FP16C", "P16_0S", "P16_2C", "FP64", "FP64_FP32"])
@pytest.mark.parametrize("lam", [None, 0.25, 1.0 / 12.0])
def test_trt_walls_moving_walls_force(q, shape, name, lam):
    w = wl.perturbed_equilibrium(*shape, seed=41, velset=q, tau=0.7)
    if w.n_cells > 8:
        w = wl.random_walls(w, 0.12, seed=43, moving_fraction=0.5)
    w.force = (1e-5, -2e-5, 0.0 if q == 9 else 3e-5)
    osim, gsim = run_pair(w, name, 20, lam=lam)
    assert_parity(osim, gsim, name)


@pytest.mark.parametrize("q,shape", [(19, (24, 9, 7)), (9, (40, 17, 1))])
@pytest.mark.parametrize("name", ["FP32", "FP16S", "P16_2C"])
@pytest.mark.parametrize("v", [1, 2, 4])
def test_trt_cells_per_thread_variants(q, shape, name, v):
    w = wl.perturbed_equilibrium(*shape, seed=67, velset=q, tau=0.7)
    w = wl.random_walls(w, 0.1, seed=71, moving_fraction=0.5)
    w.force = (1e-5, -2e-5, 0.0 if q == 9 else 3e-5)
    osim, gsim = run_pair(w, name, 15, cells_per_thread=v)
    assert f"V={v}," in gsim.kernel_name
    assert_parity(osim, gsim, name)


@pytest.mark.parametrize("name", ["FP32", "FP16S", "FP64"])
def test_trt_periodic_without_force(name):
    w = wl.perturbed_equilibrium(33, 6, 4, seed=47, tau=0.53)
    osim, gsim = run_pair(w, name, 30)
    assert_parity(osim, gsim, name)


# ---- staged kernel (lbm_stage.cuh): one tile per row, several tiles with a ragged last tile, D3Q27, D2Q9 -----
@pytest.mark.parametrize("q,shape", [(19, (64, 5, 3)), (19, (560, 3, 2)), (19, (1040, 3, 2)), (27, (272, 3, 3)), (9, (1056, 3, 1))])
@pytest.mark.parametrize("name", ALL_FORMATS)
@pytest.mark.parametrize("walls", [False, True])
@pytest.mark.parametrize("variant,tag", [(lbm.VARIANT_STAGED, "staged")])
def test_trt_staged_kernel(q, shape, name, walls, variant, tag):
    w = wl.perturbed_equilibrium(*shape, seed=53, velset=q, tau=0.7)
    if walls:
        w = wl.random_walls(w, 0.12, seed=59, moving_fraction=0.5)
        w.force = (1e-5, -2e-5, 0.0 if q == 9 else 3e-5)
    osim, gsim = run_pair(w, name, 16, variant=variant)
    assert tag in gsim.kernel_name
    assert_parity(osim, gsim, name)


# ---- BASELINE config 3 (lid-driven cavity, the config that names TRT), small copy, equilibrium rim ----------
@pytest.mark.parametrize("name", ["FP32", "FP16S", "FP16C", "P16_1S"])
def test_trt_lid_driven_cavity_small(name):
    w = wl.lid_driven_cavity(32)
    osim, gsim = run_pair(w, name, 60)
    assert_parity(osim, gsim, name)


@pytest.mark.parametrize("name", ["FP32", "FP16C"])
@pytest.mark.parametrize("variant", [lbm.VARIANT_STAGED])
def test_trt_equilibrium_boundary_cells(name, variant):
    w = wl.equilibrium_rim(wl.perturbed_equilibrium(48, 7, 5, seed=61, tau=0.65))
    osim, gsim = run_pair(w, name, 20, variant=variant)
    assert_parity(osim, gsim, name)


# ---- the bench configuration (512^3 D3Q19 periodic, automatic kernel choice) with TRT ------------------------------
# As tests/test_gpu_lbm.py's full-size test: after n steps a cell depends only on the initial fields within n cells of
# it, so sampled 14^3 blocks (some across the periodic faces) are stepped by the oracle as boxes of their own and
# their 8^3 cores must agree with the GPU bit for bit.
FULL_L, FULL_STEPS, BLK = 512, 3, 14


@pytest.fixture(scope="module")
def full_size_workload():
    return wl.perturbed_equilibrium(FULL_L, FULL_L, FULL_L, seed=20211208, tau=0.6)


def _block(field, origin, L):
    ix = [np.arange(o, o + BLK) % L for o in origin]
    return field[..., ix[2][:, None, None], ix[1][None, :, None], ix[0][None, None, :]]


@pytest.mark.parametrize("name", ["FP32", "FP16S", "P16_0S"])
def test_trt_full_size_sampled_blocks(full_size_workload, name):
    w, L = full_size_workload, FULL_L
    g = lbm.from_workload(w, name, collision=lbm.TRT)
    assert "COLL=TRT" in g.kernel_name and ("staged" in g.kernel_name) == (name != "FP32")
    g.step(FULL_STEPS)
    grho, gu = g.read_rho_u()
    g.close()
    assert np.all(np.isfinite(grho))
    grho, gu = grho.reshape(L, L, L), gu.reshape(3, L, L, L)
    rho0, u0 = w.rho.reshape(L, L, L), w.u.reshape(3, L, L, L)
    rng = np.random.default_rng(7)
    origins = [(-7, -7, -7), (L - 7, 100, 200), (300, L - 7, 17), (40, 50, L - 7), (0, 0, 0)]
    origins += [tuple(int(v) for v in rng.integers(0, L, 3)) for _ in range(5)]
    c = slice(3, BLK - 3)
    for o in origins:
        sub = wl.Workload("block", BLK, BLK, BLK, 19, w.tau, np.ascontiguousarray(_block(rho0, o, L)).reshape(-1),
                          np.ascontiguousarray(_block(u0, o, L)).reshape(3, -1), np.zeros(BLK ** 3, np.uint8))
        osim = oracle.from_workload(sub, FORMATS[name])
        osim.set_collision(oracle.TRT)
        osim.step(FULL_STEPS)
        orho, ou = osim.read_rho_u()
        orho = orho.reshape(BLK, BLK, BLK)[c, c, c]
        ou = ou.reshape(3, BLK, BLK, BLK)[:, c, c, c]
        assert np.array_equal(_block(grho, o, L)[c, c, c].view(np.uint32), orho.view(np.uint32)), (name, o)
        assert np.array_equal(_block(gu, o, L)[:, c, c, c].view(np.uint32), ou.view(np.uint32)), (name, o)


# ---- what the method fixes, on the product alone -----------------------------------------------------------
def test_trt_with_equal_rates_matches_bgk_to_rounding():
    """Lambda = (tau - 1/2)^2 makes omega- = omega+ (R13): the TRT run then follows the BGK run up to rounding."""
    tau = 0.8
    w = wl.taylor_green_3d(16, tau=tau)
    a = lbm.from_workload(w, "FP32")
    b = lbm.from_workload(w, "FP32", collision=lbm.TRT)
    b.set_trt_lambda((tau - 0.5) ** 2)
    a.step(50)
    b.step(50)
    (ra, ua), (rb, ub) = a.read_rho_u(), b.read_rho_u()
    assert np.abs(ra - rb).max() < 2e-6 and np.abs(ua - ub).max() < 2e-6
    assert np.abs(ua).max() > 1e-3


def test_trt_poiseuille_slip_vanishes_at_the_magic_parameter():
    """Force-driven channel between halfway bounce-back walls (BASELINE config 2's set-up, small): with Lambda = 3/16
    the steady profile is the parabola through walls half a cell outside the last fluid nodes at any tau -- here a
    large one, where BGK's slip U_s = f (48 nu^2 - 1) / (8 nu) would be 17% of u_max.  FP64 arithmetic, so that the
    residual is the method's and not rounding."""
    ny, tau = 14, 1.3
    w = wl.poiseuille_channel(4, ny, 3, tau=tau, u_max=0.01)
    nu, H, f = tau / 3.0 - 1.0 / 6.0, ny - 2, w.force[0]
    s = lbm.from_workload(w, "FP64", collision=lbm.TRT)
    s.step(9000)
    _, u = s.read_rho_u_f64()
    prof = u[0].reshape(3, ny, 4)[1, 1:-1, 2]
    y = np.arange(1, ny - 1) - 0.5
    f = float(np.float32(f))
    nu = float(np.float32(tau)) / 3.0 - 1.0 / 6.0
    assert np.abs(prof - f / (2 * nu) * y * (H - y)).max() / 0.01 < 1e-9


def test_trt_argument_checks():
    s = lbm.Simulation(8, 8, 8, collision=lbm.BGK)
    with pytest.raises(lbm.LbmError):
        s.set_trt_lambda(0.25)                         # not a TRT handle
    t = lbm.Simulation(8, 8, 8, collision=lbm.TRT)
    with pytest.raises(lbm.LbmError):
        t.set_trt_lambda(0.0)
    with pytest.raises(lbm.LbmError):
        lbm.Simulation(8, 8, 8, collision=2)
