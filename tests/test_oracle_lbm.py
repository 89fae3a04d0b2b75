"""Pins for the oracle's LBM step (oracle/lbm.cpp) -- CPU only.

Checked against what the paper and the mathematics fix, not against the oracle itself:
  * Table 1 (tests/golden/table1_delta.txt)            -> velocity sets, weights, eq (3)
  * moment identities of the equilibrium (eq (2)-(4))
  * exact mass conservation on periodic boxes (eq (25)-(28))
  * fixed points: fluid at rest, uniform flow
  * Taylor-Green closed form, eqs (15)-(18)
  * planar Poiseuille: exact steady solution of BGK + halfway bounce-back + Guo forcing (eq (9), (13))
  * planar Couette: exact linear profile (pins the moving-wall term)
  * a second, differently built implementation (push streaming on UNshifted DDFs, eqs (19)-(23),
    PAPER.md:651-667, numpy in float64) on tiny boxes with walls, moving walls and a force
  * mirror / axis-permutation symmetry, velocity clamp
"""
import math
import os

import numpy as np
import pytest

import oracle
import workloads as wl

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
F64 = oracle.ARITH_F64


def sim64(w):
    s = oracle.Sim(w.nx, w.ny, w.nz, w.velset, oracle.FP64, w.tau, w.force, F64)
    s.set_flags(w.flags)
    s.init(w.rho.astype(np.float64), w.u.astype(np.float64))
    return s


# ------------------------------------------------------------------------------------------------
def test_table1_number_range():
    names = {"D2Q9": 9, "D3Q19": 19, "D3Q27": 27}
    for line in open(os.path.join(GOLDEN, "table1_delta.txt")):
        if line.startswith("#") or not line.strip():
            continue
        name, d, ds = line.split()
        q = names[name]
        c, w, opp = oracle.velocity_set(q)
        cs = 1.0 / math.sqrt(3.0)
        us = [np.zeros(3)] + [cs * c[j] / np.linalg.norm(c[j]) for j in range(1, q)]
        delta = delta_s = 0.0
        for u in us:
            fs = oracle.equilibrium(q, 1.0, *u)
            delta_s = max(delta_s, np.abs(fs).max())
            delta = max(delta, np.abs(fs + w).max())
        # "rounded up to 2 digits" reproduces the printed table
        assert math.ceil(delta * 100 - 1e-9) / 100 == pytest.approx(float(d)), (name, delta)
        assert math.ceil(delta_s * 100 - 1e-9) / 100 == pytest.approx(float(ds)), (name, delta_s)


@pytest.mark.parametrize("q", [9, 19, 27])
def test_velocity_set_and_equilibrium_moments(q):
    c, w, opp = oracle.velocity_set(q)
    assert w.sum() == pytest.approx(1.0, abs=1e-15)
    assert np.array_equal(c[opp], -c) and opp[0] == 0               # (i, i+1) opposite
    assert len({tuple(r) for r in c.tolist()}) == q
    # lattice isotropy: sum w c_a c_b = c^2 delta_ab, c^2 = 1/3
    assert np.allclose(np.einsum("i,ia,ib->ab", w, c, c), np.eye(3)[: , :] / 3 * (np.abs(c).sum(0) > 0)[None, :] * (np.abs(c).sum(0) > 0)[:, None], atol=1e-15)
    if q == 19:
        # numbering printed in the momentum sums, PAPER.md:62 / 955-959
        assert [i for i in range(q) if c[i, 0] == 1] == [1, 7, 9, 13, 15]
        assert [i for i in range(q) if c[i, 1] == 1] == [3, 7, 11, 14, 17]
        assert [i for i in range(q) if c[i, 2] == 1] == [5, 9, 11, 16, 18]
    rng = np.random.default_rng(0)
    for _ in range(20):
        rho = 1 + 0.1 * rng.standard_normal()
        u = 0.1 * rng.uniform(-1, 1, 3)
        if q == 9:
            u[2] = 0
        f = oracle.equilibrium(q, rho, *u) + w                      # unshifted, eq (1)
        assert f.sum() == pytest.approx(rho, abs=1e-14)             # eq (4)
        assert np.allclose(f @ c, rho * u, atol=1e-15)
        P = np.einsum("i,ia,ib->ab", f, c, c)
        want = rho * (np.eye(3) / 3 + np.outer(u, u))
        if q == 9:
            want[2, :] = want[:, 2] = 0
        assert np.allclose(P, want, atol=1e-15)                     # second moment of eq (2)
    # float arithmetic follows the same formula: agrees with double to FP32 rounding
    f32 = oracle.equilibrium(q, 1.01, 0.03, -0.02, 0.0 if q == 9 else 0.01, arith=oracle.ARITH_F32)
    f64 = oracle.equilibrium(q, np.float32(1.01), np.float32(0.03), np.float32(-0.02),
                             0.0 if q == 9 else np.float32(0.01))
    assert np.allclose(f32, f64, rtol=0, atol=3e-8)


# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("q,shape", [(19, (12, 10, 8)), (27, (8, 8, 6)), (9, (16, 12, 1))])
def test_mass_and_momentum_conservation_periodic(q, shape):
    w = wl.perturbed_equilibrium(*shape, seed=3, velset=q, rho_sigma=1e-2)
    s = sim64(w)
    rho0, u0 = s.read_rho_u(f64=True)
    m0 = s.sum_ddf()
    p0 = (rho0[None] * u0).sum(1)
    s.step(200)
    rho1, u1 = s.read_rho_u(f64=True)
    assert abs(s.sum_ddf() - m0) / w.n_cells < 1e-14                # mass M = N + sum f_shifted
    assert abs(rho1.sum() - rho0.sum()) / rho0.sum() < 1e-14
    assert np.allclose((rho1[None] * u1).sum(1), p0, rtol=0, atol=1e-12)
    # FP32 arithmetic + FP32 storage: conserved to FP32 rounding
    s32 = oracle.from_workload(w, oracle.FP32)
    r0, _ = s32.read_rho_u()
    s32.step(200)
    r1, _ = s32.read_rho_u()
    assert abs(r1.astype(np.float64).sum() - r0.astype(np.float64).sum()) / w.n_cells < 1e-6


@pytest.mark.parametrize("name", list(wl.FORMATS))
def test_rest_state_is_a_fixed_point_in_every_format(name):
    n = 6
    w = wl.taylor_green_3d(n)
    w.u[:] = 0
    s = oracle.from_workload(w, wl.FORMATS[name])
    s.step(5)
    for i in range(19):
        raw = s.read_ddf(i)
        if name == "FP32":
            assert np.all(raw == 0)
        else:
            assert np.all((raw & 0x7FFF) == 0)                      # +-0 codes only
    rho, u = s.read_rho_u()
    assert np.all(rho == 1) and np.all(u == 0)


def test_uniform_flow_stays_uniform():
    w = wl.taylor_green_3d(6)
    w.rho[:] = 1.02
    w.u[0], w.u[1], w.u[2] = 0.03, -0.02, 0.01
    s = sim64(w)
    s.step(50)
    rho, u = s.read_rho_u(f64=True)
    assert np.allclose(rho, np.float32(1.02), atol=1e-14)
    for a in range(3):
        assert np.allclose(u[a], w.u[a, 0].astype(np.float64), atol=1e-14)


# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("q,nz", [(9, 1), (19, 3)])
def test_taylor_green_2d_closed_form(q, nz):
    """eqs (15)-(18): u decays as exp(-2 nu k^2 t), E as exp(-4 nu k^2 t), vortices stay in place."""
    n, u0, tau = 32, 0.05, 0.6
    w = wl.taylor_green_2d(n, n, nz, u0=u0, tau=tau, velset=q, with_density=True)
    nu = tau / 3 - 1 / 6
    k = 2 * math.pi / n
    s = oracle.Sim(n, n, nz, q, oracle.FP64, tau, None, F64)
    s.init(w.rho.astype(np.float64), w.u.astype(np.float64))
    E = {}
    for t in (0, 50, 100, 200):
        if t:
            s.step(50 if t <= 100 else 100)
        rho, u = s.read_rho_u(f64=True)
        E[t] = 0.5 * (rho * (u[0] ** 2 + u[1] ** 2 + u[2] ** 2)).sum()
        # shape preserved: u(t) is the initial field times one scalar
        amp = (u[0] * w.u[0]).sum() / (w.u[0].astype(np.float64) ** 2).sum()
        assert np.abs(u[0] - amp * w.u[0]).max() < 2e-3 * u0
        assert amp == pytest.approx(math.exp(-2 * nu * k * k * t), rel=6e-3)
        assert np.abs(u[2]).max() < 1e-15
    for t in (50, 100, 200):
        assert E[t] / E[0] == pytest.approx(math.exp(-4 * nu * k * k * t), rel=1.2e-2)
    # decay RATE between t = 50 and t = 200 (independent of initialisation transients)
    rate = -math.log(E[200] / E[50]) / 150
    assert rate == pytest.approx(4 * nu * k * k, rel=5e-3)


def test_taylor_green_3d_sanity_band():
    """config 1: not an exact Navier-Stokes solution; Stokes-limit decay exp(-2 nu |k|^2 t), |k|^2 = 3 k^2."""
    w = wl.taylor_green_3d(32)
    s = sim64(w)
    nu = w.tau / 3 - 1 / 6
    k2 = 3 * w.meta["k"] ** 2
    rho, u = s.read_rho_u(f64=True)
    E0 = 0.5 * (rho * (u ** 2).sum(0)).sum()
    s.step(100)
    rho, u = s.read_rho_u(f64=True)
    E = 0.5 * (rho * (u ** 2).sum(0)).sum()
    ratio = (E / E0) / math.exp(-2 * nu * k2 * 100)
    assert 0.90 < ratio < 1.0


# ------------------------------------------------------------------------------------------------
def test_poiseuille_exact_steady_state():
    """BGK + halfway bounce-back + Guo forcing has an exact steady solution in a planar channel:
    the parabola of eq (9) (planar form f/(2 nu) y (H - y), walls half a cell outside the first
    fluid node) plus the constant slip U_s = f (48 nu^2 - 1) / (8 nu) (He et al. 1997)."""
    ny, tau, u_max = 18, 0.8, 0.01
    w = wl.poiseuille_channel(4, ny, 3, tau=tau, u_max=u_max)
    nu, H, f = w.meta["nu"], w.meta["H"], w.force[0]
    s = sim64(w)
    s.step(12000)
    rho, u = s.read_rho_u(f64=True)
    ux = u[0].reshape(3, ny, 4)
    assert np.abs(ux - ux[0:1, :, 0:1]).max() < 1e-15               # x- and z-invariant
    prof = ux[1, 1:-1, 2]
    y = np.arange(1, ny - 1) - 0.5
    exact = f / (2 * nu) * y * (H - y) + f * (48 * nu * nu - 1) / (8 * nu)
    assert np.abs(prof - exact).max() / u_max < 1e-10
    assert np.abs(u[1]).max() < 1e-15 and np.abs(u[2]).max() < 1e-15
    # eq (14) L2 error against the plain parabola = the slip, small but not zero
    par = f / (2 * nu) * y * (H - y)
    E = math.sqrt(((prof - par) ** 2).sum() / (par ** 2).sum())
    assert 1e-4 < E < 5e-3
    s.step(1)
    _, u2 = s.read_rho_u(f64=True)
    assert np.abs(u2 - u).max() < 1e-13                             # steady


def test_couette_exact_linear_profile():
    """Moving-wall bounce-back: a wall moving along x at y = ny-1 and a resting wall at
    y = 0 give the exact linear profile u_x = u_w (y - 1/2) / H, walls half-way."""
    ny, uw = 14, float(np.float32(0.05))       # the field is stored as float32
    w = wl.poiseuille_channel(3, ny, 4, tau=0.9)
    w.force = (0.0, 0.0, 0.0)
    uu = w.u.reshape(3, 4, ny, 3)
    uu[0, :, ny - 1, :] = uw
    s = sim64(w)
    s.step(8000)
    rho, u = s.read_rho_u(f64=True)
    prof = u[0].reshape(4, ny, 3)[2, 1:-1, 1]
    y = np.arange(1, ny - 1) - 0.5
    assert np.abs(prof - uw * y / (ny - 2)).max() < 1e-12
    assert np.allclose(rho.reshape(4, ny, 3)[:, 1:-1], 1.0, atol=1e-12)
    # wall cells read back the fields given to init
    assert np.all(u[0].reshape(4, ny, 3)[:, ny - 1, :] == np.float32(uw))


# ------------------------------------------------------------------------------------------------
def _reference_push_unshifted(w, steps):
    """Second implementation, built differently: UNshifted DDFs, eq (22) equilibrium typed in its plain
    form, collide-then-PUSH streaming with np.roll, halfway bounce-back applied on the pushed field,
    float64.  Returns (rho, u) with the oracle's read-out convention (moments of the post-collision
    state, u without the half-force for the physical field: (j - F/2)/rho)."""
    c, wts, opp = oracle.velocity_set(w.velset)
    q = len(wts)
    shape = (w.nz, w.ny, w.nx)
    rho = w.rho.astype(np.float64).reshape(shape)
    u = w.u.astype(np.float64).reshape((3,) + shape)
    wall = (w.flags.reshape(shape) & wl.FLAG_WALL) != 0
    eqb = (w.flags.reshape(shape) & wl.FLAG_EQ) != 0                 # equilibrium boundary cells (R15)
    outb = (w.flags.reshape(shape) & wl.FLAG_OUT) != 0               # zero-gradient outflow cells (R18)
    F = np.array(w.force, np.float64)
    omega = 1.0 / w.tau

    def feq(rho, u):
        uu = (u ** 2).sum(0)
        out = np.empty((q,) + shape)
        for i in range(q):
            cu = c[i, 0] * u[0] + c[i, 1] * u[1] + c[i, 2] * u[2]
            out[i] = wts[i] * rho * (4.5 * cu * cu + 3.0 * cu + 1.0 - 1.5 * uu)      # eq (22), c^2 = 1/3
        return out

    f = feq(rho, u)                                                  # post-"collision" state at t = 0
    f_imposed = f.copy()
    uw = np.where(wall[None], u, 0.0)
    cs = 1 / math.sqrt(3)
    for _ in range(steps):
        # push: population i of cell x moves to x + c_i  (axis order z, y, x)
        g = np.empty_like(f)
        for i in range(q):
            moved = np.roll(f[i], shift=(c[i, 2], c[i, 1], c[i, 0]), axis=(0, 1, 2))
            from_wall = np.roll(wall, shift=(c[i, 2], c[i, 1], c[i, 0]), axis=(0, 1, 2))
            uw_src = np.roll(uw, shift=(c[i, 2], c[i, 1], c[i, 0]), axis=(1, 2, 3))
            cuw = c[i, 0] * uw_src[0] + c[i, 1] * uw_src[1] + c[i, 2] * uw_src[2]
            bounced = f[opp[i]] + 6.0 * wts[i] * cuw                 # reflected at the half-way wall
            g[i] = np.where(from_wall, bounced, moved)
        rho_n = g.sum(0)
        j = np.einsum("ia,i...->a...", c.astype(np.float64), g)
        un = (j + 0.5 * F[:, None, None, None]) / rho_n
        un = np.clip(un, -cs, cs)
        fe = feq(rho_n, un)
        new = (1 - omega) * g + omega * fe
        if np.any(F != 0):
            for i in range(q):
                cu = c[i, 0] * un[0] + c[i, 1] * un[1] + c[i, 2] * un[2]
                cF = c[i] @ F
                uF = un[0] * F[0] + un[1] * F[1] + un[2] * F[2]
                new[i] += (1 - 0.5 * omega) * wts[i] * (3 * (cF - uF) + 9 * cu * cF)
        if outb.any():
            # outflow cells: equilibrium of the upstream (x - 1) neighbour's state before this step
            rho_up = np.roll(f.sum(0), 1, axis=2)
            j_up = np.roll(np.einsum("ia,i...->a...", c.astype(np.float64), f), 1, axis=3)
            new = np.where(outb[None], feq(rho_up, (j_up - 0.5 * F[:, None, None, None]) / rho_up), new)
        f = np.where(wall[None], f, new)                             # wall cells are never updated
        f = np.where(eqb[None], f_imposed, f)                        # E cells are reset to their imposed equilibrium
    rho_o = f.sum(0)
    j = np.einsum("ia,i...->a...", c.astype(np.float64), f)
    u_o = (j - 0.5 * F[:, None, None, None]) / rho_o
    rho_o = np.where(wall | eqb, rho, rho_o)
    u_o = np.where((wall | eqb)[None], u, u_o)
    return rho_o.reshape(-1), u_o.reshape(3, -1)


@pytest.mark.parametrize("q,shape,force", [
    (19, (5, 4, 6), (0.0, 0.0, 0.0)),
    (19, (6, 5, 4), (1e-4, -2e-4, 3e-4)),
    (27, (4, 5, 4), (2e-4, 0.0, -1e-4)),
    (9, (7, 6, 1), (1e-4, 2e-4, 0.0)),
])
def test_against_push_unshifted_reference(q, shape, force):
    w = wl.perturbed_equilibrium(*shape, seed=11, velset=q, rho_sigma=1e-2, tau=0.7)
    w = wl.random_walls(w, 0.15, seed=5, moving_fraction=0.5)
    w.force = force
    s = sim64(w)
    steps = 7
    s.step(steps)
    rho, u = s.read_rho_u(f64=True)
    rref, uref = _reference_push_unshifted(w, steps)
    assert np.abs(rho - rref).max() < 5e-14
    assert np.abs(u - uref).max() < 5e-14


@pytest.mark.parametrize("q,shape", [(19, (7, 6, 5)), (27, (6, 6, 4)), (9, (8, 7, 1))])
def test_equilibrium_boundaries_against_push_reference(q, shape):
    """R15: equilibrium boundary cells, walls and moving walls together, vs the second implementation (which
    resets E cells to their imposed equilibrium after every step)."""
    w = wl.perturbed_equilibrium(*shape, seed=13, velset=q, rho_sigma=1e-2, tau=0.8)
    w = wl.random_walls(w, 0.1, seed=6, moving_fraction=0.5)
    w = wl.equilibrium_rim(w, rho_e=1.01)
    s = sim64(w)
    s.step(9)
    rho, u = s.read_rho_u(f64=True)
    rref, uref = _reference_push_unshifted(w, 9)
    assert np.abs(rho - rref).max() < 5e-14
    assert np.abs(u - uref).max() < 5e-14


def test_equilibrium_perimeter_drives_the_box_to_its_velocity():
    """A box whose x / y perimeter imposes (rho, u) by equilibrium cells and whose fluid starts at
    rest ends in the uniform state (rho, u): E cells feed the flow (they are not walls) and uniform flow is the
    fixed point; started in that state it stays there to rounding."""
    ue = (0.04, -0.02, 0.0)
    w = wl.perturbed_equilibrium(10, 9, 2, seed=3, rho_sigma=0.0, u_abs_max=0.0, tau=0.9)
    w = wl.equilibrium_rim(w, rho_e=1.0, u_e=ue)
    fluid = w.flags == 0
    s = sim64(w)
    s.step(3000)
    rho, u = s.read_rho_u(f64=True)
    for a in range(3):
        assert np.abs(u[a][fluid] - np.float32(ue[a])).max() < 1e-9
    assert np.abs(rho[fluid] - 1.0).max() < 1e-9
    w.u = np.tile(np.array(ue, np.float32)[:, None], (1, w.n_cells))
    s = sim64(w)
    s.step(50)
    rho, u = s.read_rho_u(f64=True)
    assert np.abs(u[0] - np.float32(ue[0])).max() < 1e-14 and np.abs(rho - 1.0).max() < 1e-14


def test_axis_permutation_symmetry():
    """Swapping the roles of x and y in the input must swap them in the output (catches a wrong
    direction vector, opposite index or weight)."""
    n = 8
    w = wl.perturbed_equilibrium(n, n, n, seed=2, rho_sigma=1e-2)
    w = wl.random_walls(w, 0.1, seed=9, moving_fraction=0.5)
    w.force = (1e-4, 2e-4, -1e-4)
    s = sim64(w)
    s.step(10)
    rho, u = s.read_rho_u(f64=True)
    # transposed problem: (x, y) -> (y, x)
    w2 = wl.perturbed_equilibrium(n, n, n, seed=2, rho_sigma=1e-2)
    T = lambda a: a.reshape(n, n, n).transpose(0, 2, 1).reshape(-1)
    w2.rho = T(w.rho).copy()
    w2.flags = T(w.flags).copy()
    w2.u = np.stack([T(w.u[1]), T(w.u[0]), T(w.u[2])]).copy()
    w2.force = (w.force[1], w.force[0], w.force[2])
    s2 = sim64(w2)
    s2.step(10)
    rho2, u2 = s2.read_rho_u(f64=True)
    assert np.abs(T(rho2) - rho).max() < 1e-14
    assert np.abs(T(u2[1]) - u[0]).max() < 1e-14 and np.abs(T(u2[0]) - u[1]).max() < 1e-14
    assert np.abs(T(u2[2]) - u[2]).max() < 1e-14


def test_velocity_clamp():
    """u is limited to +-c = 1/sqrt(3) before the equilibrium."""
    w = wl.taylor_green_3d(4, tau=1.0)
    w.u[:] = 0
    w.u[0] = 0.9
    s = sim64(w)
    s.step(1)                       # tau = 1: post-collision state = equilibrium of the clamped velocity
    rho, u = s.read_rho_u(f64=True)
    assert np.allclose(u[0], 1 / math.sqrt(3), atol=1e-15)


def test_storage_formats_track_fp64_on_taylor_green():
    """Accuracy ordering the paper reports (Fig. 8): with DDF-shifting every 16-bit format
    follows the FP64 energy decay at early times; FP32 storage is far closer than any 16-bit format."""
    w = wl.taylor_green_3d(16)
    ref = sim64(w)
    ref.step(40)
    _, uref = ref.read_rho_u(f64=True)
    err = {}
    for name, fmt in wl.FORMATS.items():
        s = oracle.from_workload(w, fmt)
        s.step(40)
        _, u = s.read_rho_u()
        err[name] = np.abs(u - uref).max() / np.abs(uref).max()
    assert err["FP32"] < 1e-5
    for name in wl.FORMATS_16BIT:
        assert err["FP32"] < err[name] < 2e-2, (name, err)
    assert err["FP16C"] < err["FP16S"]                               # one more mantissa bit


def test_fp64_arithmetic_with_fp32_storage_mode():
    """The paper's FP64/FP32 column (arithmetic / storage): the oracle's arith = F64, fmt = FP32
    mode is the FP64 step with one rounding to float per stored DDF.  Pins: (a) after init its stored DDFs are exactly
    the FP64/FP64 ones rounded to nearest float; (b) over a run it stays closer to
    FP64/FP64 than FP32/FP32 does (FP32 arithmetic adds its own rounding, Fig. 8) and mass is conserved to the
    storage rounding."""
    w = wl.taylor_green_3d(16)
    ref = sim64(w)
    mix = oracle.from_workload(w, oracle.FP32, F64)
    f32 = oracle.from_workload(w, oracle.FP32)
    for i in range(19):
        assert np.array_equal(mix.read_ddf(i), ref.read_ddf(i).astype(np.float32))
    m0 = mix.sum_ddf()
    ref.step(40); mix.step(40); f32.step(40)
    _, uref = ref.read_rho_u(f64=True)
    _, umix = mix.read_rho_u(f64=True)
    _, u32 = f32.read_rho_u()
    e_mix = np.abs(umix - uref).max() / np.abs(uref).max()
    e_32 = np.abs(u32 - uref).max() / np.abs(uref).max()
    assert e_mix < 1e-6 and e_mix <= e_32
    assert abs(mix.sum_ddf() - m0) < 40 * 19 * 16 ** 3 * 2.0 ** -36      # each store rounds |f| < 2^-11 to 2^-36 at worst


# ---- TRT (R13: textbook definition, NOT the paper's -- it only names the operator) --------------
def test_trt_magic_parameter_removes_the_poiseuille_slip():
    """With Lambda = 3/16 the halfway bounce-back wall of a force-driven planar channel sits exactly half a cell
    outside the first fluid node for every tau (Ginzburg & d'Humieres): the steady profile is the plain parabola
    of eq (9), no slip term -- where BGK has U_s = f (48 nu^2 - 1) / (8 nu) (test_poiseuille_exact_steady_state)."""
    for tau in (0.8, 1.3):
        ny, u_max = 18, 0.01
        w = wl.poiseuille_channel(4, ny, 3, tau=tau, u_max=u_max)
        nu, H, f = w.meta["nu"], w.meta["H"], w.force[0]
        s = sim64(w)
        s.set_collision(oracle.TRT, 3.0 / 16.0)
        s.step(14000)
        rho, u = s.read_rho_u(f64=True)
        prof = u[0].reshape(3, ny, 4)[1, 1:-1, 2]
        y = np.arange(1, ny - 1) - 0.5
        assert np.abs(prof - f / (2 * nu) * y * (H - y)).max() / u_max < 1e-10, tau
        assert np.abs(u[1]).max() < 1e-15 and np.abs(u[2]).max() < 1e-15
        assert np.abs(rho[w.flags == 0] - 1.0).max() < 1e-12


def test_trt_with_equal_rates_is_bgk():
    """Lambda = (tau - 1/2)^2 makes omega- = omega+: symmetric and antisymmetric parts relax alike, which is BGK
    (eq (28)), Guo source included -- with walls, moving walls and a force, to FP64 rounding."""
    tau = 0.7
    w = wl.random_walls(wl.perturbed_equilibrium(10, 7, 6, seed=2, tau=tau), 0.15, seed=4, moving_fraction=0.5)
    w.force = (1e-5, -2e-5, 3e-5)
    a, b = sim64(w), sim64(w)
    b.set_collision(oracle.TRT, (tau - 0.5) ** 2)
    a.step(30); b.step(30)
    for i in range(19):
        assert np.abs(a.read_ddf(i) - b.read_ddf(i)).max() < 1e-15, i


@pytest.mark.parametrize("q,shape", [(19, (8, 6, 5)), (27, (6, 5, 4)), (9, (12, 9, 1))])
def test_trt_conserves_mass_and_momentum_and_keeps_the_viscosity(q, shape):
    w = wl.perturbed_equilibrium(*shape, seed=8, velset=q, tau=0.9)
    s = sim64(w)
    s.set_collision(oracle.TRT)
    rho0, u0 = s.read_rho_u(f64=True)
    s.step(25)
    rho, u = s.read_rho_u(f64=True)
    assert abs(rho.sum() - rho0.sum()) < 1e-11
    assert np.abs((rho * u).sum(1) - (rho0 * u0).sum(1)).max() < 1e-12
    # the shear viscosity is set by omega+ alone: 2-D Taylor-Green decays as exp(-2 nu k^2 t), as with BGK
    n, tau = 32, 0.6
    w = wl.taylor_green_2d(n, n, 1 if q == 9 else 3, u0=0.05, tau=tau, velset=q if q != 27 else 19, with_density=True)
    s = oracle.Sim(w.nx, w.ny, w.nz, w.velset, oracle.FP64, tau, None, F64)
    s.set_collision(oracle.TRT)
    s.init(w.rho.astype(np.float64), w.u.astype(np.float64))
    s.step(50)
    _, u50 = s.read_rho_u(f64=True)
    s.step(150)
    _, u200 = s.read_rho_u(f64=True)
    amp = lambda u: (u[0] * w.u[0]).sum() / (w.u[0].astype(np.float64) ** 2).sum()
    rate = -math.log(amp(u200) / amp(u50)) / 150
    assert rate == pytest.approx(2 * (tau / 3 - 1 / 6) * (2 * math.pi / n) ** 2, rel=5e-3)


# ---- R18: zero-gradient outflow cells (BASELINE configs[3]; not in the paper) ---------------------------------------
@pytest.mark.parametrize("q,shape", [(19, (8, 6, 5)), (27, (7, 5, 4)), (9, (9, 7, 1))])
def test_outflow_cells_against_push_reference(q, shape):
    """walls, moving walls, an equilibrium inflow plane, an outflow plane and a body force together, vs the second
    implementation (which imposes on an outflow cell the equilibrium of its upstream neighbour's previous state)"""
    w = wl.perturbed_equilibrium(*shape, seed=17, velset=q, rho_sigma=1e-2, tau=0.8)
    w = wl.random_walls(w, 0.1, seed=8, moving_fraction=0.5)
    f = w.flags.reshape(w.nz, w.ny, w.nx).copy()
    f[:, :, 0] = wl.FLAG_EQ
    f[:, :, -1] = wl.FLAG_OUT
    w.flags = f.reshape(-1)
    w.force = (1e-4, -2e-4, 0.0 if q == 9 else 3e-4)
    s = sim64(w)
    s.step(9)
    rho, u = s.read_rho_u(f64=True)
    rref, uref = _reference_push_unshifted(w, 9)
    assert np.abs(rho - rref).max() < 5e-14
    assert np.abs(u - uref).max() < 5e-14


def test_outflow_keeps_uniform_flow_and_has_zero_gradient():
    """Inflow by equilibrium cells at x = 0, outflow cells at x = nx-1, periodic in y and z.  (i) A uniform state is a
    fixed point.  (ii) Started at rest, the channel starts to flow, and at the outflow plane density and velocity equal
    the upstream neighbour's of the step before (that is the definition), so the gradient there vanishes as the flow
    becomes steady."""
    ue = (0.05, 0.0, 0.0)

    def box(u_init):
        w = wl.perturbed_equilibrium(24, 5, 3, seed=1, rho_sigma=0.0, u_abs_max=0.0, tau=0.8)
        f = w.flags.reshape(w.nz, w.ny, w.nx).copy()
        f[:, :, 0] = wl.FLAG_EQ
        f[:, :, -1] = wl.FLAG_OUT
        w.flags = f.reshape(-1)
        u = np.zeros((3, w.nz, w.ny, w.nx), np.float32)
        u[0] = u_init
        u[0, :, :, 0] = ue[0]
        w.u = u.reshape(3, -1)
        return w
    w = box(ue[0])
    s = sim64(w)
    s.step(50)
    rho, u = s.read_rho_u(f64=True)
    assert np.abs(rho - 1.0).max() < 1e-13 and np.abs(u[0] - np.float32(ue[0])).max() < 1e-13 and np.abs(u[1:]).max() < 1e-14
    w = box(0.0)
    s = sim64(w)
    s.step(1999)
    rho_a, u_a = s.read_rho_u(f64=True)
    s.step(1)
    rho_b, u_b = s.read_rho_u(f64=True)
    ux_a, ux_b = u_a[0].reshape(w.nz, w.ny, w.nx), u_b[0].reshape(w.nz, w.ny, w.nx)
    assert np.abs(ux_b[:, :, -1] - ux_a[:, :, -2]).max() < 1e-15          # the definition, one step apart
    assert np.abs(rho_b.reshape(w.nz, w.ny, w.nx)[:, :, -1] - rho_a.reshape(w.nz, w.ny, w.nx)[:, :, -2]).max() < 1e-15
    assert ux_b[:, :, 1:].min() > 0.2 * ue[0]                              # the channel flows downstream, out through the plane
    assert np.abs(ux_b[:, :, -1] - ux_b[:, :, -2]).max() < 1e-6            # zero gradient at the outflow


# ---- R17: without DDF-shifting, eqs (19)-(23): the paper's negative control -------------------------
@pytest.mark.parametrize("q,shape,force", [(19, (6, 5, 4), (1e-4, -2e-4, 3e-4)), (27, (4, 5, 4), (0.0, 0.0, 0.0)), (9, (7, 6, 1), (1e-4, 2e-4, 0.0))])
def test_unshifted_variant(q, shape, force):
    """In FP64 the unshifted step equals the second implementation (itself unshifted, plain eq (22)) and the shifted
    step to rounding, and what it stores is the shifted DDF plus the lattice weight."""
    w = wl.perturbed_equilibrium(*shape, seed=19, velset=q, rho_sigma=1e-2, tau=0.7)
    w = wl.random_walls(w, 0.15, seed=5, moving_fraction=0.5)
    w.force = force
    a = oracle.from_workload(w, oracle.FP64, oracle.ARITH_F64, shifted=False)
    b = sim64(w)
    a.step(7)
    b.step(7)
    rho, u = a.read_rho_u(f64=True)
    rref, uref = _reference_push_unshifted(w, 7)
    assert np.abs(rho - rref).max() < 5e-14 and np.abs(u - uref).max() < 5e-14
    rho_s, u_s = b.read_rho_u(f64=True)
    assert np.abs(rho - rho_s).max() < 5e-14 and np.abs(u - u_s).max() < 5e-14
    _, wts, _ = oracle.velocity_set(q)
    fluid = w.flags == 0
    for i in range(q):
        assert np.abs(a.read_ddf(i)[fluid] - b.read_ddf(i)[fluid] - wts[i]).max() < 5e-15


def test_shifting_is_what_makes_16_bit_storage_accurate():
    """PAPER.md:314-316 (Fig. 8, dashed curves): without DDF-shifting the 16-bit formats lose the Taylor-Green decay;
    with it they follow the FP64 run.  2-D Taylor-Green, D2Q9, FP16C and FP16S storage, FP32 arithmetic."""
    w = wl.taylor_green_2d(32, 32, 1)
    ref = sim64(w)
    ref.step(100)
    _, uref = ref.read_rho_u(f64=True)
    for fmt in (oracle.FP16C, oracle.FP16S, oracle.P16_1S):
        err = {}
        for shifted in (True, False):
            s = oracle.from_workload(w, fmt, shifted=shifted)
            s.step(100)
            _, u = s.read_rho_u()
            err[shifted] = np.abs(u - uref).max() / np.abs(uref).max()
        assert err[True] < 0.02 and err[False] > 5 * err[True], (fmt, err)
