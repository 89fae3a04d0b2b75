"""Seeded, synthetic input generators shared by the oracle tests, the GPU parity tests and bench.py.

This module holds NONE of the method's arithmetic (no equilibrium, no codec, no collision): it only
builds the *inputs* of the hot path -- box size, flags, initial density / velocity fields, tau, force --
for the five workload shapes of BASELINE.json `configs` (which take their shapes from the paper's
set-ups, PAPER.md:229-360 sections 4.1-4.4 and PAPER.md:432 section 5).  Every field is generated in
float64 and rounded ONCE to float32, so the oracle and the CUDA path read bit-identical arrays.

Layout conventions (PAPER.md:938 `n = x+(y+z*sy)*sx`, PAPER.md:996 SoA velocity):
  cell index  n = x + nx*(y + ny*z)
  rho   float32 [N]
  u     float32 [3, N]   (ux | uy | uz)
  flags uint8   [N]      bit 0x01 = wall (TYPE_W)
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

FLAG_WALL = 0x01
FLAG_EQ = 0x02      # equilibrium boundary cell (TYPE_E)
FLAG_OUT = 0x04     # zero-gradient outflow cell (BASELINE configs[3]; R18)

# velocity-set / collision / storage-format ids of include/lbm.h (interface constants, not arithmetic)
D2Q9, D3Q19, D3Q27 = 9, 19, 27
FORMATS = {"FP32": 0, "FP16S": 1, "FP16C": 2, "P16_0S": 3, "P16_1S": 4, "P16_2C": 5, "FP16": 6}
FORMAT_NAMES = {v: k for k, v in FORMATS.items()}
FORMATS_16BIT = [k for k in FORMATS if k != "FP32"]


@dataclass
class Workload:
    name: str
    nx: int
    ny: int
    nz: int
    velset: int
    tau: float
    rho: np.ndarray            # float32 [N]
    u: np.ndarray              # float32 [3, N]
    flags: np.ndarray          # uint8 [N]
    force: tuple = (0.0, 0.0, 0.0)
    steps: int = 0             # the step count the config names
    meta: dict = field(default_factory=dict)

    @property
    def n_cells(self) -> int:
        return self.nx * self.ny * self.nz


def _grid(nx, ny, nz):
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    return x.reshape(-1).astype(np.float64), y.reshape(-1).astype(np.float64), z.reshape(-1).astype(np.float64)


def _pack(ux, uy, uz):
    return np.ascontiguousarray(np.stack([ux, uy, uz]).astype(np.float32))


def taylor_green_3d(n: int = 32, u0: float = 0.05, tau: float = 0.6, velset: int = D3Q19) -> Workload:
    """BASELINE.json configs[0]: 3-D Taylor-Green vortex, fully periodic cube, rho0 = 1,
    u = (u0 sin kx cos ky cos kz, -u0 cos kx sin ky cos kz, 0), k = 2 pi / n, 200 steps."""
    x, y, z = _grid(n, n, n)
    k = 2.0 * math.pi / n
    ux = u0 * np.sin(k * x) * np.cos(k * y) * np.cos(k * z)
    uy = -u0 * np.cos(k * x) * np.sin(k * y) * np.cos(k * z)
    uz = np.zeros_like(ux)
    N = n ** 3
    return Workload("taylor_green_3d", n, n, n, velset, tau, np.ones(N, np.float32), _pack(ux, uy, uz),
                    np.zeros(N, np.uint8), steps=200, meta={"u0": u0, "k": k})


def taylor_green_2d(nx: int = 32, ny: int = 32, nz: int = 1, u0: float = 0.05, tau: float = 0.6,
                    velset: int = D2Q9, with_density: bool = False) -> Workload:
    """2-D Taylor-Green vortices of PAPER.md:285-293 (eqs 15-17) at t = 0, z-invariant.
    `with_density` also imposes the density field of eq (17); otherwise rho0 = 1."""
    x, y, z = _grid(nx, ny, nz)
    kx, ky = 2.0 * math.pi / nx, 2.0 * math.pi / ny
    ux = u0 * np.cos(kx * x) * np.sin(ky * y)
    uy = -u0 * np.sin(kx * x) * np.cos(ky * y)
    rho = np.ones_like(ux)
    if with_density:
        rho = 1.0 - 0.75 * u0 * u0 * (np.cos(2 * kx * x) + np.cos(2 * ky * y))
    N = nx * ny * nz
    return Workload("taylor_green_2d", nx, ny, nz, velset, tau, rho.astype(np.float32),
                    _pack(ux, uy, np.zeros_like(ux)), np.zeros(N, np.uint8), steps=200,
                    meta={"u0": u0, "kx": kx, "ky": ky})


def poiseuille_channel(nx: int = 16, ny: int = 64, nz: int = 16, tau: float = 0.8, u_max: float = 0.01,
                       velset: int = D3Q19) -> Workload:
    """BASELINE.json configs[1]: planar channel, periodic in x and z, wall cells at y = 0 and y = ny-1,
    fluid at rest, uniform body force along x sized for a centre-line velocity u_max.
    The walls of a halfway bounce-back channel sit half a cell outside the first fluid node, so the
    channel width is H = ny - 2 and f = 8 nu u_max / H^2 (planar analogue of PAPER.md:252 eq 13)."""
    nu = tau / 3.0 - 1.0 / 6.0
    H = ny - 2
    fx = 8.0 * nu * u_max / (H * H)
    N = nx * ny * nz
    flags = np.zeros((nz, ny, nx), np.uint8)
    flags[:, 0, :] = FLAG_WALL
    flags[:, ny - 1, :] = FLAG_WALL
    return Workload("poiseuille_channel", nx, ny, nz, velset, tau, np.ones(N, np.float32),
                    np.zeros((3, N), np.float32), flags.reshape(-1), force=(fx, 0.0, 0.0), steps=20000,
                    meta={"nu": nu, "H": H, "u_max": u_max})


def lid_driven_cavity(L: int = 32, u_lid: float = 0.1, tau: float | None = None, Re: float = 1000.0,
                      velset: int = D3Q19) -> Workload:
    """BASELINE.json configs[2]: cubic box, one-cell wall shell on all six faces, the
    z = L-1 face is the lid and carries the wall velocity (0, u_lid, 0) ("velocity parallel to the
    y-axis").  tau defaults to the value Re = L u_lid / nu gives at this L."""
    if tau is None:
        nu = L * u_lid / Re
        tau = 3.0 * nu + 0.5
    N = L ** 3
    flags = np.zeros((L, L, L), np.uint8)          # [z, y, x]
    flags[0, :, :] = flags[L - 1, :, :] = FLAG_WALL
    flags[:, 0, :] = flags[:, L - 1, :] = FLAG_WALL
    flags[:, :, 0] = flags[:, :, L - 1] = FLAG_WALL
    uy = np.zeros((L, L, L), np.float64)
    uy[L - 1, :, :] = u_lid
    u = _pack(np.zeros(N), uy.reshape(-1), np.zeros(N))
    return Workload("lid_driven_cavity", L, L, L, velset, float(tau), np.ones(N, np.float32), u,
                    flags.reshape(-1), steps=50000, meta={"u_lid": u_lid, "Re": Re})


def perturbed_equilibrium(nx: int, ny: int, nz: int, seed: int = 20211208, tau: float = 0.6,
                          velset: int = D3Q19, rho_sigma: float = 1e-3, u_abs_max: float = 0.05) -> Workload:
    """BASELINE.json configs[4] (paper's benchmark box: cubic, periodic, no boundary
    nodes): rho = 1 + N(0, rho_sigma), u uniform in [-1,1]^3 scaled so |u| <= u_abs_max."""
    rng = np.random.default_rng(seed)
    N = nx * ny * nz
    rho = (1.0 + rho_sigma * rng.standard_normal(N)).astype(np.float32)
    u = np.empty((3, N), np.float32)
    s = u_abs_max / math.sqrt(3.0)                 # |(a,b,c)| <= sqrt(3) for a,b,c in [-1,1]
    for a in range(3):
        u[a] = (s * rng.uniform(-1.0, 1.0, N)).astype(np.float32)
    if velset == D2Q9:
        u[2] = 0.0
    return Workload("perturbed_equilibrium", nx, ny, nz, velset, tau, rho, u, np.zeros(N, np.uint8),
                    steps=1000, meta={"seed": seed})


def random_walls(w: Workload, fraction: float, seed: int = 7, moving_fraction: float = 0.0,
                 u_wall: float = 0.05) -> Workload:
    """Test helper: sprinkle wall cells (and optionally moving walls) into a workload, seeded."""
    rng = np.random.default_rng(seed)
    N = w.n_cells
    wall = rng.uniform(size=N) < fraction
    w.flags = np.where(wall, FLAG_WALL, w.flags).astype(np.uint8)
    if moving_fraction > 0.0:
        mv = wall & (rng.uniform(size=N) < moving_fraction)
        uw = (u_wall * rng.uniform(-1.0, 1.0, (3, N))).astype(np.float32)
        if w.velset == D2Q9:
            uw[2] = 0.0
        w.u = np.where(mv[None, :], uw, np.where(wall[None, :], np.float32(0), w.u)).astype(np.float32)
    else:
        w.u = np.where(wall[None, :], np.float32(0), w.u).astype(np.float32)
    return w



def karman_vortex_street(nx: int = 256, ny: int = 64, nz: int = 16, radius: float = 4.0, x_cyl: int | None = None,
                         u_in: float = 0.05, tau: float | None = None, Re: float = 200.0, velset: int = D3Q19,
                         outflow: bool = False) -> Workload:
    """BASELINE.json configs[3] (shape of PAPER.md:320-336): a channel with a z-spanning cylinder of wall cells at
    (x_cyl, ny/2), flow along +x.  The x = 0, x = nx-1, y = 0 and y = ny-1 planes are equilibrium boundary cells
    holding rho = 1, u = (u_in, 0, 0) (the paper enforces the velocity on the box perimeter with equilibrium
    boundaries); z is periodic.  Asymmetric start as in PAPER.md:330: the fluid moves with u_in in
    one half of the box (y < ny/2) and rests in the other, so that shedding starts at once in every number format.
    outflow=True replaces the equilibrium cells of the x = nx-1 plane by zero-gradient outflow cells (BASELINE's wording).
    tau defaults to the value Re = 2 R u_in / nu gives."""
    if x_cyl is None:
        x_cyl = nx // 4
    if tau is None:
        nu = 2.0 * radius * u_in / Re
        tau = 3.0 * nu + 0.5
    nzz = 1 if velset == D2Q9 else nz
    N = nx * ny * nzz
    z, y, x = np.meshgrid(np.arange(nzz), np.arange(ny), np.arange(nx), indexing="ij")
    flags = np.zeros((nzz, ny, nx), np.uint8)
    flags[(x - x_cyl) ** 2 + (y - ny // 2) ** 2 <= radius * radius] = FLAG_WALL
    rim = (x == 0) | (x == nx - 1) | (y == 0) | (y == ny - 1)
    flags[rim] = FLAG_EQ
    if outflow:                                    # BASELINE's "zero-gradient outflow": the x = nx-1 plane between the y rims
        flags[(x == nx - 1) & (y > 0) & (y < ny - 1)] = FLAG_OUT
    ux = np.where(rim | (y < ny // 2), u_in, 0.0)
    ux[flags == FLAG_WALL] = 0.0
    u = _pack(ux.reshape(-1), np.zeros(N), np.zeros(N))
    return Workload("karman_vortex_street", nx, ny, nzz, velset, float(tau), np.ones(N, np.float32), u,
                    flags.reshape(-1), steps=100000,
                    meta={"u_in": u_in, "radius": radius, "x_cyl": x_cyl, "probe": (nx // 2, ny // 2, nzz // 2)})


def equilibrium_rim(w: Workload, rho_e: float = 1.0, u_e=(0.03, -0.01, 0.02)) -> Workload:
    """Test helper: turn the x and y faces of a workload into equilibrium boundary cells holding (rho_e, u_e)."""
    f = w.flags.reshape(w.nz, w.ny, w.nx).copy()
    rim = np.zeros_like(f, bool)
    rim[:, :, 0] = rim[:, :, -1] = True
    rim[:, 0, :] = rim[:, -1, :] = True
    f[rim] = FLAG_EQ
    w.flags = f.reshape(-1)
    r = rim.reshape(-1)
    w.rho = np.where(r, np.float32(rho_e), w.rho).astype(np.float32)
    ue = np.array(u_e, np.float32)
    if w.velset == D2Q9:
        ue[2] = 0.0
    w.u = np.where(r[None, :], ue[:, None], w.u).astype(np.float32)
    return w

def codec_probe_inputs(seed: int = 1, per_binade: int = 4096) -> np.ndarray:
    """float32 inputs for encoder parity: every binade 2^-70 .. 2^24 sampled `per_binade` times with
    both signs, plus zeros, infinities and NaN.  (The tie / boundary inputs of each format are added
    by the tests from the oracle's value table -- they depend on the format definition, not on a seed.)"""
    rng = np.random.default_rng(seed)
    out = []
    for e in range(-70, 25):
        m = rng.uniform(1.0, 2.0, per_binade)
        out.append(np.ldexp(m, e))
    x = np.concatenate(out).astype(np.float32)
    special = np.array([0.0, -0.0, np.inf, -np.inf, np.nan, 1.0, -1.0, 2.0, -2.0, 65504.0, 65520.0,
                        3.4e38, 1e-45, 1.1754944e-38], np.float32)
    return np.concatenate([x, -x, special])


def generated_fields(cells, seed: int, two_d: bool = False):
    """rho [k], u [3, k] (float32) of the cells with indices `cells` as the library's lbm_init_generated draws them on
    the device (include/lbm.h; the recipe is restated here, not shared): for cell n and k = 0..6
        z = splitmix64(seed + (8 n + k) * 0x9E3779B97F4A7C15),   a_k = (z >> 42) * 2^-22   in [0, 1)
        rho = 1 + ((a_0 + a_1) + (a_2 + a_3) - 2) * float32(1.7320508e-3)       (all float32, IEEE)
        u_a = (2 a_{4+a} - 1) * float32(0.028867513);   u_z = 0 for D2Q9.
    Inputs only: boxes too large for host arrays (BASELINE configs[4]'s largest cubes) are checked on sampled blocks."""
    n = np.asarray(cells, dtype=np.uint64).reshape(-1)
    mask = np.uint64(0xFFFFFFFFFFFFFFFF)
    a = []
    with np.errstate(over="ignore"):
        for k in range(7):
            z = (np.uint64(seed & 0xFFFFFFFFFFFFFFFF) + (np.uint64(8) * n + np.uint64(k)) * np.uint64(0x9E3779B97F4A7C15)) & mask
            z ^= z >> np.uint64(30)
            z = (z * np.uint64(0xBF58476D1CE4E5B9)) & mask
            z ^= z >> np.uint64(27)
            z = (z * np.uint64(0x94D049BB133111EB)) & mask
            z ^= z >> np.uint64(31)
            a.append(((z >> np.uint64(42)).astype(np.float32)) * np.float32(2.0 ** -22))
    g = ((a[0] + a[1]) + (a[2] + a[3])) - np.float32(2.0)
    rho = np.float32(1.0) + g * np.float32(1.7320508e-3)
    u = np.stack([(np.float32(2.0) * a[4 + k] - np.float32(1.0)) * np.float32(0.028867513) for k in range(3)])
    if two_d:
        u[2] = 0.0
    return rho.astype(np.float32), u.astype(np.float32)
