"""The accuracy set-ups of BASELINE.json configs[0..3] on the GPU path, one command each: the numbers of DESIGN.md section 6.

    python -m paper_2112_08926_b200.configs 1 [--formats FP32,FP16S,...]          Taylor-Green 32^3, 200 steps
    python -m paper_2112_08926_b200.configs 2 [--steps 20000]                     Poiseuille channel 16 x 64 x 16
    python -m paper_2112_08926_b200.configs 3 [--size 128] [--steps 50000] [--collision TRT]    lid-driven cavity
    python -m paper_2112_08926_b200.configs 4 [--size 256] [--steps 100000]       Karman street 4L x L x L/4

Every step of the path runs in the library's CUDA kernels (paper_2112_08926_b200.Simulation); what is here is set-up
(workloads/), the read-out, and the EVALUATION of the results against closed forms the paper states -- the kinetic-energy
decay of eq (18), the Poiseuille profile of eqs (9), (13) and the L2 error of eq (14)
(PAPER.md:235-257), the Strouhal number of PAPER.md:330-336.  None of it is the method's arithmetic.  Each command
prints a table and one JSON line (`--json FILE` appends it to a file), with the throughput and the SM clock of the run.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads as wl  # noqa: E402

ALL16 = ["FP32", "FP16S", "FP16C", "P16_0S", "P16_1S", "P16_2C", "FP16"]


def _lbm():
    import paper_2112_08926_b200 as lbm
    return lbm


def _timed_steps(sim, n):
    """n steps, device-timed: returns milliseconds."""
    import torch
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    sim.step(n)
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1)


def _clock():
    import subprocess
    try:
        out = subprocess.run(["nvidia-smi", "--query-gpu=clocks.sm,clocks.max.sm,power.draw", "--format=csv,noheader,nounits", "-i", "0"],
                             capture_output=True, text=True, timeout=10).stdout.strip().split(",")
        return {"sm_mhz_after": float(out[0]), "sm_max_mhz": float(out[1]), "power_w_after": float(out[2])}
    except Exception:
        return {}


# ---- config 1: Taylor-Green vortex ---------------------------------------------------------------------------
def config1(formats, steps=200, collision="BGK", graphs=True):
    """3-D Taylor-Green, 32^3, tau 0.6: E(t)/E(0) with E = 1/2 sum rho |u|^2, and the drift of the total mass per cell.
    The 3-D field is not an exact Navier-Stokes solution: exp(-2 nu |k|^2 t) is the Stokes-limit band (SURVEY.md
    section 8(c)); the FP64 run is the reference the storage formats are compared with."""
    lbm = _lbm()
    w = wl.taylor_green_3d(32)
    nu = w.tau / 3.0 - 1.0 / 6.0
    k2 = 3.0 * w.meta["k"] ** 2
    rows = []
    for name in ["FP64"] + [f for f in formats if f != "FP64"]:
        sim = lbm.from_workload(w, name, collision=lbm.TRT if collision == "TRT" else lbm.BGK)
        sim.set_graphs(graphs)
        rho, u = (sim.read_rho_u_f64() if name == "FP64" else sim.read_rho_u())
        e0 = 0.5 * float((rho.astype(np.float64) * (u.astype(np.float64) ** 2).sum(0)).sum())
        m0 = float(rho.astype(np.float64).sum())
        ms = _timed_steps(sim, steps)
        rho, u = (sim.read_rho_u_f64() if name == "FP64" else sim.read_rho_u())
        e1 = 0.5 * float((rho.astype(np.float64) * (u.astype(np.float64) ** 2).sum(0)).sum())
        m1 = float(rho.astype(np.float64).sum())
        rows.append({"format": name, "E_over_E0": e1 / e0, "mass_drift_per_cell": (m1 - m0) / w.n_cells,
                     "steps_per_s": steps / (ms * 1e-3), "kernel": sim.kernel_name})
        sim.close()
    return {"config": 1, "what": f"Taylor-Green 32^3, tau 0.6, {steps} steps, {collision}" + ("" if graphs else ", CUDA graphs off"),
            "stokes_limit": math.exp(-2.0 * nu * k2 * steps), "rows": rows}


# ---- config 2: Poiseuille channel --------------------------------------------------------------------------------
def poiseuille_exact(ny, tau, u_max, t, terms=400):
    """u_x(y, t) of the channel started from rest under the force 8 nu u_max / H^2 (planar analogue of PAPER.md:235-257,
    eqs (9), (13)): the steady parabola minus its decaying Fourier modes, plus the halfway bounce-back slip
    F (48 nu^2 - 1) / (8 nu) of BGK (He et al. 1997).  y = j - 1/2 for the fluid node j = 1 .. ny-2, H = ny - 2."""
    nu = tau / 3.0 - 1.0 / 6.0
    H = ny - 2.0
    F = 8.0 * nu * u_max / (H * H)
    y = np.arange(1, ny - 1) - 0.5
    u = F / (2.0 * nu) * y * (H - y)
    for n in range(1, 2 * terms, 2):
        u -= 32.0 * u_max / (n * math.pi) ** 3 * np.sin(n * math.pi * y / H) * math.exp(-(n * math.pi / H) ** 2 * nu * t)
    slip = F * (48.0 * nu * nu - 1.0) / (8.0 * nu)
    return u + slip, F / (2.0 * nu) * y * (H - y)


def l2_error(u, ref):
    """eq (14), PAPER.md:257"""
    return math.sqrt(float(((u - ref) ** 2).sum()) / float((ref ** 2).sum()))


def config2(formats, steps=20000, collision="BGK", graphs=True):
    lbm = _lbm()
    w = wl.poiseuille_channel()
    rows = []
    for name in formats:
        sim = lbm.from_workload(w, name, collision=lbm.TRT if collision == "TRT" else lbm.BGK)
        sim.set_graphs(graphs)
        ms = _timed_steps(sim, steps)
        rho, u = sim.read_rho_u()
        ux = u[0].reshape(w.nz, w.ny, w.nx)[w.nz // 2, 1:-1, w.nx // 2].astype(np.float64)
        exact, parabola = poiseuille_exact(w.ny, w.tau, w.meta["u_max"], steps)
        rows.append({"format": name, "L2_vs_transient_plus_slip": l2_error(ux, exact), "L2_vs_parabola": l2_error(ux, parabola),
                     "u_centre": float(ux[len(ux) // 2]), "steps_per_s": steps / (ms * 1e-3), "kernel": sim.kernel_name})
        sim.close()
    return {"config": 2, "what": f"Poiseuille 16x64x16, tau 0.8, u_max 0.01, {steps} steps, {collision}"
                                 + (" (the slip term is BGK's; TRT with Lambda = 3/16 has none)" if collision == "TRT" else "")
                                 + ("" if graphs else ", CUDA graphs off"),
            "rows": rows}


# ---- config 3: lid-driven cavity ---------------------------------------------------------------------------------
def config3(formats, size=128, steps=50000, collision="BGK"):
    """Centre-line profiles u_y(z) at x = y = L/2 and u_z(y) at x = z = L/2 (Fig. 11), per storage
    format; the deviation of each format from the FIRST format of the list (FP32 by default), in units of the lid
    velocity, is the paper's measure of what a storage format costs."""
    lbm = _lbm()
    L = size
    w = wl.lid_driven_cavity(L)
    c = L // 2
    rows, ref = [], None
    for name in formats:
        sim = lbm.from_workload(w, name, collision=lbm.TRT if collision == "TRT" else lbm.BGK)
        ms = _timed_steps(sim, steps)
        rho, u = sim.read_rho_u()
        u = u.reshape(3, L, L, L)                                  # [component, z, y, x]
        uy_z = u[1, :, c, c].astype(np.float64) / w.meta["u_lid"]
        uz_y = u[2, c, :, c].astype(np.float64) / w.meta["u_lid"]
        if ref is None:
            ref = (uy_z, uz_y)
        rows.append({"format": name, "min_uy_over_ulid": float(uy_z.min()), "max_uz_over_ulid": float(uz_y.max()),
                     "max_dev_from_first": float(max(np.abs(uy_z - ref[0]).max(), np.abs(uz_y - ref[1]).max())),
                     "finite": bool(np.isfinite(rho).all()), "mlups": L ** 3 * steps / ms / 1e3, "kernel": sim.kernel_name})
        sim.close()
    return {"config": 3, "what": f"lid-driven cavity {L}^3, Re 1000 (tau {w.tau:.4f}), u_lid 0.1, {steps} steps, {collision}", "rows": rows}


# ---- config 4: Karman vortex street ------------------------------------------------------------------------------
def strouhal(signal, dt, diameter, u_in):
    """Shedding frequency from the spectrum of the probe signal (largest peak, parabolic interpolation of its
    neighbours), St = f D / u."""
    s = np.asarray(signal, np.float64)
    s = (s - s.mean()) * np.hanning(s.size)
    spec = np.abs(np.fft.rfft(s))
    k = int(spec[1:].argmax()) + 1
    if 1 <= k < spec.size - 1:
        a, b, c = spec[k - 1], spec[k], spec[k + 1]
        k = k + 0.5 * (a - c) / (a - 2 * b + c)
    f = k / (s.size * dt)
    return f * diameter / u_in


def config4(formats, size=256, steps=100000, every=10, outflow=False):
    """z-spanning cylinder in a 4L x L x L/4 box, equilibrium rim, asymmetric start; u_y at the probe behind the cylinder
    every `every` steps; the Strouhal number from the last half of the signal."""
    lbm = _lbm()
    w = wl.karman_vortex_street(4 * size, size, max(size // 4, 1), radius=size / 16.0, outflow=outflow)
    px, py, pz = w.meta["probe"]
    cell = np.array([px + w.nx * (py + w.ny * pz)], np.int64)
    rows = []
    for name in formats:
        sim = lbm.from_workload(w, name)
        sig = []
        t0 = time.perf_counter()
        for _ in range(steps // every):
            sim.step(every)
            _, u = sim.read_rho_u_at(cell)
            sig.append(float(u[1, 0]))
        sim.sync()
        dt = time.perf_counter() - t0
        half = sig[len(sig) // 2:]
        rows.append({"format": name, "strouhal": strouhal(half, every, 2.0 * w.meta["radius"], w.meta["u_in"]),
                     "probe_amplitude": float(0.5 * (max(half) - min(half))), "mlups_incl_probes": w.n_cells * steps / dt / 1e6,
                     "kernel": sim.kernel_name})
        sim.close()
    return {"config": 4, "what": f"Karman street {w.nx}x{w.ny}x{w.nz}, R {w.meta['radius']:g}, u_in 0.05, Re 200 (tau {w.tau:.4f}), "
                                 f"{steps} steps, probe every {every}" + (", zero-gradient outflow at x = nx-1" if outflow else ", equilibrium rim"),
            "rows": rows}


def main():
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("config", type=int, choices=[1, 2, 3, 4])
    ap.add_argument("--formats", default="")
    ap.add_argument("--steps", type=int, default=0)
    ap.add_argument("--size", type=int, default=0)
    ap.add_argument("--collision", default="BGK", choices=["BGK", "TRT"])
    ap.add_argument("--outflow", action="store_true", help="config 4: zero-gradient outflow plane instead of equilibrium cells at x = nx-1")
    ap.add_argument("--no-graphs", action="store_true", help="configs 1, 2: plain launches instead of CUDA graphs (lbm_set_graphs)")
    ap.add_argument("--json", default="")
    a = ap.parse_args()
    if a.config == 1:
        res = config1((a.formats or ",".join(ALL16)).split(","), a.steps or 200, a.collision, not a.no_graphs)
    elif a.config == 2:
        res = config2((a.formats or ",".join(ALL16)).split(","), a.steps or 20000, a.collision, not a.no_graphs)
    elif a.config == 3:
        res = config3((a.formats or ",".join(ALL16)).split(","), a.size or 128, a.steps or 50000, a.collision)
    else:
        res = config4((a.formats or "FP32,FP16S,FP16C,P16_1S").split(","), a.size or 256, a.steps or 100000, outflow=a.outflow)
    res["clocks"] = _clock()
    print(res["what"])
    keys = list(res["rows"][0].keys())
    print(" | ".join(keys))
    for r in res["rows"]:
        print(" | ".join(f"{r[k]:.6g}" if isinstance(r[k], float) else str(r[k]) for k in keys))
    line = json.dumps(res)
    print(line)
    if a.json:
        with open(a.json, "a") as fh:
            fh.write(line + "\n")


if __name__ == "__main__":
    main()
