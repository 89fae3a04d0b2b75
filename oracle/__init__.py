"""ctypes front end of the CPU oracle (oracle/liblbm_oracle.so).

TEST INFRASTRUCTURE, NOT PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
`--impl reference` legs may import this package.  It never imports the CUDA package and shares no code
with it.  Parity status of each function is listed in DESIGN.md section 4 ("pins").
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

FP32, FP16S, FP16C, P16_0S, P16_1S, P16_2C, FP16, FP64 = range(8)
ARITH_F32, ARITH_F64 = 0, 1
BGK, TRT = 0, 1

_lib = None


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        L.orc_table_value.restype = C.c_double
        L.orc_table_value.argtypes = [C.c_int, C.c_uint]
        L.orc_scale.restype = C.c_double
        L.orc_scale.argtypes = [C.c_int]
        L.orc_decode.argtypes = [C.c_int, C.c_void_p, C.c_void_p, C.c_long]
        L.orc_encode.argtypes = [C.c_int, C.c_void_p, C.c_void_p, C.c_long]
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.c_int] * 6 + [C.c_double, C.c_void_p]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_destroy.restype = None
        L.orc_set_collision.argtypes = [C.c_void_p, C.c_int, C.c_double]
        L.orc_set_shifting.argtypes = [C.c_void_p, C.c_int]
        for name in ("orc_set_flags",):
            getattr(L, name).argtypes = [C.c_void_p, C.c_void_p]
        for name in ("orc_init", "orc_init_f64", "orc_read_rho_u", "orc_read_rho_u_f64"):
            getattr(L, name).argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_step.argtypes = [C.c_void_p, C.c_int]
        L.orc_read_ddf.argtypes = [C.c_void_p, C.c_int, C.c_void_p]
        L.orc_sum_ddf.restype = C.c_double
        L.orc_sum_ddf.argtypes = [C.c_void_p]
        L.orc_set_threads.argtypes = [C.c_int]
        L.orc_velocity_set.argtypes = [C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_equilibrium.argtypes = [C.c_int, C.c_int] + [C.c_double] * 4 + [C.c_void_p]
        _lib = L
    return _lib


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p)


def table_value(fmt: int, mag: int) -> float:
    return lib().orc_table_value(fmt, mag)


def scale(fmt: int) -> float:
    return lib().orc_scale(fmt)


def decode(fmt: int, codes) -> np.ndarray:
    codes = np.ascontiguousarray(codes, dtype=np.uint16)
    out = np.empty(codes.shape, np.float32)
    assert lib().orc_decode(fmt, _ptr(codes), _ptr(out), codes.size) == 0
    return out


def encode(fmt: int, x) -> np.ndarray:
    x = np.ascontiguousarray(x, dtype=np.float32)
    out = np.empty(x.shape, np.uint16)
    assert lib().orc_encode(fmt, _ptr(x), _ptr(out), x.size) == 0
    return out


def set_threads(n: int) -> int:
    return lib().orc_set_threads(n)


def velocity_set(velset: int):
    c = np.zeros((27, 3), np.int32)
    w = np.zeros(27, np.float64)
    opp = np.zeros(27, np.int32)
    q = lib().orc_velocity_set(velset, _ptr(c), _ptr(w), _ptr(opp))
    assert q > 0
    return c[:q].copy(), w[:q].copy(), opp[:q].copy()


def equilibrium(velset: int, rho: float, ux: float, uy: float, uz: float, arith: int = ARITH_F64) -> np.ndarray:
    feq = np.zeros(27, np.float64)
    q = lib().orc_equilibrium(velset, arith, rho, ux, uy, uz, _ptr(feq))
    assert q > 0
    return feq[:q].copy()


_DDF_DTYPE = {FP32: np.float32, FP64: np.float64}


class Sim:
    """One oracle simulation.  Mirrors the product's call sequence: create -> set_flags -> init -> step -> read."""

    def __init__(self, nx, ny, nz, velset=19, fmt=FP32, tau=0.6, force=None, arith=ARITH_F32):
        f = None
        if force is not None:
            f = np.ascontiguousarray(force, dtype=np.float64)
        self._h = lib().orc_create(nx, ny, nz, velset, fmt, arith, float(tau), _ptr(f) if f is not None else None)
        if not self._h:
            raise ValueError("orc_create rejected the arguments")
        self.nx, self.ny, self.nz, self.q, self.fmt, self.arith = nx, ny, nz, velset, fmt, arith
        self.N = nx * ny * nz

    def close(self):
        if self._h:
            lib().orc_destroy(self._h)
            self._h = None

    def __del__(self):
        self.close()

    def set_flags(self, flags):
        flags = np.ascontiguousarray(flags, dtype=np.uint8)
        assert flags.size == self.N
        assert lib().orc_set_flags(self._h, _ptr(flags)) == 0

    def init(self, rho, u):
        if self.arith == ARITH_F64 and np.asarray(rho).dtype == np.float64:
            rho = np.ascontiguousarray(rho, dtype=np.float64)
            u = np.ascontiguousarray(u, dtype=np.float64)
            assert rho.size == self.N and u.size == 3 * self.N
            assert lib().orc_init_f64(self._h, _ptr(rho), _ptr(u)) == 0
        else:
            rho = np.ascontiguousarray(rho, dtype=np.float32)
            u = np.ascontiguousarray(u, dtype=np.float32)
            assert rho.size == self.N and u.size == 3 * self.N
            assert lib().orc_init(self._h, _ptr(rho), _ptr(u)) == 0

    def set_collision(self, collision, lam=3.0 / 16.0):
        assert lib().orc_set_collision(self._h, int(collision), float(lam)) == 0

    def set_shifting(self, on: bool):
        """DDF-shifting on (default) / off (eqs (19)-(23), the paper's negative control); call before init"""
        assert lib().orc_set_shifting(self._h, 1 if on else 0) == 0

    def step(self, n=1):
        assert lib().orc_step(self._h, int(n)) == 0

    def read_rho_u(self, f64=False):
        if f64:
            rho = np.empty(self.N, np.float64)
            u = np.empty((3, self.N), np.float64)
            assert lib().orc_read_rho_u_f64(self._h, _ptr(rho), _ptr(u)) == 0
        else:
            rho = np.empty(self.N, np.float32)
            u = np.empty((3, self.N), np.float32)
            assert lib().orc_read_rho_u(self._h, _ptr(rho), _ptr(u)) == 0
        return rho, u

    def read_ddf(self, i: int) -> np.ndarray:
        out = np.empty(self.N, _DDF_DTYPE.get(self.fmt, np.uint16))
        assert lib().orc_read_ddf(self._h, i, _ptr(out)) == 0
        return out

    def sum_ddf(self) -> float:
        return lib().orc_sum_ddf(self._h)


def from_workload(w, fmt=FP32, arith=ARITH_F32, shifted=True) -> Sim:
    s = Sim(w.nx, w.ny, w.nz, w.velset, fmt, w.tau, w.force, arith)
    if not shifted:
        s.set_shifting(False)
    s.set_flags(w.flags)
    s.init(w.rho, w.u)
    return s
