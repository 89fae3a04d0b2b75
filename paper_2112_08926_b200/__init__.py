"""paper_2112_08926_b200 -- thin Python binding of liblbm_b200.so (include/lbm.h).

Argument marshalling only: every step of the stream-collide path (pull, decode, collide, encode, store,
init, read-out, the codecs) runs in the library's sm_100a CUDA kernels.  PyTorch is used for device
memory (the two DDF buffers, optional device-side init / read-out tensors) and for the CUDA stream.
There is no CPU fallback: importing works without a GPU (so that the symbols can be checked), but any
compute call fails loudly when the library or a CUDA device is missing.

    import paper_2112_08926_b200 as lbm
    sim = lbm.Simulation(nx, ny, nz, velset=19, ddf_format="FP16S", tau=0.6)
    sim.set_flags(flags_u8)            # optional, numpy uint8 [N]
    sim.init(rho_f32, u_f32)           # numpy [N], [3, N]  (or torch CUDA tensors)
    sim.step(200)
    rho, u = sim.read_rho_u()
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "liblbm_b200.so")

D2Q9, D3Q19, D3Q27 = 9, 19, 27
BGK, TRT = 0, 1
FORMATS = {"FP32": 0, "FP16S": 1, "FP16C": 2, "P16_0S": 3, "P16_1S": 4, "P16_2C": 5, "FP16": 6,
           "FP64": 7, "FP64_FP32": 8}     # 7, 8: FP64 arithmetic with double / float storage
FORMAT_NAMES = {v: k for k, v in FORMATS.items()}
FLAG_WALL, FLAG_EQ, FLAG_OUT = 0x01, 0x02, 0x04
VARIANT_AUTO, VARIANT_BULK, VARIANT_STAGED = 0, 16, 32
STATIC_PROBES_MAX = 4096           # include/lbm.h LBM_STATIC_PROBES_MAX
OK, E_INVAL, E_UNSUPPORTED, E_NOMEM, E_CUDA, E_STATE = 0, -1, -2, -3, -4, -5

# every symbol include/lbm.h declares: (restype, argtypes)
_p, _i, _ll, _f = C.c_void_p, C.c_int, C.c_longlong, C.c_float
SYMBOLS = {
    "lbm_create": (_i, [C.POINTER(_p), _i, _i, _i, _i, _i, _i, _f, _p]),
    "lbm_bind": (_i, [_p, _p, _p, _p]),
    "lbm_set_variant": (_i, [_p, _i]),
    "lbm_set_trt_lambda": (_i, [_p, C.c_double]),
    "lbm_set_cells_per_thread": (_i, [_p, _i]),
    "lbm_set_flags": (_i, [_p, _p]),
    "lbm_init": (_i, [_p, _p, _p]),
    "lbm_init_device": (_i, [_p, _p, _p]),
    "lbm_init_generated": (_i, [_p, C.c_ulonglong]),
    "lbm_step": (_i, [_p, _i]),
    "lbm_set_graphs": (_i, [_p, _i]),
    "lbm_set_shifting": (_i, [_p, _i]),
    "lbm_read_rho_u": (_i, [_p, _p, _p]),
    "lbm_read_rho_u_device": (_i, [_p, _p, _p]),
    "lbm_read_rho_u_f64": (_i, [_p, _p, _p]),
    "lbm_read_rho_u_at": (_i, [_p, _p, _i, _p, _p]),
    "lbm_read_rho_u_at_static": (_i, [_p, _p, _i, _p, _p]),
    "lbm_read_ddf": (_i, [_p, _i, _p]),
    "lbm_sync": (_i, [_p]),
    "lbm_steps_done": (_ll, [_p]),
    "lbm_destroy": (_i, [_p]),
    "lbm_last_error": (C.c_char_p, []),
    "lbm_codec_encode": (_i, [_i, _p, _p, _ll]),
    "lbm_codec_decode": (_i, [_i, _p, _p, _ll]),
    "lbm_codec_encode_device": (_i, [_i, _p, _p, _ll, _p]),
    "lbm_codec_decode_device": (_i, [_i, _p, _p, _ll, _p]),
    "lbm_codec_pair_selftest": (_i, [_i, C.POINTER(_ll)]),
    "lbm_div_selftest": (_i, [C.POINTER(_ll)]),
    "lbm_ddf_buffer_bytes": (_ll, [_i, _i, _i, _i, _i]),
    "lbm_bytes_per_cell": (_ll, [_i, _i]),
    "lbm_kernel_name": (C.c_char_p, [_p]),
    "lbm_launch_count": (_ll, []),
}

_lib = None


class LbmError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"liblbm_b200 error {code}: {msg}")
        self.code = code


def lib() -> C.CDLL:
    """Load liblbm_b200.so (built in-tree by `python -m paper_2112_08926_b200.build`)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2112_08926_b200.build` "
                               "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        for name, (res, args) in SYMBOLS.items():
            fn = getattr(L, name)
            fn.restype = res
            fn.argtypes = args
        _lib = L
    return _lib


def last_error() -> str:
    return lib().lbm_last_error().decode()


def _check(rc: int):
    if rc != 0:
        raise LbmError(rc, last_error())


def _np_ptr(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


def _fmt(f) -> int:
    return FORMATS[f] if isinstance(f, str) else int(f)


def bytes_per_cell(velset: int, ddf_format) -> int:
    return int(lib().lbm_bytes_per_cell(velset, _fmt(ddf_format)))


def ddf_buffer_bytes(nx, ny, nz, velset, ddf_format) -> int:
    return int(lib().lbm_ddf_buffer_bytes(nx, ny, nz, velset, _fmt(ddf_format)))


def launch_count() -> int:
    return int(lib().lbm_launch_count())


def _is_torch(x) -> bool:
    return type(x).__module__.startswith("torch")


class Simulation:
    """One LBM box on the current CUDA device.  Mirrors the C ABI call for call."""

    def __init__(self, nx, ny, nz, velset=D3Q19, ddf_format="FP32", tau=0.6, force=None, collision=BGK,
                 use_torch_memory=True, cells_per_thread=0, variant=0, shifted=True):
        self._h = C.c_void_p()
        self.nx, self.ny, self.nz, self.q = int(nx), int(ny), int(nz), int(velset)
        self.N = self.nx * self.ny * self.nz
        self.fmt = _fmt(ddf_format)
        self.tau = float(tau)
        self._keep = []          # tensors the library holds raw pointers to
        fptr = None
        if force is not None:
            self._force = (C.c_float * 3)(*[float(v) for v in force])
            fptr = C.cast(self._force, C.c_void_p)
        _check(lib().lbm_create(C.byref(self._h), self.nx, self.ny, self.nz, self.q, int(collision), self.fmt,
                                self.tau, fptr))
        if use_torch_memory:
            import torch
            nbytes = ddf_buffer_bytes(self.nx, self.ny, self.nz, self.q, self.fmt)
            a = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
            b = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
            stream = torch.cuda.current_stream().cuda_stream
            self._keep += [a, b]
            _check(lib().lbm_bind(self._h, a.data_ptr(), b.data_ptr(), stream))
        if cells_per_thread:
            _check(lib().lbm_set_cells_per_thread(self._h, int(cells_per_thread)))
        if variant:
            _check(lib().lbm_set_variant(self._h, int(variant)))
        if not shifted:
            _check(lib().lbm_set_shifting(self._h, 0))

    # -- lifetime ------------------------------------------------------------------------------
    def close(self):
        if getattr(self, "_h", None) is not None and self._h:
            lib().lbm_destroy(self._h)
            self._h = C.c_void_p()
            self._keep = []

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    # -- the ABI -------------------------------------------------------------------------------
    def set_cells_per_thread(self, v: int):
        _check(lib().lbm_set_cells_per_thread(self._h, int(v)))

    def set_trt_lambda(self, lam: float):
        _check(lib().lbm_set_trt_lambda(self._h, float(lam)))

    def set_variant(self, v: int):
        _check(lib().lbm_set_variant(self._h, int(v)))

    def set_flags(self, flags):
        flags = np.ascontiguousarray(flags, dtype=np.uint8).reshape(-1)
        if flags.size != self.N:
            raise ValueError("flags must have nx*ny*nz entries")
        _check(lib().lbm_set_flags(self._h, _np_ptr(flags)))

    def init(self, rho, u):
        """rho [N], u [3, N]: numpy float32 (host path, lbm_init) or torch CUDA float32 tensors
        (device path, lbm_init_device)."""
        if _is_torch(rho):
            import torch
            assert rho.is_cuda and u.is_cuda and rho.dtype == torch.float32 and u.dtype == torch.float32
            rho, u = rho.contiguous(), u.contiguous()
            assert rho.numel() == self.N and u.numel() == 3 * self.N
            self._init_keep = (rho, u)
            _check(lib().lbm_init_device(self._h, rho.data_ptr(), u.data_ptr()))
            return
        rho = np.ascontiguousarray(rho, dtype=np.float32).reshape(-1)
        u = np.ascontiguousarray(u, dtype=np.float32).reshape(-1)
        if rho.size != self.N or u.size != 3 * self.N:
            raise ValueError("rho must have N and u 3N entries")
        _check(lib().lbm_init(self._h, _np_ptr(rho), _np_ptr(u)))

    def init_generated(self, seed: int):
        """fields drawn on the device, cell by cell (workloads.generated_fields gives the same values on the host)"""
        _check(lib().lbm_init_generated(self._h, int(seed)))

    def step(self, n: int = 1):
        _check(lib().lbm_step(self._h, int(n)))

    def set_shifting(self, on: bool):
        _check(lib().lbm_set_shifting(self._h, 1 if on else 0))

    def set_graphs(self, enable: bool):
        _check(lib().lbm_set_graphs(self._h, 1 if enable else 0))

    def sync(self):
        _check(lib().lbm_sync(self._h))

    def read_rho_u(self, out=None):
        """Host read-out: returns (rho [N], u [3, N]) float32 numpy arrays.  `out=(rho, u)` reuses
        caller arrays (e.g. views of pinned tensors)."""
        if out is None:
            rho = np.empty(self.N, np.float32)
            u = np.empty((3, self.N), np.float32)
        else:
            rho, u = out
            for a, n in ((rho, self.N), (u, 3 * self.N)):
                if not (isinstance(a, np.ndarray) and a.dtype == np.float32 and a.flags.c_contiguous and a.size == n
                        and a.flags.writeable):
                    raise ValueError("read_rho_u(out=(rho, u)): writable C-contiguous float32 arrays of N and 3N entries")
        _check(lib().lbm_read_rho_u(self._h, _np_ptr(rho), _np_ptr(u)))
        return rho, u

    def read_rho_u_f64(self):
        """Host read-out in double (FP64-arithmetic formats only): (rho [N], u [3, N]) float64."""
        rho = np.empty(self.N, np.float64)
        u = np.empty((3, self.N), np.float64)
        _check(lib().lbm_read_rho_u_f64(self._h, _np_ptr(rho), _np_ptr(u)))
        return rho, u

    def read_rho_u_device(self):
        import torch
        rho = torch.empty(self.N, dtype=torch.float32, device="cuda")
        u = torch.empty((3, self.N), dtype=torch.float32, device="cuda")
        _check(lib().lbm_read_rho_u_device(self._h, rho.data_ptr(), u.data_ptr()))
        return rho, u

    def read_rho_u_at(self, cells):
        """Read-out at selected cells: returns (rho [k], u [3, k])."""
        cells = np.ascontiguousarray(cells, dtype=np.int64).reshape(-1)
        rho = np.empty(cells.size, np.float32)
        u = np.empty((3, cells.size), np.float32)
        _check(lib().lbm_read_rho_u_at(self._h, _np_ptr(cells), cells.size, _np_ptr(rho), _np_ptr(u)))
        return rho, u

    def read_rho_u_at_static(self, cells):
        """read_rho_u_at without any device allocation: the scratch is a fixed array in the library (at most
        STATIC_PROBES_MAX cells per call; shared by all handles -- do not overlap calls).  include/lbm.h."""
        cells = np.ascontiguousarray(cells, dtype=np.int64).reshape(-1)
        rho = np.empty(cells.size, np.float32)
        u = np.empty((3, cells.size), np.float32)
        _check(lib().lbm_read_rho_u_at_static(self._h, _np_ptr(cells), cells.size, _np_ptr(rho), _np_ptr(u)))
        return rho, u

    def read_ddf(self, i: int) -> np.ndarray:
        out = np.empty(self.N, {0: np.float32, 7: np.float64, 8: np.float32}.get(self.fmt, np.uint16))
        _check(lib().lbm_read_ddf(self._h, int(i), _np_ptr(out)))
        return out

    @property
    def steps_done(self) -> int:
        return int(lib().lbm_steps_done(self._h))

    @property
    def kernel_name(self) -> str:
        return lib().lbm_kernel_name(self._h).decode()


def from_workload(w, ddf_format="FP32", **kw) -> Simulation:
    """Build, flag and initialise a Simulation from a workloads.Workload (inputs only)."""
    force = w.force if any(float(v) != 0.0 for v in w.force) else None
    s = Simulation(w.nx, w.ny, w.nz, w.velset, ddf_format, w.tau, force, **kw)
    if w.flags.any():
        s.set_flags(w.flags)
    s.init(w.rho, w.u)
    return s


# ---- codecs (host arrays in, host arrays out; the conversion runs on the GPU) --------------------
def codec_encode(ddf_format, x) -> np.ndarray:
    x = np.ascontiguousarray(x, dtype=np.float32)
    out = np.empty(x.shape, np.uint16)
    _check(lib().lbm_codec_encode(_fmt(ddf_format), _np_ptr(x), _np_ptr(out), x.size))
    return out


def codec_decode(ddf_format, codes) -> np.ndarray:
    codes = np.ascontiguousarray(codes, dtype=np.uint16)
    out = np.empty(codes.shape, np.float32)
    _check(lib().lbm_codec_decode(_fmt(ddf_format), _np_ptr(codes), _np_ptr(out), codes.size))
    return out


def codec_pair_selftest(ddf_format) -> int:
    """Number of bit mismatches between the staged kernel's pair converters and the scalar converters,
    exhaustive over all codes / all FP32 patterns, computed on the GPU (0 = identical)."""
    n = _ll(0)
    _check(lib().lbm_codec_pair_selftest(_fmt(ddf_format), C.byref(n)))
    return int(n.value)


def div_selftest() -> int:
    """Number of bit mismatches between the staged kernel's shared-reciprocal division and IEEE division (0 = identical)."""
    n = _ll(0)
    _check(lib().lbm_div_selftest(C.byref(n)))
    return int(n.value)
