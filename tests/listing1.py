"""An independent, literal transcription of the paper's Listing 1 in numpy.

Purpose: PIN for the oracle's codecs (tests/test_oracle_codecs.py).  The oracle (oracle/codecs.cpp)
defines every format by VALUE (tables + "nearest value" encode); this file re-types the paper's own
BIT-LEVEL converters.  Two differently built descriptions of the same functions must agree where the
paper's listing is well defined.  This file is used by tests only; neither the oracle nor the CUDA
path imports it.

OpenCL semantics kept: shift counts are taken modulo 32 (OpenCL C 6.3.j), `ushort` arithmetic wraps at
16 bits, comparisons yield 0/1.  De-garbled tokens (the extraction damaged the listing) are marked
"[garbled]" with the printed text; DESIGN.md section 3 lists the same readings.
"""
import numpy as np

U32 = np.uint32
I32 = np.int32


def _u(x):
    return np.asarray(x).astype(U32)


def _shl(a, n):
    return (_u(a) << (_u(n) & U32(31))).astype(U32)


def _shr(a, n):          # logical
    return (_u(a) >> (_u(n) & U32(31))).astype(U32)


def _sar(a, n):          # arithmetic (signed int >>)
    return (np.asarray(a).astype(I32) >> (_u(n) & U32(31)).astype(I32)).astype(I32)


def _as_uint(x):
    return np.ascontiguousarray(x, dtype=np.float32).view(U32)


def _as_float(b):
    return np.ascontiguousarray(_u(b)).view(np.float32)


def _float_exp_field(t):
    """as_uint((float)t) >> 23 for small non-negative integers t (exact conversion)."""
    return (_as_uint(np.asarray(t).astype(np.float32)) >> U32(23)).astype(I32)


# ---- FP16C (prose PAPER.md:168-178) -------------------------------------------
def float_to_half_custom(x):
    b = (_as_uint(x) + U32(0x00000800)).astype(U32)          # :813
    e = ((b & U32(0x7F800000)) >> U32(23)).astype(I32)        # :814
    m = b & U32(0x007FFFFF)                                   # :815 [garbled] printed 0x007FFFFFF
    sign = (b & U32(0x80000000)) >> U32(16)
    # :816 [garbled] printed "(e-112)*(11)&0x7800": prose :170 says "bit-shifted ... by 11 places"
    norm = (e > 112) * ((_shl(e - 112, 11) & U32(0x7800)) | (m >> U32(12)))
    den = ((e < 113) & (e > 100)) * (_shr(_shr(U32(0x007FF800) + m, 124 - e) + U32(1), 1))
    sat = (e > 127) * U32(0x7FFF)
    return ((sign | norm | den | sat) & U32(0xFFFF)).astype(np.uint16)


def half_to_float_custom(x):
    x = _u(x)
    e = (x & U32(0x7800)) >> U32(11)                          # :826 [garbled] "x80x7800"
    m = (x & U32(0x07FF)) << U32(12)                          # :827
    v = _float_exp_field(m)                                   # :829
    norm = (e != 0) * (((e + U32(112)) << U32(23)) | m)
    den = ((e == 0) & (m != 0)) * (_shl(v - 37, 23) | (_shl(m, 150 - v) & U32(0x007FF000)))
    return _as_float(((x & U32(0x8000)) << U32(16)) | norm | den)


# ---- P16_0; the load/store macros scale by 2^-7 / 2^7 -----------
def float_to_p160(x):
    b = _as_uint(x)
    e = ((b & U32(0x7F800000)) >> U32(23)).astype(I32) - 127  # :837 [garbled]
    m = ((b & U32(0x007FFFFF)) >> U32(9)).astype(I32)         # :838 [garbled]
    v = np.abs(e)                                             # :841 [garbled] first "const int v"
    r = _shl(np.where(e < 0, U32(0x0002), U32(0xFFFE)), 13 - v)   # :842 [garbled] "0xFFE", second "v"
    m = _sar(_sar(m, v - (e < 0)) + 1 + (e < -13) * 2, 1)     # :843 [garbled] "m>(v-(e<0))"
    sign = (b & U32(0x80000000)) >> U32(16)
    body = (e > -16) * ((r + _u(m)) & U32(0x7FFF))
    sat = (e > 13) * U32(0x7FFF)
    return ((sign | body | sat) & U32(0xFFFF)).astype(np.uint16)


def _regime_run(x):
    """shared head of p160_to_float / p161_to_float."""
    x = _u(x)
    sr = (x >> U32(14)) & U32(1)                              # :848 [garbled] "(x>)14)&1"
    t = (x << U32(2)) & U32(0xFFFF)                           # ushort t = x<<2
    t = np.where(sr == 1, (~t) & U32(0xFFFF), t)              # :850 [garbled] printed "-t"; "~t" decodes 0x4000 to 1.0 (Fig. 2)
    r = 142 - _float_exp_field(t)                             # :851
    return x, sr, r


def p160_to_float(x):
    x, sr, r = _regime_run(x)
    m = _shl(x, r + 10) & U32(0x007FFFFF)                     # :852 [garbled] "(r+i0))&0x007FFFF"
    rs = np.where(sr == 1, r, -r - 1)                         # :853
    # :854 [garbled] printed "(r!=158)"; for the zero code r = 142 - 0 = 142
    return _as_float(((x & U32(0x8000)) << U32(16)) | (r != 142) * (_shl(rs + 127, 23) | m))


# ---- P16_1 -------------------------------------------------------------------
def float_to_p161(x):
    b = _as_uint(x)
    e = ((b & U32(0x7F800000)) >> U32(23)).astype(I32) - 127  # :869
    m = ((b & U32(0x007FFFFF)) >> U32(10)).astype(I32)        # :871
    ae = np.abs(e)                                            # :881 [garbled] "eabs(e)"
    v = ae >> 1                                               # :882
    e2 = ae & 1                                               # :883 [garbled] second "v" line, comment "%2"
    # :884 [garbled] "(e<0 ? 0x0002 : 0xFFFE<e2)+e2)<c((13-v-e2)"
    r = _shl(np.where(e < 0, U32(0x0002), _shl(U32(0xFFFE), e2)) + _u(e2), 13 - v - e2)
    # :885 [garbled] "(e<0)**(1-e2)"
    m = _sar(_sar(m, v - (e < 0) * (1 - e2)) + (e > -28) + (e < -26) * 3, 1)
    sign = (b & U32(0x80000000)) >> U32(16)
    body = (e > -31) * ((r + _u(m)) & U32(0x7FFF))            # :886 [garbled] "(x+m)"
    sat = (e > 26) * U32(0x7FFF)                              # :886 [garbled] "0x3FFFF"
    return ((sign | body | sat) & U32(0xFFFF)).astype(np.uint16)


def p161_to_float(x):
    x, sr, r = _regime_run(x)
    e = _shr(x, 12 - r) & U32(1)                              # :896 [garbled] "(x><(12-r))&i"
    m = _shl(x, r + 11) & U32(0x007FFFFF)                     # :897
    rs = np.where(sr == 1, r, -r - 1) * 2                     # :898
    return _as_float(((x & U32(0x8000)) << U32(16)) | (r != 142) * (_shl(rs + e.astype(I32) + 127, 23) | m))


# ---- P16_2C ------------------------------------------------------------------
def float_to_p162C(x):
    b = _as_uint(x)
    e = ((b & U32(0x7F800000)) >> U32(23)).astype(I32) - 127  # :908 [garbled]
    m = ((b & U32(0x007FFFFF)) >> U32(10)).astype(I32)        # :909
    ae = -e                                                   # :911
    v = ae >> 2                                               # :912
    r = _shr(U32(0x4000), v)                                  # :913
    e4 = _shl(3 - (ae & 3), 12 - v)                           # :914
    m = _sar(_sar(m, v) + (e > -54) + (e < -51) * 3, 1)       # :915
    sign = (b & U32(0x80000000)) >> U32(16)
    body = (e > -59) * ((r + e4 + _u(m)) & U32(0x7FFF))       # :919
    sat = (e > 0) * U32(0x7FFF)
    return ((sign | body | sat) & U32(0xFFFF)).astype(np.uint16)


def p162C_to_float(x):
    x = _u(x)
    r = 158 - _float_exp_field((x << U32(17)) & U32(0xFFFFFFFF))   # :922
    e = _shr(x, 12 - r) & U32(3)                              # :923 [garbled] "(12-7)"
    m = _shl(x, r + 11) & U32(0x007FFFFF)                     # :924
    return _as_float(((x & U32(0x8000)) << U32(16)) | (r != 158) * (_shl(124 - (r << 2) + e.astype(I32), 23) | m))


# store / load macros of Listing 1: the scale is an FP32 multiply
STORE = {
    "FP16C": lambda x: float_to_half_custom(x),
    "P16_0S": lambda x: float_to_p160(np.asarray(x, np.float32) * np.float32(128.0)),
    "P16_1S": lambda x: float_to_p161(np.asarray(x, np.float32) * np.float32(128.0)),
    "P16_2C": lambda x: float_to_p162C(x),
}
LOAD = {
    "FP16C": lambda c: half_to_float_custom(c),
    "P16_0S": lambda c: p160_to_float(c) * np.float32(0.0078125),
    "P16_1S": lambda c: p161_to_float(c) * np.float32(0.0078125),
    "P16_2C": lambda c: p162C_to_float(c),
}
