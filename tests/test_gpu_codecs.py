"""GPU parity: device codecs (lbm_codec_encode / lbm_codec_decode through the C ABI) vs the oracle.

Bar: bit-exact.  decode over all 65 536 codes of every 16-bit format; encode over (a) seeded inputs in
every binade with both signs, (b) every table value, every midpoint between neighbouring table values
and their FP32 neighbours (the tie / boundary cases of each format), (c) specials, (d) 2^24 random bit
patterns.  NaN results of FP16 / FP16S are compared as "is a NaN code" (the hardware conversion and the
oracle pick different NaN payloads).
"""
import numpy as np
import pytest

import oracle
import paper_2112_08926_b200 as lbm
from workloads import FORMATS, codec_probe_inputs

pytestmark = pytest.mark.gpu
FMT16 = ["FP16S", "FP16C", "P16_0S", "P16_1S", "P16_2C", "FP16"]
ALL_CODES = np.arange(65536, dtype=np.uint32).astype(np.uint16)


def _same_bits(a, b):
    return np.array_equal(a.view(np.uint32), b.view(np.uint32))


@pytest.mark.parametrize("name", FMT16)
def test_decode_all_codes_bit_exact(name):
    fmt = FORMATS[name]
    got = lbm.codec_decode(name, ALL_CODES)
    want = oracle.decode(fmt, ALL_CODES)
    nan = np.isnan(want)
    assert np.array_equal(np.isnan(got), nan)
    assert _same_bits(got[~nan], want[~nan])


def _boundary_inputs(fmt):
    """table values, midpoints and their FP32 neighbours, from the ORACLE's value table."""
    mags = np.arange(0x8000, dtype=np.uint32).astype(np.uint16)
    v = oracle.decode(fmt, mags).astype(np.float64)
    v = v[np.isfinite(v)]
    mid = ((v[:-1] + v[1:]) / 2).astype(np.float32)
    base = np.concatenate([v.astype(np.float32), mid])
    bits = base.view(np.uint32).astype(np.int64)
    out = [np.clip(bits + d, 0, 0x7F7FFFFF).astype(np.uint32).view(np.float32) for d in (-2, -1, 0, 1, 2)]
    x = np.concatenate(out)
    return np.concatenate([x, -x])


@pytest.mark.parametrize("name", FMT16)
def test_encode_bit_exact(name):
    fmt = FORMATS[name]
    rng = np.random.default_rng(42)
    x = np.concatenate([codec_probe_inputs(seed=3), _boundary_inputs(fmt),
                        rng.integers(0, 2 ** 32, 1 << 24, dtype=np.uint64).astype(np.uint32).view(np.float32)])
    got = lbm.codec_encode(name, x)
    want = oracle.encode(fmt, x)
    if name in ("FP16", "FP16S"):
        nan = np.isnan(x)
        assert np.all((got[nan] & 0x7C00) == 0x7C00) and np.all((got[nan] & 0x03FF) != 0)
        got, want = got[~nan], want[~nan]
    bad = np.nonzero(got != want)[0]
    assert bad.size == 0, [(float(x[i]), hex(got[i]), hex(want[i])) for i in bad[:8]]


@pytest.mark.parametrize("name", FMT16)
def test_roundtrip_on_device(name):
    finite = ALL_CODES if name not in ("FP16", "FP16S") else ALL_CODES[(ALL_CODES & 0x7C00) != 0x7C00]
    assert np.array_equal(lbm.codec_encode(name, lbm.codec_decode(name, finite)), finite)


def test_corner_thresholds_on_device():
    """The class-B corner vectors (tests/golden/codec_corner_vectors.txt) through the device encoders."""
    from .test_oracle_codecs import corner_vectors
    for name, x, at, below in corner_vectors():
        lo = np.nextafter(x, np.float32(0))
        got = lbm.codec_encode(name, np.array([x, lo, -x, -lo], np.float32))
        assert [int(c) for c in got] == [at, below, at | 0x8000, below | 0x8000], (name, float(x), [hex(int(c)) for c in got])


def test_codec_edge_cases():
    assert lbm.codec_encode("FP16C", np.zeros(0, np.float32)).size == 0
    with pytest.raises(lbm.LbmError):
        lbm.codec_encode("FP32", np.zeros(4, np.float32))


@pytest.mark.parametrize("name", [n for n in FORMATS if n != "FP32"])
def test_pair_codecs_equal_scalar_codecs_exhaustively(name):
    """The staged kernel's converters (PairCodec) vs the scalar ones (compared with the oracle above): all 65 536
    codes and all 2^32 FP32 bit patterns, on the device."""
    assert lbm.codec_pair_selftest(name) == 0


def test_shared_division_equals_ieee_division():
    """The staged kernel's u = j / rho with one shared reciprocal (div3) vs __fdiv_rn, ~10^8 pairs incl. signed zero
    numerators, on the device."""
    assert lbm.div_selftest() == 0
