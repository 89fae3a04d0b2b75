"""Pins for the oracle's storage-format codecs (oracle/codecs.cpp) -- CPU only.

The oracle defines each format by value; these tests check it against what the PAPER fixes:
  * Table 2 constants (tests/golden/table2_formats.txt)
  * the accuracy intervals of PAPER.md:205-207 (tests/golden/posit_intervals.txt)
  * an independent literal transcription of Listing 1 (tests/listing1.py)
  * IEEE binary16 as implemented by numpy (a library, for FP16 / FP16S)
  * invariants: strict monotonicity, sign symmetry, exhaustive round trip (north_star)
chosen so that a wrong bias, scale, regime rule, mantissa width, rounding direction or saturation fails.
"""
import os

import numpy as np
import pytest

import oracle
from workloads import FORMATS, codec_probe_inputs

from . import listing1

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
FMT16 = ["FP16S", "FP16C", "P16_0S", "P16_1S", "P16_2C", "FP16"]
SOFT = ["FP16C", "P16_0S", "P16_1S", "P16_2C"]
ALL_CODES = np.arange(65536, dtype=np.uint32).astype(np.uint16)


def finite_mags(name):
    return np.arange(0x7C00 if name in ("FP16", "FP16S") else 0x8000, dtype=np.uint32).astype(np.uint16)


def values(name):
    """decoded (scaled) value of every finite magnitude, float64."""
    return oracle.decode(FORMATS[name], finite_mags(name)).astype(np.float64)


def _table2():
    rows = {}
    for line in open(os.path.join(GOLDEN, "table2_formats.txt")):
        if line.startswith("#") or not line.strip():
            continue
        name, nm, eps, vmax, vnorm, vden = line.split()
        rows[name] = (int(nm), float(eps), float(vmax), vnorm, float(vden))
    return rows


@pytest.mark.parametrize("name", FMT16)
def test_table2_constants(name):
    nm, eps, vmax, vnorm, vden = _table2()[name]
    v = values(name)
    assert v[0] == 0.0
    assert v[-1] == pytest.approx(vmax, rel=5e-7)                # printed with 7 digits
    assert v[1] == pytest.approx(vden, rel=5e-7)                 # smallest (denormal) number
    # finest relative spacing anywhere in the table = 2^-n_m = epsilon
    rel = np.diff(v[1:]) / 2.0 ** np.floor(np.log2(v[1:-1]))     # spacing relative to the binade base
    assert rel.min() == pytest.approx(2.0 ** -nm, rel=1e-12)
    assert 2.0 ** -nm == pytest.approx(eps, rel=0.03)            # printed with 2 digits
    if vnorm != "-":
        # smallest normal number = first value from which the relative spacing is 2^-n_m
        first_normal = v[1:-1][np.isclose(rel, 2.0 ** -nm, rtol=1e-12)][0]
        if vnorm.startswith("!"):
            assert first_normal == 2.0 ** -29                    # see the fixture header
            assert first_normal != pytest.approx(float(vnorm[1:]), rel=5e-7)
        else:
            assert first_normal == pytest.approx(float(vnorm), rel=5e-7)


@pytest.mark.parametrize("name", FMT16)
def test_monotone_symmetric_roundtrip(name):
    fmt = FORMATS[name]
    v = values(name)
    assert np.all(np.diff(v) > 0), "decode must be strictly increasing over the magnitude codes"
    mags = finite_mags(name)
    neg = oracle.decode(fmt, mags | np.uint16(0x8000))
    assert np.array_equal(neg, -oracle.decode(fmt, mags))
    assert np.signbit(neg[0]) and not np.signbit(oracle.decode(fmt, mags[:1])[0])   # both zeros exist
    codes = np.concatenate([mags, mags | np.uint16(0x8000)])
    assert np.array_equal(oracle.encode(fmt, oracle.decode(fmt, codes)), codes), "encode(decode(c)) == c"


@pytest.mark.parametrize("name", FMT16)
def test_nearest_and_saturation(name):
    """encode returns a nearest table value for random inputs (brute force against the table)."""
    fmt = FORMATS[name]
    v = values(name)
    rng = np.random.default_rng(5)
    x = np.ldexp(rng.uniform(1, 2, 20000), rng.integers(-45, 2, 20000)).astype(np.float32)
    x = x[np.abs(x) <= v[-1]]
    c = oracle.encode(fmt, x)
    got = np.abs(oracle.decode(fmt, c).astype(np.float64))
    idx = np.searchsorted(v, np.abs(x.astype(np.float64)))
    idx = np.clip(idx, 1, len(v) - 1)
    lo, hi = v[idx - 1], v[idx]
    ax = np.abs(x.astype(np.float64))
    dist_best = np.minimum(ax - lo, hi - ax)
    assert np.all(np.abs(got - ax) == dist_best)
    big = np.array([4.0, 1e3, 1e30, np.inf], np.float32) * np.float32(v[-1])
    if name in ("FP16", "FP16S"):
        assert np.all(oracle.encode(fmt, big) == 0x7C00)         # IEEE overflow -> Inf (PAPER.md:156 hardware cvt)
        assert np.all(oracle.encode(fmt, -big) == 0xFC00)
    else:
        assert np.all(oracle.encode(fmt, big) == 0x7FFF)         # saturation
        assert np.all(oracle.encode(fmt, -big) == 0xFFFF)
        assert oracle.encode(fmt, np.array([np.nan], np.float32))[0] & 0x7FFF == 0x7FFF


@pytest.mark.parametrize("name", SOFT)
def test_ties_go_to_larger_magnitude(name):
    """add-half-then-truncate = ties away from zero; FP16 family = ties to even."""
    fmt = FORMATS[name]
    v = values(name)
    mid = (v[:-1] + v[1:]) / 2
    ok = mid.astype(np.float32).astype(np.float64) == mid        # midpoints representable in FP32
    assert ok.sum() > 30000
    m = mid[ok].astype(np.float32)
    expect = (np.nonzero(ok)[0] + 1).astype(np.uint16)
    assert np.array_equal(oracle.encode(fmt, m), expect)
    assert np.array_equal(oracle.encode(fmt, -m), expect | np.uint16(0x8000))
    below = np.nextafter(m, np.float32(0))
    assert np.array_equal(oracle.encode(fmt, below), expect - 1)


@pytest.mark.parametrize("name", ["FP16", "FP16S"])
def test_ieee_half_against_numpy(name):
    """FP16S = IEEE binary16 RNE of x*2^15: numpy's float16 is an independent IEEE library."""
    fmt = FORMATS[name]
    scale = np.float32(32768.0 if name == "FP16S" else 1.0)
    with np.errstate(over="ignore", invalid="ignore"):
        half = oracle.decode(fmt, ALL_CODES)
        ref = ALL_CODES.view(np.float16).astype(np.float32) * (np.float32(1.0) / scale)
        assert np.array_equal(half.view(np.uint32)[~np.isnan(ref)], ref.view(np.uint32)[~np.isnan(ref)])
        assert np.all(np.isnan(half[np.isnan(ref)]))
        x = codec_probe_inputs(seed=3, per_binade=2048)
        v = values(name)
        mid = ((v[:-1] + v[1:]) / 2).astype(np.float32)          # exact: one extra mantissa bit
        x = np.concatenate([x, mid, -mid, np.nextafter(mid, np.float32(0)), np.nextafter(mid, np.float32(9))])
        want = (x * scale).astype(np.float16).view(np.uint16)
        got = oracle.encode(fmt, x)
        nan = np.isnan(x)
        assert np.array_equal(got[~nan], want[~nan])
        assert np.all((got[nan] & 0x7C00) == 0x7C00) and np.all((got[nan] & 0x03FF) != 0)


@pytest.mark.parametrize("name", SOFT)
def test_listing1_decode_all_codes(name):
    """The paper's bit-level loader, transcribed independently, decodes every code to the oracle's value."""
    got = oracle.decode(FORMATS[name], ALL_CODES)
    ref = listing1.LOAD[name](ALL_CODES)
    diff = np.nonzero(got.view(np.uint32) != ref.view(np.uint32))[0]
    if name == "P16_2C":
        # codes 0x0003 / 0x8003: one exponent bit left after a 13-zero regime.  The listing's
        # `x>>(12-r)` has a negative shift count there and yields a duplicate of code 0x0002's value
        # (not monotone); the oracle reads the remaining bit as the high exponent bit (G7).
        assert set(diff.tolist()) == {0x0003, 0x8003}
        assert ref[3] == ref[2] and got[3] == 4 * got[2]
    else:
        assert diff.size == 0


# regular domain of |x| on which Listing 1 rounds to the nearest value (outside it the listing cuts
# exponent bits geometrically or wraps; R14): (lo, hi) as powers of two, None = unbounded
REGULAR = {"FP16C": (None, None), "P16_0S": (None, None), "P16_1S": (-33, 19), "P16_2C": (-51, None)}


@pytest.mark.parametrize("name", SOFT)
def test_listing1_encode(name):
    """The paper's bit-level store equals the oracle's 'nearest value, ties up, saturate' on random
    inputs of every binade and on every rounding boundary (each midpoint of adjacent values, its two
    FP32 neighbours, and the values themselves)."""
    fmt = FORMATS[name]
    v = values(name)
    mid = ((v[:-1] + v[1:]) / 2).astype(np.float32)
    pts = np.concatenate([mid, np.nextafter(mid, np.float32(0)), np.nextafter(mid, np.float32(9)),
                          v.astype(np.float32), codec_probe_inputs(seed=11, per_binade=8192)])
    pts = pts[np.isfinite(pts)]
    x = np.concatenate([pts, -pts]).astype(np.float32)
    lo, hi = REGULAR[name]
    ax = np.abs(x.astype(np.float64))
    keep = np.ones(x.shape, bool)
    if lo is not None:
        keep &= (ax >= 2.0 ** lo) | (ax == 0)
    if hi is not None:
        keep &= ax < 2.0 ** hi
    if name == "P16_2C":
        keep &= ax < 2.0 - 2.0 ** -13          # the listing's rounding carry wraps to code 0 in [2-2^-13, 2)
    x = x[keep]
    assert x.size > 1_000_000
    got = oracle.encode(fmt, x)
    ref = listing1.STORE[name](x)
    bad = np.nonzero(got != ref)[0]
    assert bad.size == 0, (x[bad[:5]], got[bad[:5]], ref[bad[:5]])


def test_posit_accuracy_intervals():
    """binades in which each posit resolves at least as finely as FP16S / FP16C."""
    def per_binade(name):
        v = values(name)[1:]
        k = np.floor(np.log2(v)).astype(int)
        return {kk: int(np.sum(k == kk)) for kk in range(-45, 3)}
    counts = {n: per_binade(n) for n in ["FP16S", "FP16C", "P16_0S", "P16_1S", "P16_2C"]}
    for line in open(os.path.join(GOLDEN, "posit_intervals.txt")):
        if line.startswith("#") or not line.strip():
            continue
        posit, other, lo, hi = line.split()
        lo, hi = int(lo), int(hi)
        for k in range(lo, hi):
            assert counts[posit][k] >= counts[other][k], (posit, other, k)
        assert counts[posit][lo - 1] < counts[other][lo - 1], (posit, other, "below", lo)
        if hi < 1:
            assert counts[posit][hi] < counts[other][hi], (posit, other, "above", hi)


def corner_vectors():
    """tests/golden/codec_corner_vectors.txt -> [(format, x at the threshold (float32), code at, code just below)]"""
    out = []
    for line in open(os.path.join(GOLDEN, "codec_corner_vectors.txt")):
        if line.startswith("#") or not line.strip():
            continue
        name, scale, t, at, below = line.split()
        mant, exp = t.split("*2^")
        x = np.float64(mant) * 2.0 ** int(exp) / float(scale)
        assert np.float64(np.float32(x)) == x, (name, t)          # every threshold is an FP32 number
        out.append((name, np.float32(x), int(at, 16), int(below, 16)))
    return out


def test_corner_thresholds():
    """Class-B corners (R14): the first codes above zero and the step into the saturating code, exactly at
    the midpoints the value tables fix and one FP32 step below them, both signs -- the regions test_listing1_encode
    has to mask out because the listing is not nearest-value there."""
    for name, x, at, below in corner_vectors():
        fmt = FORMATS[name]
        lo = np.nextafter(x, np.float32(0))
        got = oracle.encode(fmt, np.array([x, lo, -x, -lo], np.float32))
        assert [int(c) for c in got] == [at, below, at | 0x8000, below | 0x8000], (name, float(x), [hex(int(c)) for c in got])
    # beyond the largest number every software format saturates; zero keeps its sign
    for name in SOFT:
        got = oracle.encode(FORMATS[name], np.array([3.0, 1e30, np.inf, -1e30, 0.0, -0.0], np.float32))
        big = 0x7FFF
        if name in ("P16_0S", "P16_1S"):
            assert int(got[0]) < big                                # 3 is inside their range
            got = got[1:]
            assert [int(c) for c in got] == [big, big, big | 0x8000, 0, 0x8000], name
        else:
            assert [int(c) for c in got] == [big, big, big, big | 0x8000, 0, 0x8000], name
