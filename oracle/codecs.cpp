// oracle/codecs.cpp -- CPU oracle for the DDF storage formats.  TEST INFRASTRUCTURE, NOT PRODUCT
// (see oracle.h).  Shares no code with the CUDA codecs.
//
// What is defined here, and from where:
//   * the VALUE every 16-bit code stands for, written as arithmetic (ldexp), never as bit tricks:
//       FP16    IEEE-754 binary16, 1-5-10, bias 15                 PAPER.md:129, Table 2
//       FP16S   binary16 value x 2^-15 ("bias 30")
//       FP16C   1-4-11, bias 15, denormals, no Inf/NaN              PAPER.md:148, 166-178, Table 2 :141
//       P16_0S  posit<16,0> magnitude, sign bit, x 2^-7             PAPER.md:184-195 eq (8), 205, 219, 799
//       P16_1S  posit<16,1> magnitude, sign bit, x 2^-7
//       P16_2C  one-sided regime, 2 exponent bits, not scaled
//   * store(): the paper's converters add half an output ulp and truncate ("+0x00000800",
//     :843/:885/:915 "+1 ... >>1"), i.e. round to the NEAREST representable value with ties to the
//     larger magnitude, and saturate at the largest code.  The oracle states that
//     as a definition ("rule U", R14): nearest table value, tie -> larger code, above the
//     maximum -> 0x7FFF, sign bit copied.  FP16 / FP16S use the hardware conversion the paper names
//     (vstore_half_rte): IEEE round-to-nearest-even with overflow to infinity.
//   * load(): table value, times the inverse power-of-two scale -- exact in FP32.
//
// Readings of garbled / inconsistent passages (all listed in DESIGN.md section 3):
//   - eq (8) prints the regime base as (2^(n_e+1))^r; Table 2's smallest P16_2C number 2^-59 and the
//     listing's `124-(r<<2)+e` need 16^r for n_e = 2, i.e. base 2^(2^n_e) (2, 4, 16).
//   - exponent bits cut off by a long regime count as 0; if one of P16_2C's two bits is left it is the
//     HIGH bit (posit convention), which keeps the value table strictly monotone.
//
// PARITY UNPINNED: the class-B corners of rule U (P16_1S outside 2^-33 <= |x| < 2^19, P16_2C below 2^-51 and in
// [2 - 2^-13, 2)), where the paper's listing is not a nearest-value converter (R14).
// Pins (tests/test_oracle_codecs.py): Table 2 constants, strict monotonicity, exhaustive round trip,
// numpy float16 for FP16/FP16S, and an independent transcription of Listing 1 kept in tests/.
#include "oracle.h"

#include <cmath>
#include <cstring>
#include <limits>
#include <vector>

namespace {

const unsigned MAG_MAX = 0x7FFF;

// ---- value of a magnitude field ---------------------------------------------------------------
// IEEE binary16 (eq (7): (-1)^s 2^(e-b) (1 + 2^-nm m), denormals when e = 0)
double value_fp16(unsigned mag) {
    const unsigned e = mag >> 10, m = mag & 0x3FF;
    if (e == 31) return m ? std::numeric_limits<double>::quiet_NaN() : std::numeric_limits<double>::infinity();
    if (e == 0) return std::ldexp((double)m, -24);           // m * 2^-10 * 2^(1-15)
    return std::ldexp(1.0 + m / 1024.0, (int)e - 15);
}

// FP16C: one exponent bit less, one mantissa bit more, bias still 15, no Inf/NaN
double value_fp16c(unsigned mag) {
    const unsigned e = mag >> 11, m = mag & 0x7FF;
    if (e == 0) return std::ldexp((double)m, -25);           // m * 2^-11 * 2^(1-15)
    return std::ldexp(1.0 + m / 2048.0, (int)e - 15);
}

// Two-sided posit magnitude with n_e exponent bits in a 15-bit field:
// regime = run of k identical leading bits, closed by one terminator bit of the opposite value
// (absent when the run fills the field); r = k-1 for a run of ones, r = -k for a run of zeros
// (PAPER.md:193); then n_e exponent bits, then the mantissa, as far as bits are left.
double value_posit(unsigned mag, int n_e) {
    if (mag == 0) return 0.0;
    int bit[15];
    for (int p = 0; p < 15; ++p) bit[p] = (mag >> (14 - p)) & 1;  // bit[0] is the leftmost
    int k = 1;
    while (k < 15 && bit[k] == bit[0]) ++k;
    const int r = bit[0] ? k - 1 : -k;
    int pos = k + 1;                                               // skip the terminator
    int e = 0;
    for (int j = 0; j < n_e; ++j) {                                // missing exponent bits read as 0
        e <<= 1;
        if (pos < 15) e |= bit[pos];
        ++pos;
    }
    int nf = 0;
    double F = 0.0;
    for (; pos < 15; ++pos) { F = 2.0 * F + bit[pos]; ++nf; }
    const double frac = 1.0 + (nf ? std::ldexp(F, -nf) : 0.0);
    return std::ldexp(frac, r * (1 << n_e) + e);
}

// P16_2C: only the lower flank is covered, so there is no regime sign: the regime is the
// run of r leading ZEROS (r = 0..14) closed by a 1; then 2 exponent bits, then the mantissa.
// value = 2^(e - 3 - 4 r) (1 + F)  (PAPER.md:925 `124-(r<<2)+e` is 127 - 3 - 4r + e);
// largest value (2 - 2^-12), smallest 2^-59 (Table 2).
double value_p162c(unsigned mag) {
    if (mag == 0) return 0.0;
    int bit[15];
    for (int p = 0; p < 15; ++p) bit[p] = (mag >> (14 - p)) & 1;
    int r = 0;
    while (bit[r] == 0) ++r;                                       // mag != 0, so this stops
    int pos = r + 1;
    int e = 0;
    for (int j = 0; j < 2; ++j) {
        e <<= 1;
        if (pos < 15) e |= bit[pos];
        ++pos;
    }
    int nf = 0;
    double F = 0.0;
    for (; pos < 15; ++pos) { F = 2.0 * F + bit[pos]; ++nf; }
    const double frac = 1.0 + (nf ? std::ldexp(F, -nf) : 0.0);
    return std::ldexp(frac, e - 3 - 4 * r);
}

double table_value(int fmt, unsigned mag) {
    switch (fmt) {
        case ORC_FP16:
        case ORC_FP16S: return value_fp16(mag);
        case ORC_FP16C: return value_fp16c(mag);
        case ORC_P16_0S: return value_posit(mag, 0);
        case ORC_P16_1S: return value_posit(mag, 1);
        case ORC_P16_2C: return value_p162c(mag);
    }
    return std::numeric_limits<double>::quiet_NaN();
}

// scale applied by store(); load() applies its inverse
double scale_of(int fmt) {
    switch (fmt) {
        case ORC_FP16S: return 32768.0;     // 2^15
        case ORC_P16_0S:
        case ORC_P16_1S: return 128.0;      // 2^7
    }
    return 1.0;
}

struct Table {
    std::vector<double> v;   // finite table values, ascending, v[mag]
    bool ieee;               // FP16 / FP16S: RNE + overflow to Inf
};

const Table &table_of(int fmt) {
    static Table tabs[8];
    static bool built[8] = {false};
    Table &t = tabs[fmt];
    if (!built[fmt]) {
        t.ieee = (fmt == ORC_FP16 || fmt == ORC_FP16S);
        const unsigned last = t.ieee ? 0x7BFF : MAG_MAX;   // 0x7C00.. are Inf/NaN in binary16
        t.v.resize(last + 1);
        for (unsigned m = 0; m <= last; ++m) t.v[m] = table_value(fmt, m);
        built[fmt] = true;
    }
    return t;
}

uint16_t encode_one(int fmt, float x) {
    uint32_t bits;
    std::memcpy(&bits, &x, 4);
    const uint16_t sign = (uint16_t)((bits >> 16) & 0x8000);
    const Table &t = table_of(fmt);
    // the store macro multiplies in FP32 before converting
    const float xs = x * (float)scale_of(fmt);
    if (std::isnan(xs)) return sign | (t.ieee ? 0x7E00 : 0x7FFF);
    const double X = std::fabs((double)xs);
    const unsigned last = (unsigned)t.v.size() - 1;
    // largest lo with v[lo] <= X
    unsigned lo = 0, hi = last;
    while (lo < hi) {
        const unsigned mid = (lo + hi + 1) / 2;
        if (t.v[mid] <= X) lo = mid; else hi = mid - 1;
    }
    if (lo == last) {
        if (!t.ieee) return sign | MAG_MAX;                        // saturate
        // binary16: values at or above max + half ulp (65504 + 16) round to infinity
        return sign | (X >= 65520.0 ? 0x7C00 : 0x7BFF);
    }
    const double below = X - t.v[lo], above = t.v[lo + 1] - X;     // exact in double
    unsigned code;
    if (below < above) code = lo;
    else if (below > above) code = lo + 1;
    else code = t.ieee ? ((lo & 1) ? lo + 1 : lo)                  // tie: even code (vstore_half_rte)
                       : lo + 1;                                   // tie: larger magnitude (rule U)
    return sign | (uint16_t)code;
}

float decode_one(int fmt, uint16_t code) {
    const double v = table_value(fmt, code & 0x7FFF) / scale_of(fmt);   // power-of-two scale: exact
    const float f = (float)v;                                            // every value is an FP32 number
    return (code & 0x8000) ? -f : f;
}

}  // namespace

extern "C" {

double orc_table_value(int fmt, unsigned mag) { return table_value(fmt, mag & 0x7FFF); }
double orc_scale(int fmt) { return scale_of(fmt); }

int orc_decode(int fmt, const uint16_t *codes, float *out, long n) {
    if (fmt < ORC_FP16S || fmt > ORC_FP16) return -1;
    for (long i = 0; i < n; ++i) out[i] = decode_one(fmt, codes[i]);
    return 0;
}

int orc_encode(int fmt, const float *x, uint16_t *out, long n) {
    if (fmt < ORC_FP16S || fmt > ORC_FP16) return -1;
    table_of(fmt);
#pragma omp parallel for schedule(static)
    for (long i = 0; i < n; ++i) out[i] = encode_one(fmt, x[i]);
    return 0;
}

}  // extern "C"

// used by lbm.cpp (same library, oracle-internal)
uint16_t orc_encode_one(int fmt, float x) { return encode_one(fmt, x); }
float orc_decode_one(int fmt, uint16_t c) { return decode_one(fmt, c); }
void orc_prepare_table(int fmt) { if (fmt >= ORC_FP16S && fmt <= ORC_FP16) table_of(fmt); }
