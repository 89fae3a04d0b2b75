// lbm_codecs.cuh -- device-side load()/store() of the DDF storage formats.
//
// Every decoder returns exactly the value the format's definition assigns to the code (Table 2,
// PAPER.md:134-146; eq (7)/(8)) and every encoder returns the NEAREST
// representable value, ties to the larger magnitude, saturating at the largest code (what the paper's
// converters do by adding half an output ulp and truncating);
// FP16/FP16S use the hardware binary16 conversion with round-to-nearest-even.
// The bit manipulation below is NOT the paper's Listing 1 (written for 2021 OpenCL devices, with data
// dependent selects and an int->float conversion as a leading-zero counter): it is re-derived for
// sm_100a from the value definitions, branch-free on the regular domain:
//   FP16C   decode: place the 15 magnitude bits at FP32 bits 26..12 and multiply by 2^112 (the e = 0
//           codes become FP32 denormals, which the multiply normalises -- needs -ftz=false);
//           encode: multiply |x| by 2^-112 rounding toward zero, add half an ulp (0x800), shift.
//   posits  decode: one FLO (clz) gives the regime length; regime, exponent bits and fraction are
//           merged into the FP32 word with one shift and one add (the exponent bits land on the low
//           bits of the FP32 exponent field);
//           encode: build the unbounded posit string "10|e|M" / "01|e|M" in a 32-bit word, one
//           arithmetic shift by the regime length produces the run, then add-half-and-truncate.
//           Where a long regime cuts exponent bits off, string rounding is geometric, not nearest:
//           those slivers (|x| < 2^-33 or >= 2^19 for P16_1S, |x| < 2^-51 for P16_2C) take a rarely
//           executed patch so that the result is the nearest value there too (R14).
#pragma once
#include <cuda_fp16.h>
#include <stdint.h>

namespace lbmk {

enum : int { F_FP32 = 0, F_FP16S = 1, F_FP16C = 2, F_P16_0S = 3, F_P16_1S = 4, F_P16_2C = 5, F_FP16 = 6 };

template <int F>
struct Codec;

// ---- FP32: identity ---------------------------------------------------------
template <>
struct Codec<F_FP32> {
    typedef float elem_t;
    static __device__ __forceinline__ float dec(float s) { return s; }
    static __device__ __forceinline__ float enc(float x) { return x; }
};

// ---- IEEE binary16 --------------------------------------------------------------
template <>
struct Codec<F_FP16> {
    typedef unsigned short elem_t;
    static __device__ __forceinline__ float dec(unsigned c) {
        return __half2float(__ushort_as_half((unsigned short)c));
    }
    static __device__ __forceinline__ unsigned enc(float x) { return __half_as_ushort(__float2half_rn(x)); }
};

// ---- FP16S: binary16 of x * 2^15 -----------------------------------
template <>
struct Codec<F_FP16S> {
    typedef unsigned short elem_t;
    static __device__ __forceinline__ float dec(unsigned c) {
        return __fmul_rn(__half2float(__ushort_as_half((unsigned short)c)), 3.0517578125e-5f);  // 2^-15, exact
    }
    static __device__ __forceinline__ unsigned enc(float x) {
        return __half_as_ushort(__float2half_rn(__fmul_rn(x, 32768.0f)));
    }
};

// ---- FP16C: 1-4-11, bias 15, denormals, no Inf/NaN ----------------------
template <>
struct Codec<F_FP16C> {
    typedef unsigned short elem_t;
    static __device__ __forceinline__ float dec(unsigned c) {
        const unsigned b = ((c & 0x8000u) << 16) | ((c & 0x7FFFu) << 12);
        return __fmul_rn(__uint_as_float(b), __uint_as_float(0x77800000u));  // * 2^112 (exact)
    }
    static __device__ __forceinline__ unsigned enc(float x) {
        const unsigned xb = __float_as_uint(x);
        const float y = __fmul_rz(__uint_as_float(xb & 0x7FFFFFFFu), __uint_as_float(0x07800000u));  // |x| * 2^-112
        const unsigned m = min((__float_as_uint(y) + 0x800u) >> 12, 0x7FFFu);
        return ((xb >> 16) & 0x8000u) | m;
    }
};

// ---- two-sided posit magnitude with NE exponent bits, scaled by 2^7 --
template <int NE>
struct PositS {
    static __device__ __forceinline__ float dec(unsigned c) {
        const unsigned mm = c << 17;                        // 15-bit magnitude, top aligned
        const int sg = (int)mm >> 31;                       // -1: regime of ones, 0: regime of zeros
        const unsigned t = (mm ^ (unsigned)sg) | 0x10000u;  // guard bit: run length k <= 15
        const int k = __clz((int)t);
        const unsigned rem = mm << (k + 1);                 // exponent bit(s) + fraction, top aligned
        const int r = (k - 1) ^ ~sg;                        // k-1 (ones) or -k (zeros)
        // value = 2^((r << NE) + e) * (1 + F) * 2^-7; e rides on the low exponent bits of the add
        const unsigned bits = ((unsigned)(r * (1 << NE) + 120) << 23) + (rem >> (9 - NE));
        const unsigned sign = (c & 0x8000u) << 16;
        return __uint_as_float((c & 0x7FFFu) ? (bits | sign) : sign);
    }
    static __device__ __forceinline__ unsigned enc(float x) {
        const unsigned xb = __float_as_uint(x);
        const unsigned Xb = __float_as_uint(__fmul_rn(__uint_as_float(xb & 0x7FFFFFFFu), 128.0f));
        const int E = (int)(Xb >> 23) - 127;
        const int r = E >> NE;
        const unsigned e = (unsigned)E & ((1u << NE) - 1u);
        const unsigned W = (r >= 0 ? 0x80000000u : 0x40000000u) | (e << (30 - NE)) | ((Xb & 0x007FFFFFu) << (7 - NE));
        const int sh = min(r ^ (r >> 31), 31);              // r (ones run) or -r-1 (zeros run)
        const unsigned Ws = (unsigned)((int)W >> sh);
        unsigned code = min(((Ws >> 16) + 1u) >> 1, 0x7FFFu);
        if (NE == 1) {
            // exponent bit cut off by the regime: nearest-value thresholds instead of the string's
            const unsigned LO = 0x32800000u /* 2^-26 */, HI = 0x4C800000u /* 2^26 */;
            if (Xb - LO >= HI - LO) {
                code = Xb < LO ? (unsigned)(Xb >= 0x31000000u /* 2^-29 */) + (unsigned)(Xb >= 0x32200000u /* 1.25*2^-27 */)
                               : 0x7FFEu + (unsigned)(Xb >= 0x4D200000u /* 1.25*2^27 */);
            }
        }
        return ((xb >> 16) & 0x8000u) | code;
    }
};
template <>
struct Codec<F_P16_0S> : PositS<0> {
    typedef unsigned short elem_t;
};
template <>
struct Codec<F_P16_1S> : PositS<1> {
    typedef unsigned short elem_t;
};

// ---- P16_2C: regime of zeros only, 2 exponent bits, unscaled ----
template <>
struct Codec<F_P16_2C> {
    typedef unsigned short elem_t;
    static __device__ __forceinline__ float dec(unsigned c) {
        const unsigned mm = c << 17;
        const int r = __clz((int)(mm | 0x10000u));          // 0..15
        const unsigned rem = mm << (r + 1);
        const unsigned bits = ((unsigned)(124 - 4 * r) << 23) + (rem >> 7);   // 2^(e-3-4r) (1+F)
        const unsigned sign = (c & 0x8000u) << 16;
        return __uint_as_float((c & 0x7FFFu) ? (bits | sign) : sign);
    }
    static __device__ __forceinline__ unsigned enc(float x) {
        const unsigned xb = __float_as_uint(x);
        const unsigned Xb = xb & 0x7FFFFFFFu;
        const int g = (int)(Xb >> 23) - 64;                 // E + 63
        const unsigned W = 0x80000000u | (((unsigned)g & 3u) << 29) | ((Xb & 0x007FFFFFu) << 6);
        const int r = 15 - (g >> 2);
        unsigned code = min((((W >> (r & 31)) >> 16) + 1u) >> 1, 0x7FFFu);
        const unsigned LO = 0x26000000u /* 2^-51 */, HI = 0x40000000u /* 2 */;
        if (Xb - LO >= HI - LO) {
            code = Xb >= HI ? 0x7FFFu
                            : (unsigned)(Xb >= 0x21800000u /* 2^-60 */) + (unsigned)(Xb >= 0x23880000u /* 1.0625*2^-56 */) +
                                  (unsigned)(Xb >= 0x24A00000u /* 1.25*2^-54 */) + (unsigned)(Xb >= 0x25A00000u /* 1.25*2^-52 */);
        }
        return ((xb >> 16) & 0x8000u) | code;
    }
};

// ---- codecs on pairs: two 16-bit codes in one 32-bit word (low half = the lower x) ----------------------
// Used by the shared-memory-staged kernel (lbm_bulk.cuh), which handles two neighbouring cells per thread.
//   SC        the decoded values are 2^SC times the DDFs and enc2 expects 2^SC times the DDFs: FP16S leaves its
//             2^15 scaling to the collision (collide_bgk<.., SC>), which folds it into operations it executes
//             anyway -- decode is one HADD2.F32, encode half an F2FP.PACK_AB per value;
//   dec1(c)   c = one code SIGN-EXTENDED to 32 bits (ld.shared.s16);
//   dec2(w)   both codes of a word;  enc2(a, b) packs the codes of a (low) and b (high).
//   TABLE     enc2 reads the format's 512-entry encoder table (EncEntry, below) from shared memory;
//   CHECK     codes with (code & CHECK) != 0 are outside the domain of dec1 / dec2: the caller ORs the raw words
//             together and, if a CHECK bit shows up, decodes again with PairCodec<F>::Full (all codes, dearer).
// Every function returns bit for bit what Codec<F>::dec / enc return (times 2^SC).
struct EncEntry {
    // code = base + hi32(min(bits(X) + add, tmax) * mult).  tmax is used by the formats that clamp (CLAMP below) and is
    // ZERO for the others: their code is the high word of ONE 64-bit multiply-add, t * mult + {tmax = 0 : base}, whose
    // addend is the entry's second register pair as loaded
    unsigned add, mult, tmax, base;
};

template <int F>
struct PairCodec {
    static constexpr int SC = 0;
    static constexpr bool TABLE = false;
    static constexpr unsigned CHECK = 0;
    static constexpr bool SEXT = false;         // dec1 wants its code sign-extended to 32 bits
    static constexpr bool FAST = false;         // enc2_fast exists (a table-free encoder for part of the range)
    static __device__ __forceinline__ float dec1(int c) { return Codec<F>::dec((unsigned)c & 0xFFFFu); }
    static __device__ __forceinline__ void dec2(unsigned w, float &a, float &b) {
        a = Codec<F>::dec(w & 0xFFFFu);
        b = Codec<F>::dec(w >> 16);
    }
    static __device__ __forceinline__ unsigned enc2(float a, float b, const EncEntry *) {
        return Codec<F>::enc(a) | (Codec<F>::enc(b) << 16);
    }
    static __device__ __forceinline__ unsigned enc1(float a, const EncEntry *) { return Codec<F>::enc(a); }   // one code
};

template <int SCALE>
struct PairHalf {
    static constexpr int SC = SCALE;
    static constexpr bool TABLE = false;
    static constexpr unsigned CHECK = 0;
    static constexpr bool SEXT = false;
    static constexpr bool FAST = false;         // enc2_fast exists (a table-free encoder for part of the range)
    static __device__ __forceinline__ float dec1(int c) { return __half2float(__ushort_as_half((unsigned short)c)); }
    static __device__ __forceinline__ void dec2(unsigned w, float &a, float &b) {
        const float2 v = __half22float2(*reinterpret_cast<const __half2 *>(&w));
        a = v.x;
        b = v.y;
    }
    static __device__ __forceinline__ unsigned enc2(float a, float b, const EncEntry *) {
        const __half2 h = __floats2half2_rn(a, b);          // one F2FP.F16.F32.PACK_AB, round-to-nearest-even
        return *reinterpret_cast<const unsigned *>(&h);
    }
    static __device__ __forceinline__ unsigned enc1(float a, const EncEntry *) { return __half_as_ushort(__float2half_rn(a)); }
};
template <>
struct PairCodec<F_FP16> : PairHalf<0> {};
template <>
struct PairCodec<F_FP16S> : PairHalf<15> {};

// FP16C: the sign-extended code shifted left by 12 has the sign in bits 31..27 and the magnitude in bits 26..12;
// one AND leaves sign | magnitude, the multiply by 2^112 does exponent re-bias and denormals (Codec<F_FP16C>).
// Encode: clamp |x| to the largest value (NaN -> largest, as Codec does), fmul.rz by 2^-112, add half an ulp;
// the magnitude code then sits in bits 26..12: shifted left by 4 it is the upper half-word, and one PRMT packs
// two of them; a second PRMT gathers the two sign bytes.
template <>
struct PairCodec<F_FP16C> {
    static constexpr int SC = 0;
    static constexpr bool TABLE = false;
    static constexpr unsigned CHECK = 0;
    static constexpr bool SEXT = true;
    static constexpr bool FAST = false;         // enc2_fast exists (a table-free encoder for part of the range)
    static __device__ __forceinline__ float bits2f(unsigned t) {
        return __fmul_rn(__uint_as_float(t & 0x87FFF000u), __uint_as_float(0x77800000u));   // * 2^112, exact
    }
    static __device__ __forceinline__ float dec1(int c) { return bits2f((unsigned)c << 12); }
    static __device__ __forceinline__ void dec2(unsigned w, float &a, float &b) {
        a = bits2f((unsigned)((int)(w << 16) >> 4));
        b = bits2f((unsigned)((int)w >> 4));
    }
    static __device__ __forceinline__ unsigned mag4(float x) {      // magnitude code in bits 30..16
        const float y = __fmul_rz(fminf(fabsf(x), __uint_as_float(0x3FFFF000u) /* 2 - 2^-11 */), __uint_as_float(0x07800000u));
        return (__float_as_uint(y) + 0x800u) << 4;
    }
    static __device__ __forceinline__ unsigned enc2(float a, float b, const EncEntry *) {
        const unsigned mags = __byte_perm(mag4(a), mag4(b), 0x7632);
        const unsigned signs = __byte_perm(__float_as_uint(a), __float_as_uint(b), 0x7632);
        return (mags & 0x7FFF7FFFu) | (signs & 0x80008000u);
    }
    static __device__ __forceinline__ unsigned enc1(float a, const EncEntry *t) { return enc2(a, a, t) & 0xFFFFu; }
};

// ---- posits on pairs ------------------------------------------------------------------------------------
// Encode, all three posits: the code of X = +-2^E (1 + M 2^-23) is, inside one binade, base(E) plus the rounded
// leading fraction bits of M -- and where the regime leaves no fraction bits, base(E) plus one step at one
// threshold.  Both are  base + ((M + add) >> sh)  with per-binade constants (carries run from the fraction into
// exponent and regime because posit codes are monotone; the paper's converters use the same
// fact).  The 512 (sign, exponent) entries are derived ON THE DEVICE from Codec<F>::enc
// (enc_table_kernel, lbm_aux.cu) and then checked against it on all 2^32 inputs (lbm_codec_pair_selftest).
// One table read, one add and one multiply-high replace the regime arithmetic; sign, scaling (2^7 for P16_0S /
// P16_1S), saturation and the nearest-value corners of DESIGN.md R14 are all inside the table.
// CLAMP: the top binade of an unscaled format ends in the saturating code (P16_2C: [1, 2) -> 0x7000..0x7FFF): the
// entry's fourth word bounds (M + add) so that values within half a step of 2 stay at 0x7FFF.
template <bool CLAMP>
__device__ __forceinline__ unsigned enc_by_table(float X, const EncEntry *tab) {
    const unsigned xb = __float_as_uint(X);
    const uint4 e = *reinterpret_cast<const uint4 *>(tab + (xb >> 23));
    const unsigned t = xb + e.x;
    if (CLAMP) return __umulhi(min(t, e.z), e.y) + e.w;
    const unsigned long long acc = (unsigned long long)e.z | ((unsigned long long)e.w << 32);      // e.z == 0
    return (unsigned)(((unsigned long long)t * e.y + acc) >> 32);
}

// Decode for a regime of ZEROS (value below 1 before scaling; P16_2C has no other kind).  The 15 magnitude bits
// "0..01 e F" read as an integer n are 2^(14-k) (1 + [e F]): normalising n (one multiply of the FP32 denormal
// n 2^-141 by 2^127) yields exponent field 127-k and the bits [e F] left-aligned in the mantissa, which is the
// posit's value up to a fixed affine map of the FP32 word:
//   es = 0   value = n 2^-14 exactly -- posits with es = 0 are linear below 1;
//   es = 1   word = 2 b - 0x43000000        (exponent field 120 - 2k + e, scale 2^-7 included);
//   es = 2   word = 4 b + 0x40000000        (exponent field 124 - 4r + e; mod 2^32);
// max(b, .) maps the zero code to zero.  A regime of ONES (bit 14 set, |f| >= 2^-7) is not handled here: CHECK.
// Full-range posit decoders (both regime signs), used where the zero-regime decoders above do not apply.
// Sign-extending the 15 magnitude bits from bit 14 gives t = n for a regime of zeros and t = -(2^15 - n) for a regime
// of ones; |t| normalised (int -> float) has the regime length in its exponent and, for ones, the COMPLEMENT of the
// payload [e F] in its mantissa: 2^15 - n = 2^(L+1) - P for a payload P of L bits, so its float is 2^L (2 - P/2^L) and
// subtracting the word from a constant both negates the exponent and turns 1 - P/2^L back into P/2^L.  Hence
//   regime of zeros: word = MUL * b - KZ,      regime of ones: word = KO - MUL * b     (mod 2^32, b = float word of t)
// with MUL = 2^es moving the exponent bit(s) from the mantissa top into the exponent field.
template <int MUL, unsigned KZ, unsigned KO, unsigned FLOOR>
struct PositFull {
    static __device__ __forceinline__ float word(int t, unsigned sign) {        // t = magnitude sign-extended from bit 14
        const unsigned b = __float_as_uint(__int2float_rn(t));
        const unsigned wz = max(b, FLOOR) * (unsigned)MUL - KZ;                 // FLOOR: the zero code gives zero
        const unsigned wo = KO - b * (unsigned)MUL;
        return __uint_as_float(((t < 0 ? wo : wz) & 0x7FFFFFFFu) | (sign & 0x80000000u));
    }
    static __device__ __forceinline__ float dec1(int c) { return word((c << 17) >> 17, (unsigned)c << 16); }
    static __device__ __forceinline__ void dec2(unsigned w, float &a, float &b) {
        a = word((int)(w << 17) >> 17, w << 16);
        b = word((int)(w << 1) >> 17, w);
    }
};

template <>
struct PairCodec<F_P16_0S> {
    static constexpr int SC = -1;           // decoded = n 2^-22 = f / 2: one multiply, the factor 2 rides on SC
    static constexpr bool TABLE = true;
    static constexpr unsigned CHECK = 0x4000u;
    static constexpr bool SEXT = true;
    static constexpr bool FAST = true;
    typedef PositFull<1, 0x0B000000u, 0x02000000u, 0x0B000000u> Full;           // same scaling: f / 2
    static __device__ __forceinline__ float sm2f(unsigned t) {      // t = sign-extended code
        return __fmul_rn(__uint_as_float(t & 0x80007FFFu), __uint_as_float(0x7F000000u));   // * 2^127, exact
    }
    static __device__ __forceinline__ float dec1(int c) { return sm2f((unsigned)c); }
    static __device__ __forceinline__ void dec2(unsigned w, float &a, float &b) {
        a = sm2f(__byte_perm(w, 0, 0x9910));                        // sign-extend the low half-word
        b = sm2f((unsigned)((int)w >> 16));
    }
    static __device__ __forceinline__ unsigned enc2(float a, float b, const EncEntry *tab) {
        return __byte_perm(enc_by_table<false>(a, tab), enc_by_table<false>(b, tab), 0x5410);
    }
    static __device__ __forceinline__ unsigned enc1(float a, const EncEntry *tab) { return enc_by_table<false>(a, tab) & 0xFFFFu; }
    // The table-free encoder for a regime of zeros.  Below 1 a posit with es = 0 is FIXED POINT -- the magnitude code n is
    // the value 2^7 |f| in units of 2^-14 (the decoder above uses the same fact) -- so rule U (nearest value, ties to the
    // larger magnitude, R14) is n = floor(2^21 |f| + 1/2) = floor(2^22 |X| + 1/2) for X = f / 2 (SC = -1).  Two FP32
    // operations rounded TOWARDS ZERO compute it exactly: s = fma.rz(|X|, 2^22, 1/2) is the largest float <= the true sum,
    // so it never crosses an integer downwards (integers below 2^24 are floats); fadd.rz(s, 2^23) leaves floor(s) in the
    // mantissa.  (Round-to-nearest would fail: 2^22 |X| = 1/2 - 2^-25 gives 1 - 2^-25, a tie that rounds up to 1.)
    // No shared-memory table read, no integer pipe.  `acc` collects every bit above bit 13 of the results: if any is set
    // -- |2^7 f| >= 1, a regime of ones, or a NaN -- the caller encodes again with enc2 (the table).  Checked against
    // Codec<F_P16_0S>::enc on all 2^32 inputs by lbm_codec_pair_selftest.
    static __device__ __forceinline__ unsigned enc2_fast(float a, float b, unsigned &acc) {
        const float sa = __fmaf_rz(fabsf(a), 4194304.0f, 0.5f), sb = __fmaf_rz(fabsf(b), 4194304.0f, 0.5f);
        const unsigned ta = __float_as_uint(__fadd_rz(sa, 8388608.0f)) ^ 0x4B000000u;       // = n while n < 2^23
        const unsigned tb = __float_as_uint(__fadd_rz(sb, 8388608.0f)) ^ 0x4B000000u;
        acc |= ta | tb;
        const unsigned signs = __byte_perm(__float_as_uint(a), __float_as_uint(b), 0x7632);
        return __byte_perm(ta, tb, 0x5410) | (signs & 0x80008000u);
    }
    static __device__ __forceinline__ unsigned enc1_fast(float a, unsigned &acc) {          // one code (in the low 16 bits)
        const unsigned ta = __float_as_uint(__fadd_rz(__fmaf_rz(fabsf(a), 4194304.0f, 0.5f), 8388608.0f)) ^ 0x4B000000u;
        acc |= ta;
        return ta | ((__float_as_uint(a) >> 16) & 0x8000u);
    }
    static constexpr unsigned FAST_BAD = 0xFFFFC000u;       // acc & FAST_BAD != 0: outside enc2_fast's domain
};

template <int MUL, unsigned OFF, unsigned FLOOR, unsigned CHK>
struct PairPositLow {
    static constexpr int SC = 0;
    static constexpr bool TABLE = true;
    static constexpr unsigned CHECK = CHK;
    static constexpr bool SEXT = false;
    static constexpr bool FAST = false;         // enc2_fast exists (a table-free encoder for part of the range)
    // t = the code shifted so that the magnitude sits in bits 22..8 and the sign in bit 31
    static __device__ __forceinline__ float word(unsigned t) {
        const unsigned b = __float_as_uint(__fmul_rn(__uint_as_float(t & 0x007FFF00u), __uint_as_float(0x7F000000u)));
        const unsigned v = max(b, FLOOR) * (unsigned)MUL + OFF;
        return __uint_as_float(v | (t & 0x80000000u));
    }
    // one PRMT builds t from a code: bytes [0, low, high, high] -- magnitude in bits 22..8, the sign (top bit of the high
    // byte) in bit 31; word() masks the rest
    static __device__ __forceinline__ float dec1(int c) { return word(__byte_perm((unsigned)c, 0, 0x1104)); }
    static __device__ __forceinline__ void dec2(unsigned w, float &a, float &b) {
        a = word(__byte_perm(w, 0, 0x1104));
        b = word(__byte_perm(w, 0, 0x3324));
    }
    static __device__ __forceinline__ unsigned enc2(float a, float b, const EncEntry *tab) {
        return __byte_perm(enc_by_table<CHK == 0>(a, tab), enc_by_table<CHK == 0>(b, tab), 0x5410);
    }
    static __device__ __forceinline__ unsigned enc1(float a, const EncEntry *tab) { return enc_by_table<CHK == 0>(a, tab) & 0xFFFFu; }
};
template <>
struct PairCodec<F_P16_1S> : PairPositLow<2, 0xBD000000u /* -0x43000000 */, 0x21800000u, 0x4000u> {
    typedef PositFull<2, 0x51000000u, 0xC9000000u, 0x28800000u> Full;
};
template <>
struct PairCodec<F_P16_2C> : PairPositLow<4, 0x40000000u, 0x30000000u, 0u> {};

}  // namespace lbmk
