// lbm_aux.cu -- small kernels beside the hot path: the FLAG_NEAR pass of lbm_set_flags and the
// stand-alone codec kernels behind lbm_codec_encode / lbm_codec_decode (bit-level parity tests).
#include <atomic>
#include <cstdio>
#include <mutex>

#include "lbm_internal.h"
#include "lbm_kernels.cuh"
#include "lbm_bulk.cuh"

namespace lbmk {

static std::atomic<long long> g_launches{0};
void count_launch(long long n) { g_launches += n; }
long long launches() { return g_launches.load(); }

// out[n] = in[n] | FLAG_NEAR if cell n is fluid and at least one of its q-1 pull sources (x - c_i,
// periodic, R2) is a wall cell.  stream_collide then reads ONE flag byte per cell instead of the q
// the paper's kernel gathers.
template <int Q>
__global__ void __launch_bounds__(256) mark_near_kernel(const unsigned char *__restrict__ in, unsigned char *__restrict__ out,
                                                        unsigned *__restrict__ bounce, int nx, int ny, int nz) {
    typedef Lat<Q> L;
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y, z = blockIdx.z;
    if (x >= nx) return;
    const long long n = x + (long long)nx * (y + (long long)ny * z);
    unsigned fl = in[n] & (FLAG_FIXED | FLAG_OUT);          // (an outflow cell pulls nothing: no FLAG_NEAR for it)
    unsigned mask = 0;                                       // bit i: the pull source of direction i is a wall cell
    if (!fl) {
        unsigned near = 0;
#pragma unroll
        for (int i = 1; i < Q; ++i) {
            int xs = x - L::c(i, 0), ys = y - L::c(i, 1), zs = z - L::c(i, 2);
            xs = xs < 0 ? nx - 1 : xs >= nx ? 0 : xs;
            ys = ys < 0 ? ny - 1 : ys >= ny ? 0 : ys;
            zs = zs < 0 ? nz - 1 : zs >= nz ? 0 : zs;
            const unsigned wsrc = in[xs + (long long)nx * (ys + (long long)ny * zs)] & FLAG_WALL;
            near |= wsrc;
            mask |= wsrc << i;
        }
        if (near) fl |= FLAG_NEAR;
    }
    out[n] = (unsigned char)fl;
    bounce[n] = mask;
}

cudaError_t launch_mark_near(int q, const unsigned char *in, unsigned char *out, unsigned *bounce, int nx, int ny, int nz,
                             cudaStream_t st) {
    const dim3 block(256), grid((nx + 255) / 256, ny, nz);
    if (q == 9) mark_near_kernel<9><<<grid, block, 0, st>>>(in, out, bounce, nx, ny, nz);
    else if (q == 19) mark_near_kernel<19><<<grid, block, 0, st>>>(in, out, bounce, nx, ny, nz);
    else if (q == 27) mark_near_kernel<27><<<grid, block, 0, st>>>(in, out, bounce, nx, ny, nz);
    else return cudaErrorInvalidValue;
    count_launch();
    return cudaGetLastError();
}

// bounce[n] bit 31 := one of the wall cells this cell bounces on has a non-zero velocity (R9); run by lbm_init,
// when the wall velocities are known.  Cells whose walls all rest never load a wall velocity in the time step.
template <int Q>
__global__ void __launch_bounds__(256) mark_moving_kernel(unsigned *__restrict__ bounce, const float *__restrict__ u0, int nx, int ny,
                                                          int nz) {
    typedef Lat<Q> L;
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y, z = blockIdx.z;
    if (x >= nx) return;
    const long long N = (long long)nx * ny * nz, n = x + (long long)nx * (y + (long long)ny * z);
    unsigned m = bounce[n] & 0x7FFFFFFFu;
    if (m == 0) return;
    bool moving = false;
#pragma unroll
    for (int i = 1; i < Q; ++i) {
        if (!((m >> i) & 1u)) continue;
        int xs = x - L::c(i, 0), ys = y - L::c(i, 1), zs = z - L::c(i, 2);
        xs = xs < 0 ? nx - 1 : xs >= nx ? 0 : xs;
        ys = ys < 0 ? ny - 1 : ys >= ny ? 0 : ys;
        zs = zs < 0 ? nz - 1 : zs >= nz ? 0 : zs;
        const long long src = xs + (long long)nx * (ys + (long long)ny * zs);
        moving |= u0[src] != 0.0f || u0[N + src] != 0.0f || u0[2 * N + src] != 0.0f;
    }
    bounce[n] = m | (moving ? 0x80000000u : 0u);
}

cudaError_t launch_mark_moving(int q, unsigned *bounce, const float *u0, int nx, int ny, int nz, cudaStream_t st) {
    const dim3 block(256), grid((nx + 255) / 256, ny, nz);
    if (q == 9) mark_moving_kernel<9><<<grid, block, 0, st>>>(bounce, u0, nx, ny, nz);
    else if (q == 19) mark_moving_kernel<19><<<grid, block, 0, st>>>(bounce, u0, nx, ny, nz);
    else if (q == 27) mark_moving_kernel<27><<<grid, block, 0, st>>>(bounce, u0, nx, ny, nz);
    else return cudaErrorInvalidValue;
    count_launch();
    return cudaGetLastError();
}

// ---- per-tile lists of flagged cells (built at the first step after lbm_set_flags / lbm_init, for the staged kernel's
// tile geometry; lbm_stage.cuh) ---------------------------------------------------------------------------
// counts[t] = number of cells of tile t with a flag bit set (wall, equilibrium boundary, next to a wall)
__global__ void __launch_bounds__(128) fix_count_kernel(const Params p, const BulkGeom g, unsigned *__restrict__ counts) {
    __shared__ unsigned total;
    for (int t = blockIdx.x; t < g.n_tiles; t += gridDim.x) {
        if (threadIdx.x == 0) total = 0;
        __syncthreads();
        const TileCoord c = tile_coord(t, g, p);
        const int cells = c.rows * c.w;
        const long long first = (long long)p.nx * (c.y + (long long)p.ny * c.z) + c.x0;
        unsigned n = 0;
        for (int ci = threadIdx.x; ci < cells; ci += blockDim.x) n += p.flags[first + ci] != 0;
        if (n) atomicAdd(&total, n);
        __syncthreads();
        if (threadIdx.x == 0) counts[t] = total;
        __syncthreads();
    }
}

// off[0..n] = exclusive prefix sums of counts[0..n-1]; one CTA
__global__ void __launch_bounds__(1024) fix_scan_kernel(const unsigned *__restrict__ counts, unsigned *__restrict__ off, int n) {
    __shared__ unsigned wsum[32];
    __shared__ unsigned carry;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    if (tid == 0) carry = 0;
    __syncthreads();
    for (int base = 0; base < n; base += 1024) {
        const int i = base + tid;
        const unsigned v = i < n ? counts[i] : 0u;
        unsigned s = v;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const unsigned o = __shfl_up_sync(0xffffffffu, s, d);
            if (lane >= d) s += o;
        }
        if (lane == 31) wsum[wid] = s;
        __syncthreads();
        if (wid == 0) {
            unsigned ws = wsum[lane];
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const unsigned o = __shfl_up_sync(0xffffffffu, ws, d);
                if (lane >= d) ws += o;
            }
            wsum[lane] = ws;                                                // inclusive over the warps
        }
        __syncthreads();
        const unsigned before = carry + (wid ? wsum[wid - 1] : 0u) + s - v;
        if (i < n) off[i] = before;
        __syncthreads();
        if (tid == 1023) carry = before + v;
        __syncthreads();
    }
    if (tid == 0) off[n] = carry;
}

__global__ void __launch_bounds__(128) fix_fill_kernel(const Params p, const BulkGeom g, const unsigned *__restrict__ off,
                                                      uint2 *__restrict__ list) {
    __shared__ unsigned cursor;
    for (int t = blockIdx.x; t < g.n_tiles; t += gridDim.x) {
        if (threadIdx.x == 0) cursor = 0;
        __syncthreads();
        const unsigned lo = off[t];
        if (off[t + 1] != lo) {
            const TileCoord c = tile_coord(t, g, p);
            const int cells = c.rows * c.w;
            const long long first = (long long)p.nx * (c.y + (long long)p.ny * c.z) + c.x0;
            for (int ci = threadIdx.x; ci < cells; ci += blockDim.x) {
                const unsigned fl = p.flags[first + ci];
                if (fl != 0) list[lo + atomicAdd(&cursor, 1u)] = make_uint2((unsigned)ci | (fl << 16), p.bounce ? p.bounce[first + ci] : 0u);
            }
        }
        __syncthreads();
    }
}

// Per-tile lists of flagged cells for the staged kernel's tile geometry g (Params::fix_off / fix_cells); p.flags
// must hold the final flag bytes (FLAG_NEAR set).  The caller owns (cudaFree) both arrays.  Synchronises the stream.
cudaError_t build_fix_lists_for(const Params &p, const BulkGeom &g, unsigned **off_out, uint2 **list_out, cudaStream_t st) {
    *off_out = nullptr;
    *list_out = nullptr;
    unsigned *counts = nullptr, *off = nullptr;
    uint2 *list = nullptr;
    cudaError_t e = cudaMalloc((void **)&counts, (size_t)g.n_tiles * 4);
    if (e == cudaSuccess) e = cudaMalloc((void **)&off, ((size_t)g.n_tiles + 1) * 4);
    const int grid = g.n_tiles < 148 * 32 ? g.n_tiles : 148 * 32;
    unsigned total = 0;
    if (e == cudaSuccess) {
        fix_count_kernel<<<grid, 128, 0, st>>>(p, g, counts);
        fix_scan_kernel<<<1, 1024, 0, st>>>(counts, off, g.n_tiles);
        count_launch(2);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpyAsync(&total, off + g.n_tiles, 4, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e == cudaSuccess) e = cudaMalloc((void **)&list, (size_t)(total ? total : 1) * sizeof(uint2));
    if (e == cudaSuccess) {
        fix_fill_kernel<<<grid, 128, 0, st>>>(p, g, off, list);
        count_launch();
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (counts) cudaFree(counts);
    if (e != cudaSuccess) {
        (void)cudaGetLastError();
        if (off) cudaFree(off);
        if (list) cudaFree(list);
        return e;
    }
    *off_out = off;
    *list_out = list;
    return cudaSuccess;
}

template <int F>
__global__ void __launch_bounds__(256) encode_kernel(const float *__restrict__ x, unsigned short *__restrict__ c, long long n) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        c[i] = (unsigned short)Codec<F>::enc(x[i]);
}
template <int F>
__global__ void __launch_bounds__(256) decode_kernel(const unsigned short *__restrict__ c, float *__restrict__ x, long long n) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        x[i] = Codec<F>::dec((unsigned)c[i]);
}

template <int F>
static cudaError_t codec_launch(bool encode, const void *in, void *out, long long n, cudaStream_t st) {
    long long b = (n + 255) / 256;
    if (b > 148LL * 32) b = 148LL * 32;
    if (b < 1) b = 1;
    if (encode) encode_kernel<F><<<(int)b, 256, 0, st>>>((const float *)in, (unsigned short *)out, n);
    else decode_kernel<F><<<(int)b, 256, 0, st>>>((const unsigned short *)in, (float *)out, n);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_codec(int fmt, bool encode, const void *in, void *out, long long count, cudaStream_t st) {
    switch (fmt) {
        case F_FP16S: return codec_launch<F_FP16S>(encode, in, out, count, st);
        case F_FP16C: return codec_launch<F_FP16C>(encode, in, out, count, st);
        case F_P16_0S: return codec_launch<F_P16_0S>(encode, in, out, count, st);
        case F_P16_1S: return codec_launch<F_P16_1S>(encode, in, out, count, st);
        case F_P16_2C: return codec_launch<F_P16_2C>(encode, in, out, count, st);
        case F_FP16: return codec_launch<F_FP16>(encode, in, out, count, st);
    }
    return cudaErrorInvalidValue;
}

// ---- encoder tables of the table-driven pair codecs (lbm_codecs.cuh, "posits on pairs") -----------------
// One entry per (sign, FP32 exponent) of the encoder's input X = 2^SC x, derived from Codec<F>::enc itself:
//   c0, c1 = codes of the first and last value of the binade; d = c1 - c0
//   d = 0        constant code                                      -> mult = 1 (hi32 = 0)
//   d = 1        one threshold, found by bisection (enc is monotone) -> (M + 2^23 - thr) >> 23
//   d = 2^nf     nf fraction bits, round half up                     -> (M + 2^(22-nf)) >> (23-nf)
//   d = 2^nf - 1 and c1 saturated (0x7FFF): same, with M + add bounded so the top half step stays at 0x7FFF
// anything else would make the entry unusable: mult = 0 marks it and lbm_codec_pair_selftest reports it.
__device__ EncEntry g_enc_tables[7][512];

template <int F>
__global__ void __launch_bounds__(512) enc_table_kernel(EncEntry *tab) {
    const unsigned idx = threadIdx.x;
    const float dn = pow2f(-PairCodec<F>::SC);
    auto probe = [&](unsigned M) { return Codec<F>::enc(__fmul_rn(__uint_as_float((idx << 23) | M), dn)); };
    // exponent 255: M = 0 is infinity (saturates), M != 0 a NaN, whose code is not pinned: the binade gets infinity's code
    const unsigned c0 = probe(0), c1 = (idx & 255u) == 255u ? c0 : probe(0x7FFFFFu), d = c1 - c0;
    EncEntry e;
    e.base = c0;
    constexpr bool CLAMPS = PairCodec<F>::TABLE && PairCodec<F>::CHECK == 0;      // (P16_2C; see enc_by_table)
    e.tmax = CLAMPS ? 0xFFFFFFFFu : 0u;
    unsigned add = 0;
    if (d == 0) {
        e.mult = 1u;
    } else if (d == 1) {
        unsigned lo = 0, hi = 0x7FFFFFu;                    // probe(lo) = c0, probe(hi) = c1
        while (hi - lo > 1) {
            const unsigned mid = (lo + hi) >> 1;
            if (probe(mid) == c0) lo = mid; else hi = mid;
        }
        add = (1u << 23) - hi;
        e.mult = 1u << 9;
    } else if ((d & (d - 1)) == 0 || (((d + 1) & d) == 0 && (c1 & 0x7FFFu) == 0x7FFFu)) {
        const bool sat = (d & (d - 1)) != 0;
        const int nf = 31 - __clz((int)(sat ? d + 1 : d)), sh = 23 - nf;
        add = 1u << (sh - 1);
        e.mult = 1u << (32 - sh);
        if (sat && CLAMPS) e.tmax = (d << sh) | ((1u << sh) - 1u);
    } else {
        e.mult = 0u;
#ifdef LBM_SELFTEST_DEBUG
        printf("enc_table F=%d idx=%u c0=%04x c1=%04x\n", F, idx, c0, c1);
#endif
    }
    e.add = add - (idx << 23);
    tab[idx] = e;
}

// The table of a format is built once per device, synchronously and under a lock: it is complete, and known to be, before
// any caller on any stream gets its address (a flag set after an asynchronous launch would let a second handle on
// another stream read a half-written table).  A failed build leaves the flag clear.
cudaError_t enc_table(int fmt, const EncEntry **out, cudaStream_t st) {
    static std::mutex mu;
    static bool built[64][7];
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64 || fmt < 0 || fmt > 6) return cudaErrorInvalidValue;
    EncEntry *base = nullptr;
    if ((e = cudaGetSymbolAddress((void **)&base, g_enc_tables)) != cudaSuccess) return e;
    EncEntry *tab = base + fmt * 512;
    *out = tab;
    if (fmt != F_P16_0S && fmt != F_P16_1S && fmt != F_P16_2C) return cudaSuccess;      // formats without a table
    std::lock_guard<std::mutex> lock(mu);
    if (built[dev][fmt]) return cudaSuccess;
    // cudaStreamSynchronize is not allowed while `st` is being captured into a graph: build on the legacy stream
    (void)st;
    switch (fmt) {
        case F_P16_0S: enc_table_kernel<F_P16_0S><<<1, 512>>>(tab); break;
        case F_P16_1S: enc_table_kernel<F_P16_1S><<<1, 512>>>(tab); break;
        default: enc_table_kernel<F_P16_2C><<<1, 512>>>(tab); break;
    }
    count_launch();
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    if ((e = cudaDeviceSynchronize()) != cudaSuccess) return e;
    built[dev][fmt] = true;
    return cudaSuccess;
}

// ---- pair codecs vs scalar codecs, exhaustively, on the device ----------------------------------------
// PairCodec<F> (the staged kernel's converters) must return bit for bit what Codec<F> returns (times 2^SC):
// all 65 536 codes through dec1 / dec2 (both halves) and ALL 2^32 FP32 bit patterns through enc2 (both halves).
// Codec<F> itself is compared with the oracle by the tests; this closes the chain for PairCodec<F>.
template <int F>
__global__ void __launch_bounds__(256) pair_selftest_kernel(unsigned long long *mismatches, const EncEntry *tab) {
    typedef PairCodec<F> PC;
    const float up = pow2f(PC::SC);
    unsigned long long bad = 0;
    if (PC::TABLE)
        for (int i = 0; i < 512; ++i) bad += tab[i].mult == 0;                 // an entry the table kernel could not express
    const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
    for (unsigned long long v = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; v < (1ull << 32); v += stride) {
        const unsigned b = (unsigned)v;
        const float x = __uint_as_float(b);
        const float other = __uint_as_float(b * 2654435761u + 12345u);          // an unrelated partner value
        const unsigned ref = Codec<F>::enc(x), ref_o = Codec<F>::enc(other);
        const unsigned w1 = PC::enc2(__fmul_rn(x, up), __fmul_rn(other, up), tab);
        const unsigned w2 = PC::enc2(__fmul_rn(other, up), __fmul_rn(x, up), tab);
        const bool nan = x != x || other != other;                              // NaN payloads of binary16 are not pinned
        if (!nan) bad += (w1 != (ref | (ref_o << 16))) + (w2 != (ref_o | (ref << 16)));
        if constexpr (PC::FAST) {                                               // the table-free encoder, wherever it claims to be valid
            unsigned acc = 0;
            const unsigned w3 = PC::enc2_fast(__fmul_rn(x, up), __fmul_rn(other, up), acc);
            if (!nan && !(acc & PC::FAST_BAD)) bad += w3 != (ref | (ref_o << 16));
            acc = 0;
            const unsigned w5 = PC::enc1_fast(__fmul_rn(x, up), acc) & 0xFFFFu;                 // the one-code form
            if (!nan && !(acc & PC::FAST_BAD)) bad += w5 != ref;
            acc = 0;
            const unsigned w4 = PC::enc2_fast(__fmul_rn(x, up), __fmul_rn(x, up), acc);
            // (and it must claim validity on the whole regime of zeros: |2^7 x| < 1)
            if (!nan && (b & 0x7FFFFFFFu) < 0x3BFFF000u /* just below 2^-7 */) bad += (acc & PC::FAST_BAD) != 0 || w4 != (ref | (ref << 16));
        }
#ifdef LBM_SELFTEST_DEBUG
        if (!nan && (w1 & 0xFFFFu) != ref && (b % 977u) == 0) printf("enc x=%08x ref=%04x got=%04x\n", b, ref, w1 & 0xFFFFu);
#endif
        if (v < 65536) {
            unsigned c = (unsigned)v, c2 = (c * 40503u + 7u) & 0xFFFFu;
            if constexpr (PC::CHECK != 0) {                                     // the full-range decoders: every code
                typedef typename PC::Full FD;
                const float r = __fmul_rn(Codec<F>::dec(c), up), r2 = __fmul_rn(Codec<F>::dec(c2), up);
                float a, d;
                FD::dec2(c | (c2 << 16), a, d);
                const float e = FD::dec1(PC::SEXT ? (int)(short)c : (int)c);
                bad += (__float_as_uint(a) != __float_as_uint(r)) + (__float_as_uint(d) != __float_as_uint(r2)) +
                       (__float_as_uint(e) != __float_as_uint(r));
            }
            if (PC::CHECK) { c2 &= ~PC::CHECK; if (c & PC::CHECK) continue; }  // outside the fast decoders' domain: the kernel falls back
            const float r = __fmul_rn(Codec<F>::dec(c), up), r2 = __fmul_rn(Codec<F>::dec(c2), up);
            float a, d;
            PC::dec2(c | (c2 << 16), a, d);
            const float e = PC::dec1(PC::SEXT ? (int)(short)c : (int)c);
            const bool cn = r != r || r2 != r2;
#ifdef LBM_SELFTEST_DEBUG
            if (!cn && __float_as_uint(a) != __float_as_uint(r)) printf("dec2lo c=%04x ref=%08x got=%08x\n", c, __float_as_uint(r), __float_as_uint(a));
            if (!cn && __float_as_uint(e) != __float_as_uint(r)) printf("dec1 c=%04x ref=%08x got=%08x\n", c, __float_as_uint(r), __float_as_uint(e));
            if (!cn && __float_as_uint(d) != __float_as_uint(r2)) printf("dec2hi c=%04x ref=%08x got=%08x\n", c2, __float_as_uint(r2), __float_as_uint(d));
#endif
            if (cn) bad += !(a != a || !(r != r)) + !(d != d || !(r2 != r2)) + !(e != e || !(r != r));
            else bad += (__float_as_uint(a) != __float_as_uint(r)) + (__float_as_uint(d) != __float_as_uint(r2)) +
                        (__float_as_uint(e) != __float_as_uint(r));
        }
    }
    if (bad) atomicAdd(mismatches, bad);
}

cudaError_t launch_pair_selftest(int fmt, unsigned long long *mismatches_dev, cudaStream_t st) {
    const int blocks = 148 * 16;
    const EncEntry *tab = nullptr;
    cudaError_t e = enc_table(fmt, &tab, st);
    if (e != cudaSuccess) return e;
    switch (fmt) {
        case F_FP16S: pair_selftest_kernel<F_FP16S><<<blocks, 256, 0, st>>>(mismatches_dev, tab); break;
        case F_FP16C: pair_selftest_kernel<F_FP16C><<<blocks, 256, 0, st>>>(mismatches_dev, tab); break;
        case F_P16_0S: pair_selftest_kernel<F_P16_0S><<<blocks, 256, 0, st>>>(mismatches_dev, tab); break;
        case F_P16_1S: pair_selftest_kernel<F_P16_1S><<<blocks, 256, 0, st>>>(mismatches_dev, tab); break;
        case F_P16_2C: pair_selftest_kernel<F_P16_2C><<<blocks, 256, 0, st>>>(mismatches_dev, tab); break;
        case F_FP16: pair_selftest_kernel<F_FP16><<<blocks, 256, 0, st>>>(mismatches_dev, tab); break;
        default: return cudaErrorInvalidValue;
    }
    count_launch();
    return cudaGetLastError();
}


// ---- div3 (lbm_lattice.cuh) vs the compiler's IEEE division, on the device --------------------------------------
// Denominators: every 2^7-th float in [2^-2, 2^2) and one pseudo-random float per index from all of [2^-60, 2^60];
// numerators per denominator: +-0, pseudo-random multiples of the 16-bit formats' smallest steps (2^-39, 2^-25, 2^-21,
// 2^-35, 2^-59), products k * b (exact quotients) and their FP32 neighbours, and pseudo-random floats of every
// magnitude the guard's contract admits.  Every result must equal __fdiv_rn's bit for bit.
__device__ __forceinline__ unsigned mix32(unsigned x) {
    x ^= x >> 16; x *= 0x7FEB352Du; x ^= x >> 15; x *= 0x846CA68Bu; x ^= x >> 16;
    return x;
}
__global__ void __launch_bounds__(256) div_selftest_kernel(unsigned long long *mismatches) {
    const unsigned gid = blockIdx.x * blockDim.x + threadIdx.x, n_threads = gridDim.x * blockDim.x;
    unsigned long long bad = 0;
    for (unsigned bi = gid; bi < (1u << 19); bi += n_threads) {
        float bs[2];
        bs[0] = __uint_as_float(0x3E800000u + (bi << 7));                               // [2^-2, 2^2)
        bs[1] = __uint_as_float(0x21800000u + mix32(bi * 2654435761u + 17u) % (0x5D800000u - 0x21800000u));
        for (int w = 0; w < 2; ++w) {
            const float b = bs[w];
            for (unsigned k = 0; k < 96; k += 3) {
                float a[3], q[3];
                for (unsigned m = 0; m < 3; ++m) {
                    const unsigned h = mix32((bi * 96u + k + m) * 0x9E3779B9u + (unsigned)w);
                    const unsigned kind = (k + m) % 8u, sel = (h >> 20) % 5u;
                    float v;
                    if (kind == 0) v = 0.0f;
                    else if (kind == 1) v = ldexpf((float)(h & 0xFFFFFu), -39);          // the FP16S grid
                    else if (kind == 2) v = ldexpf((float)(h & 0xFFFFu), sel == 0 ? -25 : sel == 1 ? -21 : sel == 2 ? -35 : -59);
                    else if (kind == 3) v = __fmul_rn(b, (float)(int)(h & 0xFFFu));     // exact quotients (where the product is exact)
                    else if (kind == 4) v = __uint_as_float(__float_as_uint(__fmul_rn(b, (float)(int)(1u + (h & 0xFFu)))) + (h >> 30));
                    else v = __uint_as_float(0x13000000u + h % (0x5D800000u - 0x13000000u));  // 2^-89 .. 2^60
                    a[m] = (h & 0x80000u) ? -v : v;
                }
                div3<1>(a, b, q, true);
                for (int m = 0; m < 3; ++m) bad += __float_as_uint(q[m]) != __float_as_uint(__fdiv_rn(a[m], b));
            }
        }
    }
    if (bad) atomicAdd(mismatches, bad);
}

cudaError_t launch_div_selftest(unsigned long long *mismatches_dev, cudaStream_t st) {
    div_selftest_kernel<<<148 * 8, 256, 0, st>>>(mismatches_dev);
    count_launch();
    return cudaGetLastError();
}

}  // namespace lbmk
