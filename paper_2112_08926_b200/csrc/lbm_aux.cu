// lbm_aux.cu -- small kernels beside the hot path: the FLAG_NEAR pass of lbm_set_flags and the
// stand-alone codec kernels behind lbm_codec_encode / lbm_codec_decode (bit-level parity tests).
#include <atomic>

#include "lbm_internal.h"
#include "lbm_kernels.cuh"

namespace lbmk {

static std::atomic<long long> g_launches{0};
void count_launch(long long n) { g_launches += n; }
long long launches() { return g_launches.load(); }

// out[n] = in[n] | FLAG_NEAR if cell n is fluid and at least one of its q-1 pull sources (x - c_i,
// periodic, R2) is a wall cell.  stream_collide then reads ONE flag byte per cell instead of the q
// the paper's kernel gathers.
template <int Q>
__global__ void __launch_bounds__(256) mark_near_kernel(const unsigned char *__restrict__ in, unsigned char *__restrict__ out,
                                                        int nx, int ny, int nz) {
    typedef Lat<Q> L;
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y, z = blockIdx.z;
    if (x >= nx) return;
    const long long n = x + (long long)nx * (y + (long long)ny * z);
    unsigned fl = in[n] & FLAG_WALL;
    if (!fl) {
        unsigned near = 0;
#pragma unroll
        for (int i = 1; i < Q; ++i) {
            int xs = x - L::c(i, 0), ys = y - L::c(i, 1), zs = z - L::c(i, 2);
            xs = xs < 0 ? nx - 1 : xs >= nx ? 0 : xs;
            ys = ys < 0 ? ny - 1 : ys >= ny ? 0 : ys;
            zs = zs < 0 ? nz - 1 : zs >= nz ? 0 : zs;
            near |= in[xs + (long long)nx * (ys + (long long)ny * zs)] & FLAG_WALL;
        }
        if (near) fl |= FLAG_NEAR;
    }
    out[n] = (unsigned char)fl;
}

cudaError_t launch_mark_near(int q, const unsigned char *in, unsigned char *out, int nx, int ny, int nz, cudaStream_t st) {
    const dim3 block(256), grid((nx + 255) / 256, ny, nz);
    if (q == 9) mark_near_kernel<9><<<grid, block, 0, st>>>(in, out, nx, ny, nz);
    else if (q == 19) mark_near_kernel<19><<<grid, block, 0, st>>>(in, out, nx, ny, nz);
    else if (q == 27) mark_near_kernel<27><<<grid, block, 0, st>>>(in, out, nx, ny, nz);
    else return cudaErrorInvalidValue;
    count_launch();
    return cudaGetLastError();
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

// ---- pair codecs vs scalar codecs, exhaustively, on the device ----------------------------------------
// PairCodec<F> (the staged kernel's converters) must return bit for bit what Codec<F> returns (times 2^SC):
// all 65 536 codes through dec1 / dec2 (both halves) and ALL 2^32 FP32 bit patterns through enc2 (both halves).
// Codec<F> itself is compared with the oracle by the tests; this closes the chain for PairCodec<F>.
template <int F>
__global__ void __launch_bounds__(256) pair_selftest_kernel(unsigned long long *mismatches) {
    typedef PairCodec<F> PC;
    const float up = pow2f(PC::SC);
    unsigned long long bad = 0;
    const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
    for (unsigned long long v = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; v < (1ull << 32); v += stride) {
        const unsigned b = (unsigned)v;
        const float x = __uint_as_float(b);
        const float other = __uint_as_float(b * 2654435761u + 12345u);          // an unrelated partner value
        const unsigned ref = Codec<F>::enc(x), ref_o = Codec<F>::enc(other);
        const unsigned w1 = PC::enc2(__fmul_rn(x, up), __fmul_rn(other, up));
        const unsigned w2 = PC::enc2(__fmul_rn(other, up), __fmul_rn(x, up));
        const bool nan = x != x || other != other;                              // NaN payloads of binary16 are not pinned
        if (!nan) bad += (w1 != (ref | (ref_o << 16))) + (w2 != (ref_o | (ref << 16)));
        if (v < 65536) {
            const unsigned c = (unsigned)v, c2 = (c * 40503u + 7u) & 0xFFFFu;
            const float r = __fmul_rn(Codec<F>::dec(c), up), r2 = __fmul_rn(Codec<F>::dec(c2), up);
            float a, d;
            PC::dec2(c | (c2 << 16), a, d);
            const float e = PC::dec1((int)(short)c);
            const bool cn = r != r || r2 != r2;
            if (cn) bad += !(a != a || !(r != r)) + !(d != d || !(r2 != r2)) + !(e != e || !(r != r));
            else bad += (__float_as_uint(a) != __float_as_uint(r)) + (__float_as_uint(d) != __float_as_uint(r2)) +
                        (__float_as_uint(e) != __float_as_uint(r));
        }
    }
    if (bad) atomicAdd(mismatches, bad);
}

cudaError_t launch_pair_selftest(int fmt, unsigned long long *mismatches_dev, cudaStream_t st) {
    const int blocks = 148 * 16;
    switch (fmt) {
        case F_FP16S: pair_selftest_kernel<F_FP16S><<<blocks, 256, 0, st>>>(mismatches_dev); break;
        case F_FP16C: pair_selftest_kernel<F_FP16C><<<blocks, 256, 0, st>>>(mismatches_dev); break;
        case F_P16_0S: pair_selftest_kernel<F_P16_0S><<<blocks, 256, 0, st>>>(mismatches_dev); break;
        case F_P16_1S: pair_selftest_kernel<F_P16_1S><<<blocks, 256, 0, st>>>(mismatches_dev); break;
        case F_P16_2C: pair_selftest_kernel<F_P16_2C><<<blocks, 256, 0, st>>>(mismatches_dev); break;
        case F_FP16: pair_selftest_kernel<F_FP16><<<blocks, 256, 0, st>>>(mismatches_dev); break;
        default: return cudaErrorInvalidValue;
    }
    count_launch();
    return cudaGetLastError();
}

}  // namespace lbmk
