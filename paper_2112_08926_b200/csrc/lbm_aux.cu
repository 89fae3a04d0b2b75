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

}  // namespace lbmk
