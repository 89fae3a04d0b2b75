// lbm_unit64.cu -- one (velocity set, storage type) instantiation unit of the FP64-arithmetic kernels in
// lbm_fp64.cuh.  Compiled once per pair with -DLBM_Q=<9|19|27> -DLBM_F=<7|8> (7 = LBM_FP64: double storage,
// 8 = LBM_FP64_FP32: float storage; see build.py).
#include <cmath>

#include "lbm_internal.h"
#include "lbm_fp64.cuh"

#ifndef LBM_Q
#error "compile with -DLBM_Q=<velocity set> -DLBM_F=<7|8>"
#endif

#define LBM_CAT_(a, b, c, d) a##b##c##d
#define LBM_CAT(a, b, c, d) LBM_CAT_(a, b, c, d)
#define LBM_UNIT_SYMBOL LBM_CAT(lbm_unit_q, LBM_Q, _f, LBM_F)
#define LBM_STR_(x) #x
#define LBM_STR(x) LBM_STR_(x)

namespace lbmk {
namespace {

using namespace f64;

constexpr int Q = LBM_Q;
#if LBM_F == 7
typedef double S;
#elif LBM_F == 8
typedef float S;
#else
#error "LBM_F must be 7 (FP64 storage) or 8 (FP32 storage) in this unit"
#endif

Params64 make64(const Params &p) {
    Params64 d;
    d.omega = 1.0 / (double)p.tau;
    d.one_m_omega = 1.0 - d.omega;
    d.omega_minus = 1.0 / (0.5 + p.trt_lambda / ((double)p.tau - 0.5));   // R13
    d.F[0] = (double)p.fx; d.F[1] = (double)p.fy; d.F[2] = (double)p.fz;
    d.cs = 1.0 / std::sqrt(3.0);
    return d;
}

template <bool FORCE, int COLL = 0>
cudaError_t launch_sc(const void *A, void *B, const Params &p, cudaStream_t st) {
    int bx = 32;
    while (bx < p.nx && bx < THREADS) bx <<= 1;
    const int by = THREADS / bx;
    const dim3 block(bx, by, 1);
    const dim3 grid((p.nx + bx - 1) / bx, (p.ny + by - 1) / by, p.nz);
    // resident CTAs per SM asked of the compiler (measured on 512^3 / 384^3): three (<= 80
    // registers) for double storage, where the kernel then runs at the HBM roofline; four (<= 64 registers, 28 bytes
    // of spills) for D2Q9 / D3Q19 float storage, which is bound by latency, not by bytes: 0.76 -> 0.83 of peak
    constexpr int MINB = (sizeof(S) == 4 && Q <= 19) ? 4 : 3;
    stream_collide64_kernel<Q, S, FORCE, MINB, COLL><<<grid, block, 0, st>>>((const S *)A, (S *)B, p, make64(p));
    count_launch();
    return cudaGetLastError();
}

cudaError_t stream_collide(const void *A, void *B, const Params &p, int V, int coll, bool force, cudaStream_t st) {
    (void)V;
    if (coll == 1) return force ? launch_sc<true, 1>(A, B, p, st) : launch_sc<false, 1>(A, B, p, st);   // TRT (R13)
    return force ? launch_sc<true>(A, B, p, st) : launch_sc<false>(A, B, p, st);
}

int blocks_for(long long N) {
    long long b = (N + 255) / 256;
    const long long cap = 148LL * 64;   // grid-stride loops: a few waves over the 148 SMs
    return (int)(b < cap ? (b < 1 ? 1 : b) : cap);
}

cudaError_t init(void *A, void *B, const float *rho, const float *u, long long N, bool /*shifted: always*/, cudaStream_t st) {
    init64_kernel<Q, S><<<blocks_for(N), 256, 0, st>>>((S *)A, (S *)B, rho, u, N);
    count_launch();
    return cudaGetLastError();
}

template <class OUT>
cudaError_t read_t(const void *A, const Params &p, bool force, OUT *rho, OUT *u, cudaStream_t st) {
    const Params64 d = make64(p);
    if (force) read_rho_u64_kernel<Q, S, true, OUT><<<blocks_for(p.N), 256, 0, st>>>((const S *)A, p, d, rho, u);
    else read_rho_u64_kernel<Q, S, false, OUT><<<blocks_for(p.N), 256, 0, st>>>((const S *)A, p, d, rho, u);
    count_launch();
    return cudaGetLastError();
}

cudaError_t read(const void *A, const Params &p, bool force, float *rho, float *u, cudaStream_t st) {
    return read_t<float>(A, p, force, rho, u, st);
}

cudaError_t read64(const void *A, const Params &p, bool force, double *rho, double *u, cudaStream_t st) {
    return read_t<double>(A, p, force, rho, u, st);
}

cudaError_t probe(const void *A, const Params &p, bool force, const long long *cells, int count, float *rho, float *u, cudaStream_t st) {
    const int blocks = (count + 127) / 128;
    const Params64 d = make64(p);
    if (force) probe_rho_u64_kernel<Q, S, true><<<blocks, 128, 0, st>>>((const S *)A, p, d, cells, count, rho, u);
    else probe_rho_u64_kernel<Q, S, false><<<blocks, 128, 0, st>>>((const S *)A, p, d, cells, count, rho, u);
    count_launch();
    return cudaGetLastError();
}

const char *name(int V, int coll, bool force) {
    (void)V;
    if (coll == 1)
        return force ? "stream_collide64_kernel<Q=" LBM_STR(LBM_Q) ",F=" LBM_STR(LBM_F) ",FORCE=1,COLL=TRT>"
                     : "stream_collide64_kernel<Q=" LBM_STR(LBM_Q) ",F=" LBM_STR(LBM_F) ",FORCE=0,COLL=TRT>";
    return force ? "stream_collide64_kernel<Q=" LBM_STR(LBM_Q) ",F=" LBM_STR(LBM_F) ",FORCE=1>"
                 : "stream_collide64_kernel<Q=" LBM_STR(LBM_Q) ",F=" LBM_STR(LBM_F) ",FORCE=0>";
}


}  // namespace

extern const UnitOps LBM_UNIT_SYMBOL;
const UnitOps LBM_UNIT_SYMBOL = {stream_collide, init, read, name, probe, read64};

}  // namespace lbmk
