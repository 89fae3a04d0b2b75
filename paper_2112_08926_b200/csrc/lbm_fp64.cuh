// lbm_fp64.cuh -- the stream-collide step with FP64 ARITHMETIC: the paper's FP64/FP64 and FP64/FP32 columns
// (arithmetic / storage precision; Tables 3-5; "FP64/xx") and the
// FP64 storage of config 5 of BASELINE.json.
//
// Same path as lbm_kernels.cuh (Listing 2; eqs (24)-(28)) and the same
// readings R1-R12, R15, with every FP32 operation replaced by the IEEE binary64 one in the
// same order: explicitly rounded intrinsics (never contracted), IEEE division, fma where the paper counts an FMA.
// Storage S = double (identity load / store) or float (load widens exactly, store rounds to nearest even,
// PAPER.md:787-790 with the cast of a double).  Weights are the doubles 1/3, 1/18, 1/36, ... (Table 1,
// PAPER.md:72-77), the clamp constant is 1/sqrt(3) in double.  The init fields, the wall velocity
// and the body force stay FP32 at the boundary (include/lbm.h) and are widened exactly.
//
// One cell per thread: 19 eight-byte streams per warp are 256-byte coalesced segments already, and two cells of
// doubles per thread would not fit the register file at a useful occupancy.  305 B per cell (FP64/FP64) against
// 177 FP64 instructions (86 DFMA, 55 DADD, 36 DMUL): bound by HBM, the FP64 pipe is 22% busy.
// MINB = resident CTAs per SM the register allocation is held to (chosen per storage type by the launcher).
#pragma once
#include "lbm_lattice.cuh"

namespace lbmk {

struct Params64 {
    double omega, one_m_omega;      // omega = dt / tau in double, from the float tau of lbm_create
    double omega_minus;             // TRT (R13): 1 / omega- = 1/2 + Lambda / (tau - 1/2)
    double F[3];                    // uniform body force, widened
    double cs;                      // 1 / sqrt(3)
};

namespace f64 {

__device__ __forceinline__ double add(double a, double b) { return __dadd_rn(a, b); }
__device__ __forceinline__ double sub(double a, double b) { return __dsub_rn(a, b); }
__device__ __forceinline__ double mul(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ double fma_(double a, double b, double c) { return __fma_rn(a, b, c); }

template <int Q>
__device__ __forceinline__ double wgt(int i) { return Lat<Q>::wd(i); }

// c_i . v, terms in x, y, z order, left to right, zero components skipped (i is a compile-time constant after unrolling)
template <int Q>
__device__ __forceinline__ double cdot(int i, double vx, double vy, double vz) {
    typedef Lat<Q> L;
    const double v[3] = {vx, vy, vz};
    double s = 0.0;
    bool first = true;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        if (L::c(i, a) == 0) continue;
        const double term = L::c(i, a) > 0 ? v[a] : -v[a];
        s = first ? term : add(s, term);
        first = false;
    }
    return s;
}

// R4: rho = (f0 + f1 + ... + f_{q-1}) + 1, the "+1" last; momentum by the alternating sums
// of PAPER.md:62, 955-959, left to right
template <int Q>
__device__ __forceinline__ void moments(const double (&f)[Q], double &rho, double (&j)[3]) {
    typedef Lat<Q> L;
    double sum = f[0];
#pragma unroll
    for (int i = 1; i < Q; ++i) sum = add(sum, f[i]);
    rho = add(sum, 1.0);
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        double s = 0.0;
        bool first = true;
#pragma unroll
        for (int i = 1; i < Q; i += 2) {
            if (L::c(i, a) == 0) continue;
            const int p = L::c(i, a) > 0 ? i : i + 1, m = L::c(i, a) > 0 ? i + 1 : i;
            s = first ? f[p] : add(s, f[p]);
            s = sub(s, f[m]);
            first = false;
        }
        j[a] = s;
    }
}

// R7: shifted equilibrium, eq (3): three FMAs per direction
template <int Q>
__device__ __forceinline__ void equilibrium(double rho, double ux, double uy, double uz, double (&feq)[Q]) {
    const double c3 = mul(-3.0, add(add(mul(ux, ux), mul(uy, uy)), mul(uz, uz)));
    const double rhom1 = sub(rho, 1.0);
    ux = mul(ux, 3.0);
    uy = mul(uy, 3.0);
    uz = mul(uz, 3.0);
    feq[0] = fma_(mul(wgt<Q>(0), rho), mul(0.5, c3), mul(wgt<Q>(0), rhom1));
#pragma unroll
    for (int i = 1; i < Q; i += 2) {
        const double A = mul(wgt<Q>(i), rho), D = mul(wgt<Q>(i), rhom1);
        const double B = cdot<Q>(i, ux, uy, uz);
        const double t = fma_(B, B, c3);
        feq[i] = fma_(A, fma_(0.5, t, B), D);
        feq[i + 1] = fma_(A, fma_(0.5, t, -B), D);
    }
}

// R4 moments, R5 velocity (+ F/2), R6 clamp, R7 equilibrium, R8 BGK (eq (28)), R10 Guo source
template <int Q, bool FORCE>
__device__ __forceinline__ void collide_bgk(double (&f)[Q], const Params64 &d) {
    double rho, j[3], u[3];
    moments<Q>(f, rho, j);
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const double ja = FORCE ? fma_(0.5, d.F[a], j[a]) : j[a];
        u[a] = __ddiv_rn(ja, rho);
        u[a] = fmin(fmax(u[a], -d.cs), d.cs);
    }
    double feq[Q];
    equilibrium<Q>(rho, u[0], u[1], u[2], feq);
    double uF = 0.0;
    if (FORCE) uF = add(add(mul(u[0], d.F[0]), mul(u[1], d.F[1])), mul(u[2], d.F[2]));
#pragma unroll
    for (int i = 0; i < Q; ++i) {
        double out = fma_(d.one_m_omega, f[i], mul(d.omega, feq[i]));
        if (FORCE) {
            const double pref = mul(sub(1.0, mul(0.5, d.omega)), wgt<Q>(i));
            const double cu = i == 0 ? 0.0 : cdot<Q>(i, u[0], u[1], u[2]);
            const double cF = i == 0 ? 0.0 : cdot<Q>(i, d.F[0], d.F[1], d.F[2]);
            out = add(out, mul(pref, fma_(mul(9.0, cu), cF, mul(3.0, sub(cF, uF)))));
        }
        f[i] = out;
    }
}

// TRT (R13; NOT defined by the paper, which only names it): as collide_bgk up to the equilibrium,
// then per opposite pair (i, i + 1) the symmetric part relaxes with omega+, the antisymmetric part with omega-;
// the Guo source splits the same way.
template <int Q, bool FORCE>
__device__ __forceinline__ void collide_trt(double (&f)[Q], const Params64 &d) {
    double rho, j[3], u[3];
    moments<Q>(f, rho, j);
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const double ja = FORCE ? fma_(0.5, d.F[a], j[a]) : j[a];
        u[a] = __ddiv_rn(ja, rho);
        u[a] = fmin(fmax(u[a], -d.cs), d.cs);
    }
    double feq[Q];
    equilibrium<Q>(rho, u[0], u[1], u[2], feq);
    double uF = 0.0;
    if (FORCE) uF = add(add(mul(u[0], d.F[0]), mul(u[1], d.F[1])), mul(u[2], d.F[2]));
    const double gp = sub(1.0, mul(0.5, d.omega)), gm = sub(1.0, mul(0.5, d.omega_minus));
    const double hop = mul(0.5, d.omega), hom = mul(0.5, d.omega_minus);
    f[0] = fma_(d.one_m_omega, f[0], mul(d.omega, feq[0]));
    if (FORCE) f[0] = add(f[0], mul(mul(gp, wgt<Q>(0)), -mul(3.0, uF)));
#pragma unroll
    for (int i = 1; i < Q; i += 2) {
        // the halves of f+-, e+- folded into the rates (exact scalings, as in lbm_lattice.cuh's TrtPairs)
        const double dp = sub(add(f[i], f[i + 1]), add(feq[i], feq[i + 1]));
        const double dm = sub(sub(f[i], f[i + 1]), sub(feq[i], feq[i + 1]));
        const double a = mul(hop, dp), b = mul(hom, dm);
        double o1 = sub(sub(f[i], a), b), o2 = add(sub(f[i + 1], a), b);
        if (FORCE) {
            const double cu = cdot<Q>(i, u[0], u[1], u[2]);
            const double cF = cdot<Q>(i, d.F[0], d.F[1], d.F[2]);
            const double Sp = mul(mul(gp, wgt<Q>(i)), fma_(mul(9.0, cu), cF, -mul(3.0, uF)));
            const double Sm = mul(mul(gm, wgt<Q>(i)), mul(3.0, cF));
            o1 = add(add(o1, Sp), Sm);
            o2 = sub(add(o2, Sp), Sm);
        }
        f[i] = o1;
        f[i + 1] = o2;
    }
}

template <class S>
__device__ __forceinline__ double ld(const S *p) { return (double)__ldg(p); }
template <class S>
__device__ __forceinline__ void st(S *p, double x) { *p = (S)x; }      // float: cvt.rn.f32.f64

constexpr int THREADS = 256;

// grid: x = tiles of BX cells along x, y = tiles of BY rows, z = plane; blockDim = (BX, BY), BX * BY = THREADS
template <int Q, class S, bool FORCE, int MINB, int COLL = 0>
__global__ void __launch_bounds__(THREADS, MINB)
stream_collide64_kernel(const S *__restrict__ A, S *__restrict__ B, const Params p, const Params64 d) {
    typedef Lat<Q> L;
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z;
    if (x >= p.nx || y >= p.ny) return;

    // R2: periodic neighbours without modulo.  Pull sources are addressed relative to the own cell (in-plane offsets
    // in 32 bits, the plane offset in 64) and the direction's base walks by N elements, instead of q absolute
    // 64-bit element indices.
    const int dyv[3] = {y == 0 ? p.ny - 1 : -1, 0, y == p.ny - 1 ? 1 - p.ny : 1};            // rows to y-1, y, y+1
    const long long plane = (long long)p.nx * p.ny;
    const long long dzv[3] = {z == 0 ? plane * (p.nz - 1) : -plane, 0, z == p.nz - 1 ? -plane * (p.nz - 1) : plane};
    const int dxv[3] = {x == 0 ? p.nx - 1 : -1, 0, x == p.nx - 1 ? 1 - p.nx : 1};
    const long long own = (long long)p.nx * (y + (long long)p.ny * z) + x;

    const unsigned flag = __ldg(p.flags + own);                          // a1
    if (flag & FLAG_FIXED) return;                                       // PAPER.md:1017; R15

    double f[Q];
    if (flag & FLAG_OUT) {
        // R18 (not in the paper): zero-gradient outflow cell -- the equilibrium of the upstream (x - 1) neighbour's density
        // and velocity (read-out rule R12: local moments of its stored DDFs, u = (j - F/2) / rho, no clamp)
        const S *Ai = A + own + dxv[0];
#pragma unroll
        for (int i = 0; i < Q; ++i) {
            f[i] = ld(Ai);
            Ai += p.N;
        }
        double rho, j[3], u[3];
        moments<Q>(f, rho, j);
#pragma unroll
        for (int a = 0; a < 3; ++a) u[a] = __ddiv_rn(FORCE ? fma_(-0.5, d.F[a], j[a]) : j[a], rho);
        equilibrium<Q>(rho, u[0], u[1], u[2], f);
        S *Bo = B + own;
#pragma unroll
        for (int i = 0; i < Q; ++i) {
            st(Bo, f[i]);
            Bo += p.N;
        }
        return;
    }
    if (!(flag & FLAG_NEAR)) {
        const S *Ai = A + own;
#pragma unroll
        for (int i = 0; i < Q; ++i) {                                    // a2, a3: source cell x - c_i
            const long long off = dzv[1 - L::c(i, 2)] + (dyv[1 - L::c(i, 1)] * p.nx + dxv[1 - L::c(i, 0)]);
            f[i] = ld(Ai + off);
            Ai += p.N;
        }
    } else {
        f[0] = ld(A + own);
#pragma unroll
        for (int i = 1; i < Q; ++i) {
            const long long src = own + dzv[1 - L::c(i, 2)] + (dyv[1 - L::c(i, 1)] * p.nx + dxv[1 - L::c(i, 0)]);
            if (__ldg(p.flags + src) & FLAG_WALL) {                      // R3
                double v = ld(A + (long long)L::opp(i) * p.N + own);
                const double uwx = (double)__ldg(p.u0 + src), uwy = (double)__ldg(p.u0 + p.N + src),
                             uwz = (double)__ldg(p.u0 + 2 * p.N + src);
                if (uwx != 0.0 || uwy != 0.0 || uwz != 0.0)              // R9, rho_w = 1
                    v = add(v, mul(6.0 * wgt<Q>(i), cdot<Q>(i, uwx, uwy, uwz)));
                f[i] = v;
            } else {
                f[i] = ld(A + (long long)i * p.N + src);
            }
        }
    }
    if (COLL == 0) collide_bgk<Q, FORCE>(f, d);
    else collide_trt<Q, FORCE>(f, d);
    S *Bi = B + own;
#pragma unroll
    for (int i = 0; i < Q; ++i) {                                        // a10
        st(Bi, f[i]);
        Bi += p.N;
    }
}

// init: every cell, walls included, both buffers (R11)
template <int Q, class S>
__global__ void __launch_bounds__(256)
init64_kernel(S *__restrict__ A, S *__restrict__ B, const float *__restrict__ rho, const float *__restrict__ u, long long N) {
    for (long long n = (long long)blockIdx.x * blockDim.x + threadIdx.x; n < N; n += (long long)gridDim.x * blockDim.x) {
        double feq[Q];
        equilibrium<Q>((double)__ldg(rho + n), (double)__ldg(u + n), (double)__ldg(u + N + n), (double)__ldg(u + 2 * N + n), feq);
#pragma unroll
        for (int i = 0; i < Q; ++i) {
            st(A + (long long)i * N + n, feq[i]);
            st(B + (long long)i * N + n, feq[i]);
        }
    }
}

// R12: local moments of cell n of the current buffer; flagged cells return the fields given to init
template <int Q, class S, bool FORCE>
__device__ __forceinline__ void cell_rho_u(const S *__restrict__ A, const Params &p, const Params64 &d, long long n, double &rho,
                                           double (&u)[3]) {
    const long long N = p.N;
    if (__ldg(p.flags + n) & FLAG_FIXED) {
        rho = (double)__ldg(p.rho0 + n);
#pragma unroll
        for (int a = 0; a < 3; ++a) u[a] = (double)__ldg(p.u0 + a * N + n);
    } else {
        double f[Q], j[3];
#pragma unroll
        for (int i = 0; i < Q; ++i) f[i] = ld(A + (long long)i * N + n);
        moments<Q>(f, rho, j);
#pragma unroll
        for (int a = 0; a < 3; ++a) u[a] = __ddiv_rn(FORCE ? fma_(-0.5, d.F[a], j[a]) : j[a], rho);
    }
}

// OUT = float (lbm_read_rho_u: the doubles rounded to nearest) or double (lbm_read_rho_u_f64)
template <int Q, class S, bool FORCE, class OUT>
__global__ void __launch_bounds__(256)
read_rho_u64_kernel(const S *__restrict__ A, const Params p, const Params64 d, OUT *__restrict__ rho_out, OUT *__restrict__ u_out) {
    const long long N = p.N;
    for (long long n = (long long)blockIdx.x * blockDim.x + threadIdx.x; n < N; n += (long long)gridDim.x * blockDim.x) {
        double rho, u[3];
        cell_rho_u<Q, S, FORCE>(A, p, d, n, rho, u);
        if (rho_out) rho_out[n] = (OUT)rho;
        if (u_out) {
#pragma unroll
            for (int a = 0; a < 3; ++a) u_out[a * N + n] = (OUT)u[a];
        }
    }
}

template <int Q, class S, bool FORCE>
__global__ void __launch_bounds__(128)
probe_rho_u64_kernel(const S *__restrict__ A, const Params p, const Params64 d, const long long *__restrict__ cells, int count,
                     float *__restrict__ rho_out, float *__restrict__ u_out) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= count) return;
    double rho, u[3];
    cell_rho_u<Q, S, FORCE>(A, p, d, cells[k], rho, u);
    rho_out[k] = (float)rho;
#pragma unroll
    for (int a = 0; a < 3; ++a) u_out[a * count + k] = (float)u[a];
}

}  // namespace f64
}  // namespace lbmk
