// oracle/lbm.cpp -- CPU oracle for the fused LBM stream-collide step.  TEST INFRASTRUCTURE, NOT PRODUCT
// (see oracle.h).  Shares no code with the CUDA path.
//
// One time step, for every non-wall cell, in the order of the paper's kernel (Listing 2,
// PAPER.md:1014-1042) and its equations (24)-(28), on DDFs shifted by the lattice
// weights (section 2.2):
//   R2  pull:  f_i^temp(x) = f_i^A(x - e_i), periodic wrap on all axes        eq (24)
//   R3  halfway bounce-back when the pull source is a wall cell
//   R9  moving-wall term on a bounced link (named at PAPER.md:352, formula: DESIGN.md R9)
//   R4  rho = (sum_i f_i) + 1, "+1" last; momentum by alternating +/- sums     eq (25)-(26)
//   R5  u = j / rho  (with a body force: (j + F/2) / rho, R5/R10)
//   R6  clamp u to +-c
//   R7  shifted equilibrium "exactly as presented" in eq (3), 3 FMAs
//   R8  f_i^B(x) = fma(1-omega, f_i^temp, omega f_i^eq)                        eq (28)
//   R10 Guo forcing source term (named at PAPER.md:233, formula: DESIGN.md R10)
//   R15 equilibrium boundary cells (named at PAPER.md:322): never updated, they keep f^eq(rho0, u0) from init
//   R17 the same step WITHOUT DDF-shifting, eqs (19)-(23), the paper's negative control (dashed curves,
//       PAPER.md:265, 316): the stored quantity is f_i, rho = sum f_i (no "+1"), f^eq by eq (22)
//   R18 zero-gradient outflow cells (BASELINE configs[3]; NOT in the paper: DESIGN.md R18): every step such a cell takes
//       the shifted equilibrium of the density and velocity of its upstream (x - 1) neighbour's stored DDFs
// with load()/store() = the codecs of codecs.cpp applied at every read and write.
// PARITY UNPINNED (no external pin exists; fixed by DESIGN.md section 3 only): the operation order of R5 / R10, the
// pre-computation grouping of R7, rho_w = 1 in R9, writing both buffers in R11, R12 as the definition of the
// read-out, the D2Q9 / D3Q27 direction numbering.  Everything else is pinned by tests/test_oracle_lbm.py.
// Arithmetic type T = float reproduces the paper's FP32 arithmetic (parity runs); T = double is used
// for the analytic pins (tests/test_oracle_lbm.py).  Everything is written as plain loops over the
// velocity-set table; operation order is the one stated in DESIGN.md section 3.
#include "oracle.h"

#include <cmath>
#include <cstdlib>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

uint16_t orc_encode_one(int fmt, float x);
float orc_decode_one(int fmt, uint16_t c);
void orc_prepare_table(int fmt);

namespace {

// ---- velocity sets (R1) ------------------------------------------------------------------------
// D3Q19 numbering is fixed by the momentum sums printed at PAPER.md:62 and 955-959 and by the
// (i, i+1) opposite pairs of PAPER.md:1029-1031.  D2Q9 / D3Q27 numbering is not in the paper:
// D2Q9 = the z = 0 members of D3Q19 in the same order, D3Q27 = D3Q19 + the 8 corners (R1).
// Weights are the textbook ones (PAPER.md:66 names 1/3, 1/18, 1/36 for D3Q19; Table 1 pins all three sets).
struct VelSet {
    int q;
    int c[27][3];
    double w[27];
    int opp[27];
};

const int C27[27][3] = {
    {0, 0, 0},
    {1, 0, 0},  {-1, 0, 0},  {0, 1, 0},  {0, -1, 0},  {0, 0, 1},   {0, 0, -1},
    {1, 1, 0},  {-1, -1, 0}, {1, 0, 1},  {-1, 0, -1}, {0, 1, 1},   {0, -1, -1},
    {1, -1, 0}, {-1, 1, 0},  {1, 0, -1}, {-1, 0, 1},  {0, 1, -1},  {0, -1, 1},
    {1, 1, 1},  {-1, -1, -1}, {1, 1, -1}, {-1, -1, 1}, {1, -1, 1}, {-1, 1, -1}, {-1, 1, 1}, {1, -1, -1}};

VelSet make_velset(int velset) {
    VelSet v;
    std::memset(&v, 0, sizeof v);
    if (velset == 19 || velset == 27) {
        v.q = velset;
        for (int i = 0; i < v.q; ++i)
            for (int a = 0; a < 3; ++a) v.c[i][a] = C27[i][a];
    } else if (velset == 9) {
        v.q = 9;
        int k = 0;
        for (int i = 0; i < 19; ++i)
            if (C27[i][2] == 0) {
                for (int a = 0; a < 3; ++a) v.c[k][a] = C27[i][a];
                ++k;
            }
    } else {
        v.q = 0;
        return v;
    }
    for (int i = 0; i < v.q; ++i) {
        const int n2 = v.c[i][0] * v.c[i][0] + v.c[i][1] * v.c[i][1] + v.c[i][2] * v.c[i][2];
        if (velset == 19) v.w[i] = n2 == 0 ? 1.0 / 3.0 : n2 == 1 ? 1.0 / 18.0 : 1.0 / 36.0;
        if (velset == 9) v.w[i] = n2 == 0 ? 4.0 / 9.0 : n2 == 1 ? 1.0 / 9.0 : 1.0 / 36.0;
        if (velset == 27) v.w[i] = n2 == 0 ? 8.0 / 27.0 : n2 == 1 ? 2.0 / 27.0 : n2 == 2 ? 1.0 / 54.0 : 1.0 / 216.0;
        v.opp[i] = i == 0 ? 0 : (i % 2 ? i + 1 : i - 1);
    }
    return v;
}

template <class T> T fma_t(T a, T b, T c);
template <> float fma_t<float>(float a, float b, float c) { return std::fmaf(a, b, c); }
template <> double fma_t<double>(double a, double b, double c) { return std::fma(a, b, c); }

// c_i . v with the terms taken in x, y, z order, left to right, skipping zero components
template <class T>
T cdot(const int c[3], T vx, T vy, T vz) {
    const T v[3] = {vx, vy, vz};
    bool first = true;
    T s = T(0);
    for (int a = 0; a < 3; ++a) {
        if (c[a] == 0) continue;
        const T term = c[a] > 0 ? v[a] : -v[a];
        s = first ? term : s + term;
        first = false;
    }
    return s;
}

// R7: shifted equilibrium, eq (3) "exactly as presented"; footnote 1:
// f = A (1/2 (B^2 + C) +- B) + D with A = w rho, B = 3 u.c_i, C = -3 u.u, D = w (rho - 1): 3 FMAs.
// Surviving lines of equilibrium(): c3 = -3 (ux^2 + uy^2 + uz^2), rhom1 = rho - 1,
// then u is multiplied by 3.
// R17, shifted = false: eq (22), f = w rho ((u.c)^2 / (2 c^4) + u.c / c^2 + 1 - u.u / (2 c^2)), read with the
// same A, B, C as eq (3): f = A ((1/2 (B^2 + C) +- B) + 1), the "+ 1" added last inside the bracket (grouping: DESIGN.md R17).
template <class T>
void equilibrium(const VelSet &vs, T rho, T ux, T uy, T uz, T *feq, bool shifted = true) {
    const T c3 = T(-3) * (ux * ux + uy * uy + uz * uz);
    const T rhom1 = rho - T(1);
    ux *= T(3);
    uy *= T(3);
    uz *= T(3);
    if (!shifted) {
        feq[0] = ((T)vs.w[0] * rho) * (T(0.5) * c3 + T(1));
        for (int i = 1; i < vs.q; i += 2) {
            const T A = (T)vs.w[i] * rho;
            const T B = cdot<T>(vs.c[i], ux, uy, uz);
            const T t = fma_t<T>(B, B, c3);
            feq[i] = A * (fma_t<T>(T(0.5), t, B) + T(1));
            feq[i + 1] = A * (fma_t<T>(T(0.5), t, -B) + T(1));
        }
        return;
    }
    {
        const T w = (T)vs.w[0];
        feq[0] = fma_t<T>(w * rho, T(0.5) * c3, w * rhom1);
    }
    for (int i = 1; i < vs.q; i += 2) {
        const T w = (T)vs.w[i];
        const T A = w * rho, D = w * rhom1;
        const T B = cdot<T>(vs.c[i], ux, uy, uz);
        const T t = fma_t<T>(B, B, c3);
        feq[i] = fma_t<T>(A, fma_t<T>(T(0.5), t, B), D);
        feq[i + 1] = fma_t<T>(A, fma_t<T>(T(0.5), t, -B), D);
    }
}

// R4: rho = f0 + f1 + ... + f(q-1), then + 1; momentum component a: pairs (i, i+1)
// in index order, "+ (member with c_a = +1) - (the other)", strictly left to right.
template <class T>
void moments(const VelSet &vs, const T *f, T &rho, T j[3], bool shifted = true) {
    rho = f[0];
    for (int i = 1; i < vs.q; ++i) rho += f[i];
    if (shifted) rho += T(1);                                  // eq (25); eq (20) without DDF-shifting
    for (int a = 0; a < 3; ++a) {
        bool first = true;
        T s = T(0);
        for (int i = 1; i < vs.q; i += 2) {
            if (vs.c[i][a] == 0) continue;
            const int p = vs.c[i][a] > 0 ? i : i + 1, m = vs.c[i][a] > 0 ? i + 1 : i;
            s = first ? f[p] : s + f[p];
            s = s - f[m];
            first = false;
        }
        j[a] = s;
    }
}

}  // namespace

struct orc_sim {
    int nx, ny, nz, fmt, arith;
    int collision;                    // ORC_BGK / ORC_TRT
    bool shifted;                     // DDF-shifting (default); false: eqs (19)-(23), R17
    double lambda;                    // TRT magic parameter (R13)
    long N;
    VelSet vs;
    double tau;
    double force[3];
    bool has_force;
    std::vector<uint8_t> flags;
    std::vector<float> rho0, u0;      // fields given to init (wall velocity, wall read-out)
    std::vector<double> rho0d, u0d;
    // two DDF buffers, SoA [q][N], element type by format
    std::vector<uint16_t> h[2];
    std::vector<float> f[2];
    std::vector<double> d[2];
    std::vector<float> lut;           // decode of all 65536 codes (the table of codecs.cpp, evaluated once)
    int cur;
    long steps_done;
};

namespace {

template <class T>
T load(const orc_sim *s, int buf, int i, long n) {
    const size_t o = (size_t)i * s->N + n;
    if (s->fmt == ORC_FP32) return (T)s->f[buf][o];
    if (s->fmt == ORC_FP64) return (T)s->d[buf][o];
    return (T)s->lut[s->h[buf][o]];
}

template <class T>
void store(orc_sim *s, int buf, int i, long n, T x) {
    const size_t o = (size_t)i * s->N + n;
    if (s->fmt == ORC_FP32) s->f[buf][o] = (float)x;
    else if (s->fmt == ORC_FP64) s->d[buf][o] = (double)x;
    else s->h[buf][o] = orc_encode_one(s->fmt, (float)x);
}

template <class T>
void wall_velocity(const orc_sim *s, long n, T uw[3]) {
    for (int a = 0; a < 3; ++a)
        uw[a] = s->arith == ORC_ARITH_F64 && !s->u0d.empty() ? (T)s->u0d[(size_t)a * s->N + n]
                                                                : (T)s->u0[(size_t)a * s->N + n];
}

template <class T>
void init_t(orc_sim *s, const T *rho, const T *u) {
    // R11: every cell, walls included; both buffers (R11)
    const VelSet &vs = s->vs;
#pragma omp parallel for schedule(static)
    for (long n = 0; n < s->N; ++n) {
        T feq[27];
        equilibrium<T>(vs, rho[n], u[n], u[s->N + n], u[2 * s->N + n], feq, s->shifted);
        for (int i = 0; i < vs.q; ++i) {
            store<T>(s, 0, i, n, feq[i]);
            store<T>(s, 1, i, n, feq[i]);
        }
    }
    s->cur = 0;
    s->steps_done = 0;
}

template <class T>
void step_t(orc_sim *s) {
    const VelSet &vs = s->vs;
    const int nx = s->nx, ny = s->ny, nz = s->nz, q = vs.q;
    const int A = s->cur, Bb = 1 - s->cur;
    const T omega = T(1) / (T)s->tau;                     // R8: omega = dt / tau
    const T one_m_omega = T(1) - omega;
    // TRT (R13): omega- from the magic parameter, 1/omega- = 1/2 + Lambda / (tau - 1/2)
    const T omega_m = T(1) / (T(0.5) + (T)s->lambda / ((T)s->tau - T(0.5)));
    const T cs = sizeof(T) == 4 ? (T)0.57735027f : (T)(1.0 / std::sqrt(3.0));   // R6: c = 1/sqrt(3)
    const T F[3] = {(T)s->force[0], (T)s->force[1], (T)s->force[2]};
    const bool forced = s->has_force;

#pragma omp parallel for collapse(2) schedule(static)
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                const long n = x + (long)nx * (y + (long)ny * z);
                if (s->flags[n] & (ORC_FLAG_WALL | ORC_FLAG_EQ)) continue;   // PAPER.md:1017; R15: E cells keep feq(rho0, u0)
                T fh[27];
                if (s->flags[n] & ORC_FLAG_OUT) {
                    // R18: density and velocity of the upstream neighbour's stored DDFs (read-out rule R12: local moments,
                    // u = (j - F/2) / rho, no clamp), imposed here as an equilibrium
                    const long up = (x - 1 + nx) % nx + (long)nx * (y + (long)ny * z);
                    for (int i = 0; i < q; ++i) fh[i] = load<T>(s, A, i, up);
                    T rho, j[3], u[3];
                    moments<T>(vs, fh, rho, j, s->shifted);
                    for (int a = 0; a < 3; ++a) u[a] = (forced ? fma_t<T>(T(-0.5), F[a], j[a]) : j[a]) / rho;
                    T feq[27];
                    equilibrium<T>(vs, rho, u[0], u[1], u[2], feq, s->shifted);
                    for (int i = 0; i < q; ++i) store<T>(s, Bb, i, n, feq[i]);
                    continue;
                }
                fh[0] = load<T>(s, A, 0, n);
                for (int i = 1; i < q; ++i) {
                    const int xs = (x - vs.c[i][0] + nx) % nx;        // R2, eq (24)
                    const int ys = (y - vs.c[i][1] + ny) % ny;
                    const int zs = (z - vs.c[i][2] + nz) % nz;
                    const long src = xs + (long)nx * (ys + (long)ny * zs);
                    if (s->flags[src] & ORC_FLAG_WALL) {              // R3
                        T v = load<T>(s, A, vs.opp[i], n);
                        T uw[3];
                        wall_velocity<T>(s, src, uw);
                        if (uw[0] != T(0) || uw[1] != T(0) || uw[2] != T(0)) {   // R9, rho_w = 1
                            const T w6 = (T)(6.0 * vs.w[i]);
                            v = v + w6 * cdot<T>(vs.c[i], uw[0], uw[1], uw[2]);
                        }
                        fh[i] = v;
                    } else {
                        fh[i] = load<T>(s, A, i, src);
                    }
                }
                T rho, j[3];
                moments<T>(vs, fh, rho, j, s->shifted);               // R4
                T u[3];
                for (int a = 0; a < 3; ++a) {                         // R5
                    const T ja = forced ? fma_t<T>(T(0.5), F[a], j[a]) : j[a];
                    u[a] = ja / rho;
                    u[a] = std::fmin(std::fmax(u[a], -cs), cs);       // R6
                }
                T feq[27];
                equilibrium<T>(vs, rho, u[0], u[1], u[2], feq, s->shifted);   // R7
                T uF = T(0);
                if (forced) uF = u[0] * F[0] + u[1] * F[1] + u[2] * F[2];
                if (s->collision == ORC_TRT) {
                    // R13 (NOT in the paper, which only names TRT): two-relaxation-time collision
                    // (Ginzburg et al.): per opposite pair (i, i') the symmetric part (f_i + f_i')/2 relaxes with
                    // omega+ = dt/tau, the antisymmetric part (f_i - f_i')/2 with omega-, where
                    // Lambda = (1/omega+ - 1/2)(1/omega- - 1/2); the rest DDF has no antisymmetric part.  The Guo
                    // source splits the same way: symmetric w (9 (c.u)(c.F) - 3 u.F) with (1 - omega+/2),
                    // antisymmetric 3 w c.F with (1 - omega-/2).
                    const T gp = T(1) - T(0.5) * omega, gm = T(1) - T(0.5) * omega_m;
                    {
                        T out = fma_t<T>(one_m_omega, fh[0], omega * feq[0]);
                        if (forced) out = out + (gp * (T)vs.w[0]) * (-(T(3) * uF));
                        store<T>(s, Bb, 0, n, out);
                    }
                    for (int i = 1; i < q; i += 2) {
                        const T fp = T(0.5) * (fh[i] + fh[i + 1]), fm = T(0.5) * (fh[i] - fh[i + 1]);
                        const T ep = T(0.5) * (feq[i] + feq[i + 1]), em = T(0.5) * (feq[i] - feq[i + 1]);
                        const T a = omega * (fp - ep), b = omega_m * (fm - em);
                        T o1 = (fh[i] - a) - b, o2 = (fh[i + 1] - a) + b;
                        if (forced) {
                            const T w = (T)vs.w[i];
                            const T cu = cdot<T>(vs.c[i], u[0], u[1], u[2]);
                            const T cF = cdot<T>(vs.c[i], F[0], F[1], F[2]);
                            const T Sp = (gp * w) * fma_t<T>(T(9) * cu, cF, -(T(3) * uF));
                            const T Sm = (gm * w) * (T(3) * cF);
                            o1 = (o1 + Sp) + Sm;
                            o2 = (o2 + Sp) - Sm;
                        }
                        store<T>(s, Bb, i, n, o1);
                        store<T>(s, Bb, i + 1, n, o2);
                    }
                    continue;
                }
                for (int i = 0; i < q; ++i) {
                    T out = fma_t<T>(one_m_omega, fh[i], omega * feq[i]);          // R8
                    if (forced) {                                                  // R10
                        const T pref = (T(1) - T(0.5) * omega) * (T)vs.w[i];
                        const T cu = i == 0 ? T(0) : cdot<T>(vs.c[i], u[0], u[1], u[2]);
                        const T cF = i == 0 ? T(0) : cdot<T>(vs.c[i], F[0], F[1], F[2]);
                        out = out + pref * fma_t<T>(T(9) * cu, cF, T(3) * (cF - uF));
                    }
                    store<T>(s, Bb, i, n, out);
                }
            }
    s->cur = Bb;
    s->steps_done += 1;
}

template <class T>
void read_t(orc_sim *s, T *rho_out, T *u_out) {
    // R12: local moments of the stored (post-collision) DDFs of the current buffer; with a force the
    // physical velocity is (j - F/2)/rho; wall cells return the fields given to init.
    const VelSet &vs = s->vs;
    const T F[3] = {(T)s->force[0], (T)s->force[1], (T)s->force[2]};
#pragma omp parallel for schedule(static)
    for (long n = 0; n < s->N; ++n) {
        if (s->flags[n] & (ORC_FLAG_WALL | ORC_FLAG_EQ)) {
            const bool dbl = s->arith == ORC_ARITH_F64 && !s->rho0d.empty();
            if (rho_out) rho_out[n] = dbl ? (T)s->rho0d[n] : (T)s->rho0[n];
            if (u_out)
                for (int a = 0; a < 3; ++a)
                    u_out[(size_t)a * s->N + n] = dbl ? (T)s->u0d[(size_t)a * s->N + n] : (T)s->u0[(size_t)a * s->N + n];
            continue;
        }
        T fh[27], rho, j[3];
        for (int i = 0; i < vs.q; ++i) fh[i] = load<T>(s, s->cur, i, n);
        moments<T>(vs, fh, rho, j, s->shifted);
        if (rho_out) rho_out[n] = rho;
        if (u_out)
            for (int a = 0; a < 3; ++a) {
                const T ja = s->has_force ? fma_t<T>(T(-0.5), F[a], j[a]) : j[a];
                u_out[(size_t)a * s->N + n] = ja / rho;
            }
    }
}

}  // namespace

extern "C" {

orc_sim *orc_create(int nx, int ny, int nz, int velset, int fmt, int arith, double tau, const double force[3]) {
    if (nx < 1 || ny < 1 || nz < 1 || !(tau > 0.5)) return nullptr;
    if (fmt < ORC_FP32 || fmt > ORC_FP64) return nullptr;
    if (fmt == ORC_FP64 && arith != ORC_ARITH_F64) return nullptr;
    if (velset == 9 && nz != 1) return nullptr;
    VelSet vs = make_velset(velset);
    if (vs.q == 0) return nullptr;
    orc_sim *s = new orc_sim();
    s->nx = nx; s->ny = ny; s->nz = nz; s->fmt = fmt; s->arith = arith;
    s->N = (long)nx * ny * nz;
    s->vs = vs;
    s->tau = arith == ORC_ARITH_F32 ? (double)(float)tau : tau;
    s->has_force = false;
    for (int a = 0; a < 3; ++a) {
        s->force[a] = force ? (arith == ORC_ARITH_F32 ? (double)(float)force[a] : force[a]) : 0.0;
        if (s->force[a] != 0.0) s->has_force = true;
    }
    s->flags.assign(s->N, 0);
    const size_t tot = (size_t)vs.q * s->N;
    for (int b = 0; b < 2; ++b) {
        if (fmt == ORC_FP32) s->f[b].assign(tot, 0.f);
        else if (fmt == ORC_FP64) s->d[b].assign(tot, 0.0);
        else s->h[b].assign(tot, 0);
    }
    if (fmt >= ORC_FP16S && fmt <= ORC_FP16) {
        orc_prepare_table(fmt);
        s->lut.resize(65536);
        for (unsigned c = 0; c < 65536; ++c) s->lut[c] = orc_decode_one(fmt, (uint16_t)c);
    }
    s->cur = 0;
    s->steps_done = 0;
    s->collision = ORC_BGK;
    s->shifted = true;
    s->lambda = 3.0 / 16.0;
    return s;
}

int orc_set_collision(orc_sim *s, int collision, double lambda) {
    if (!s || (collision != ORC_BGK && collision != ORC_TRT) || !(lambda > 0.0)) return -1;
    s->collision = collision;
    s->lambda = s->arith == ORC_ARITH_F32 ? (double)(float)lambda : lambda;
    return 0;
}

int orc_set_shifting(orc_sim *s, int on) {
    if (!s) return -1;
    s->shifted = on != 0;
    return 0;
}

void orc_destroy(orc_sim *s) { delete s; }

int orc_set_flags(orc_sim *s, const uint8_t *flags) {
    if (!s || !flags) return -1;
    std::memcpy(s->flags.data(), flags, s->N);
    return 0;
}

int orc_init(orc_sim *s, const float *rho, const float *u) {
    if (!s || !rho || !u) return -1;
    s->rho0.assign(rho, rho + s->N);
    s->u0.assign(u, u + 3 * s->N);
    s->rho0d.clear();
    s->u0d.clear();
    if (s->arith == ORC_ARITH_F32) init_t<float>(s, rho, u);
    else {
        std::vector<double> r(rho, rho + s->N), v(u, u + 3 * s->N);
        init_t<double>(s, r.data(), v.data());
    }
    return 0;
}

int orc_init_f64(orc_sim *s, const double *rho, const double *u) {
    if (!s || !rho || !u || s->arith != ORC_ARITH_F64) return -1;
    s->rho0d.assign(rho, rho + s->N);
    s->u0d.assign(u, u + 3 * s->N);
    s->rho0.assign(rho, rho + s->N);
    s->u0.assign(u, u + 3 * s->N);
    init_t<double>(s, rho, u);
    return 0;
}

int orc_step(orc_sim *s, int n) {
    if (!s || n < 0) return -1;
    for (int k = 0; k < n; ++k) {
        if (s->arith == ORC_ARITH_F32) step_t<float>(s);
        else step_t<double>(s);
    }
    return 0;
}

int orc_read_rho_u(orc_sim *s, float *rho, float *u) {
    if (!s) return -1;
    if (s->arith == ORC_ARITH_F32) read_t<float>(s, rho, u);
    else {
        std::vector<double> r(s->N), v(3 * s->N);
        read_t<double>(s, r.data(), v.data());
        if (rho) for (long n = 0; n < s->N; ++n) rho[n] = (float)r[n];
        if (u) for (long n = 0; n < 3 * s->N; ++n) u[n] = (float)v[n];
    }
    return 0;
}

int orc_read_rho_u_f64(orc_sim *s, double *rho, double *u) {
    if (!s || s->arith != ORC_ARITH_F64) return -1;
    read_t<double>(s, rho, u);
    return 0;
}

int orc_read_ddf(orc_sim *s, int i, void *out) {
    if (!s || i < 0 || i >= s->vs.q || !out) return -1;
    const size_t o = (size_t)i * s->N;
    if (s->fmt == ORC_FP32) std::memcpy(out, s->f[s->cur].data() + o, s->N * 4);
    else if (s->fmt == ORC_FP64) std::memcpy(out, s->d[s->cur].data() + o, s->N * 8);
    else std::memcpy(out, s->h[s->cur].data() + o, s->N * 2);
    return 0;
}

double orc_sum_ddf(orc_sim *s) {
    long double acc = 0.0L;
    for (int i = 0; i < s->vs.q; ++i)
        for (long n = 0; n < s->N; ++n) acc += (long double)load<double>(s, s->cur, i, n);
    return (double)acc;
}

int orc_set_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
    return omp_get_max_threads();
#else
    (void)n;
    return 1;
#endif
}

int orc_velocity_set(int velset, int *c, double *w, int *opp) {
    VelSet vs = make_velset(velset);
    if (vs.q == 0) return -1;
    for (int i = 0; i < vs.q; ++i) {
        for (int a = 0; a < 3; ++a) c[3 * i + a] = vs.c[i][a];
        w[i] = vs.w[i];
        opp[i] = vs.opp[i];
    }
    return vs.q;
}

int orc_equilibrium(int velset, int arith, double rho, double ux, double uy, double uz, double *feq) {
    VelSet vs = make_velset(velset);
    if (vs.q == 0) return -1;
    if (arith == ORC_ARITH_F32) {
        float f[27];
        equilibrium<float>(vs, (float)rho, (float)ux, (float)uy, (float)uz, f);
        for (int i = 0; i < vs.q; ++i) feq[i] = f[i];
    } else {
        equilibrium<double>(vs, rho, ux, uy, uz, feq);
    }
    return vs.q;
}

}  // extern "C"
