// lbm_bulk.cuh -- the shared-memory-staged stream-collide kernel for sm_100a: the same time step as
// stream_collide_kernel (Listing 2; eqs (24)-(28)), with the DDF
// streams moved by the bulk-copy engine (cp.async.bulk, SASS UBLKCP) instead of per-thread loads and stores.
//
// Why (profiles/r01a_first_path.md): with per-thread LDG/STG every 16-bit format is issue-bound on B200, and
// the largest single item is 64-bit address arithmetic -- 19 streams x (base + i*N + row + x) per thread.  In
// a structure-of-arrays pull step every direction of a row of cells is ONE contiguous segment of ONE source
// row (eq (24)), so a tile needs q plain 1-D copies; once the segments sit in shared
// memory every address is "thread base + compile-time immediate".
//
// Shape of the kernel
//   * persistent CTAs (grid = SMs x resident CTAs, two per SM), tiles handed out round-robin.  A stage holds up to
//     RMAX*TX cells (TX = 2*NT = 512; RMAX = 1, 2 or 4 by velocity set and element size).  If a row fits (nx <=
//     RMAX*TX) a tile is as many whole consecutive rows of one z-plane as fit: in the SoA layout they are ONE
//     contiguous segment per direction, one copy.  Longer rows are cut into segments of RMAX*TX cells.  NT threads,
//     two neighbouring cells each, pair after pair across the tile;
//   * every warp issues a share of the copies (one lane issues; the bulk-copy instruction is warp-uniform): warp v
//     the directions v, v+NW, ... -- the copy of direction i is the segment of source row (y - c_iy, z - c_iz)
//     (periodic wrap in y and z is just a different row address, R2) -- plus one copy of the tile's flag bytes,
//     all completing on the stage's "full" mbarrier (complete_tx).  S stages are filled ahead.  A warp that has
//     its values in registers arrives on the stage's "empty" mbarrier; before issuing its share of the refill
//     (tile k+S) a warp waits for that barrier -- there is no CTA-wide barrier in the loop;
//   * the x +- 1 shift of 10 of the 19 directions is a shared-memory read at offset +- 1 element; the
//     periodic wrap in x reads the other end of the same row when the tile holds whole rows, else a 16-byte
//     halo copy per shifted direction fills the pad in front of / behind the segment;
//   * results are encoded in registers and stored directly (one aligned 32/64-bit store per direction and cell
//     pair, 128/256 contiguous bytes per warp): stores need no latency hiding, so they need no staging;
//   * cell pairs with any flag bit set (wall, equilibrium boundary, or next to a wall; lbm_set_flags marks the latter)
//     are pulled from the stage like the others and then fixed up cell by cell: fixed cells are not written, a cell
//     next to a wall replaces its bounced links from a precomputed per-cell word (bounce_links below).
// Arithmetic, operation order and codecs are those of lbm_lattice.cuh / lbm_codecs.cuh: the stored results
// are bit-identical to stream_collide_kernel's and to the oracle's.
#pragma once
#include "lbm_kernels.cuh"

namespace lbmk {

// exact n / d for 0 <= n < 2^31 as (n * M) >> sh, M = floor(2^sh / d) + 1, sh = 31 + ceil(log2 d)
struct FastDiv {
    unsigned M;
    int sh;
    __host__ static FastDiv make(int d) {
        FastDiv f;
        int s = 0;
        while ((1LL << s) < d) ++s;
        f.sh = 31 + s;
        f.M = (unsigned)((1ULL << f.sh) / (unsigned long long)d + 1ULL);
        return f;
    }
    __device__ __forceinline__ int div(int n) const { return (int)(((unsigned long long)(unsigned)n * M) >> sh); }
};

struct BulkGeom {
    int tile_w;            // cells of a full tile row: min(nx, RMAX*TX)
    int tiles_per_row;     // ceil(nx / tile_w)
    int rows_per_tile;     // RMAX*TX / nx whole rows if a row is one tile (they are contiguous in memory), else 1
    int ytiles;            // ceil(ny / rows_per_tile)
    int n_tiles;           // tiles_per_row * ytiles * nz  (< 2^31)
    FastDiv by_tpr, by_ytiles;
    FastDiv by_hw_full, by_hw_last;   // division by half the width of a full tile / of a row's last tile
    long long src_off[27]; // i*N - nx*(c_iy + ny*c_iz): source row of direction i relative to the own row, no wrap
    // the same in BYTES, and the byte offset i*N*sizeof(element) of direction i (lbm_stage.cuh: the producer warps add
    // them to a tile's base address with one uniform 64-bit add each)
    long long src_boff[27], dir_boff[27];
    int chunk_shift;       // lbm_stage.cuh: a tile has 2^chunk_shift chunk ids (>= its chunks of 32 cell pairs, >= 8)
};

// c_i of the library's numbering for a run-time direction index (copy issue only; the collision uses Lat<Q>)
static __constant__ signed char c27_table[27][3] = {{0, 0, 0},
                                             {1, 0, 0},   {-1, 0, 0},  {0, 1, 0},   {0, -1, 0},  {0, 0, 1},   {0, 0, -1},
                                             {1, 1, 0},   {-1, -1, 0}, {1, 0, 1},   {-1, 0, -1}, {0, 1, 1},   {0, -1, -1},
                                             {1, -1, 0},  {-1, 1, 0},  {1, 0, -1},  {-1, 0, 1},  {0, 1, -1},  {0, -1, 1},
                                             {1, 1, 1},   {-1, -1, -1}, {1, 1, -1}, {-1, -1, 1}, {1, -1, 1},  {-1, 1, -1},
                                             {-1, 1, 1},  {1, -1, -1}};
static __constant__ signed char d2q9_members[9] = {0, 1, 2, 3, 4, 7, 8, 13, 14};

// ---- PTX wrappers --------------------------------------------------------------------------------
__device__ __forceinline__ unsigned smem_addr(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
// the same with a suspend-time hint: a waiting thread sleeps until the phase completes (or the hint, in ns, runs out)
// instead of coming back to poll -- polling warps take issue slots from the arithmetic warps
__device__ __forceinline__ void mbar_wait_sleepy(unsigned bar, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "LBM_WAITS_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1, %2;\n"
        "@p bra LBM_DONES_%=;\n"
        "bra LBM_WAITS_%=;\n"
        "LBM_DONES_%=:\n"
        "}\n" ::"r"(bar),
        "r"(parity), "r"(0x989680u)
        : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "LBM_WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra LBM_DONE_%=;\n"
        "bra LBM_WAIT_%=;\n"
        "LBM_DONE_%=:\n"
        "}\n" ::"r"(bar),
        "r"(parity)
        : "memory");
}
// global -> shared, completes `bytes` on the mbarrier; addresses and size are multiples of 16
__device__ __forceinline__ void bulk_g2s(unsigned dst, const void *src, unsigned bytes, unsigned bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst), "l"(src),
                 "r"(bytes), "r"(bar)
                 : "memory");
}
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// ---- compile-time shape ----------------------------------------------------------------------------
template <int Q, int F, int NT>
struct BulkShape {
    typedef Elem<F> E;
    static constexpr int ES = E::SIZE;                  // bytes per stored DDF
    static constexpr int TX = 2 * NT;                   // cells per tile row
    static constexpr int PAD = 16;                      // halo pad in front of and behind every segment
    static constexpr int MAXB = (227 * 1024 - 2048) / 2;                    // two CTAs per SM
    static constexpr int TABB = PairCodec<F>::TABLE ? 512 * 16 : 0;        // the format's encoder table
    // a stage holds up to RMAX*TX cells of every direction -- several whole rows (contiguous in memory) or one segment
    // of a long row -- between one pair of pads, plus their flag bytes
    static constexpr int stage_bytes(int r) { return Q * (r * TX * ES + 2 * PAD) + r * TX; }
    static constexpr int RMAX = 2 * stage_bytes(4) + TABB <= MAXB ? 4 : 2 * stage_bytes(2) + TABB <= MAXB ? 2 : 1;
    static constexpr int ROWB = RMAX * TX * ES + 2 * PAD;                   // one direction of one stage
    static constexpr int STAGEB = stage_bytes(RMAX);
    static constexpr int S = 3 * STAGEB + TABB <= MAXB ? 3 : 2;             // input stages
    static constexpr int TAB_OFF = S * STAGEB;
    static constexpr int BAR_OFF = TAB_OFF + TABB;
    static constexpr int SMEM = BAR_OFF + 2 * S * 8;                        // full[S], empty[S]
    static constexpr int HALO_ELEMS = PAD / ES;                             // elements in one 16-byte halo copy
    static_assert(2 * STAGEB + TABB <= MAXB, "two stages of two CTAs must fit one SM");
    static_assert(STAGEB % 16 == 0 && ROWB % 16 == 0, "bulk copies need 16-byte alignment");
};

// decode policy of the full-range posit decoders: PairCodec<F>::Full, recording the codes it sees like PairCodec<F>
template <int F>
struct FullRange : PairCodec<F>::Full {
    static constexpr unsigned CHECK = PairCodec<F>::CHECK;
};

// shared-memory access (addresses are "thread base + immediate")
__device__ __forceinline__ unsigned lds_u32(const char *p) { return *reinterpret_cast<const unsigned *>(p); }
__device__ __forceinline__ int lds_s16(const char *p) { return (int)*reinterpret_cast<const short *>(p); }
__device__ __forceinline__ float lds_f32(const char *p) { return *reinterpret_cast<const float *>(p); }

// the two values of direction I for the thread's cells xl, xl+1, from the staged segment.
//   own  = address of element xl of direction 0's segment; left = element "xl - 1", right = element "xl + 2"
//   (already wrapped / pointing into the pads); direction I adds the immediate I * ROWB.
template <int Q, int F, int NT, class PC, int I>
struct PullStaged {
    typedef BulkShape<Q, F, NT> SH;
    // acc collects the raw words (pairs in both halves, single codes in the low half) for PairCodec<F>::CHECK
    static __device__ __forceinline__ void run(const char *own, const char *left, const char *right, float (&f)[2][Q],
                                               unsigned &acc) {
        typedef Lat<Q> L;
        constexpr int cx = L::c(I, 0);
        constexpr int o = I * SH::ROWB;
        if constexpr (SH::ES == 4) {
            if (cx == 0) {
                const float2 v = *reinterpret_cast<const float2 *>(own + o);
                f[0][I] = v.x;
                f[1][I] = v.y;
            } else if (cx > 0) {              // sources xl-1, xl
                f[0][I] = lds_f32(left + o);
                f[1][I] = lds_f32(own + o);
            } else {                          // sources xl+1, xl+2
                f[0][I] = lds_f32(own + o + 4);
                f[1][I] = lds_f32(right + o);
            }
        } else {
            if (cx == 0) {
                const unsigned w = lds_u32(own + o);
                if (PC::CHECK) acc |= w;
                PC::dec2(w, f[0][I], f[1][I]);
            } else {
                const int c0 = lds_s16(cx > 0 ? left + o : own + o + 2);
                const int c1 = lds_s16(cx > 0 ? own + o : right + o);
                if (PC::CHECK) acc |= (unsigned)(c0 | c1) & 0xFFFFu;
                f[0][I] = PC::dec1(c0);
                f[1][I] = PC::dec1(c1);
            }
        }
        PullStaged<Q, F, NT, PC, I + 1>::run(own, left, right, f, acc);
    }
};
template <int Q, int F, int NT, class PC>
struct PullStaged<Q, F, NT, PC, Q> {
    static __device__ __forceinline__ void run(const char *, const char *, const char *, float (&)[2][Q], unsigned &) {}
};

struct TileCoord {
    int y, z, x0, w, rows;   // first row, plane, first cell, cells per row (multiple of 16), rows of a tile
    bool last;               // the last (possibly narrower) tile of its row
};
__device__ __forceinline__ TileCoord tile_coord(int t, const BulkGeom &g, const Params &p) {
    TileCoord c;
    const int rt = g.by_tpr.div(t), xt = t - rt * g.tiles_per_row;
    c.z = g.by_ytiles.div(rt);
    c.y = (rt - c.z * g.ytiles) * g.rows_per_tile;
    c.rows = min(g.rows_per_tile, p.ny - c.y);
    c.x0 = xt * g.tile_w;
    c.w = min(g.tile_w, p.nx - c.x0);
    c.last = xt == g.tiles_per_row - 1;
    return c;
}

// This warp's share of the copies of tile t into one stage: directions i = warp, warp + NW, ... (i = Q: the flag
// bytes).  The direction index is warp-uniform; lane 0 issues.
template <int Q, int F, int NT>
__device__ __forceinline__ void issue_tile_loads(const typename Elem<F>::T *__restrict__ A, const Params &p, const BulkGeom &g,
                                                 int t, unsigned stage, unsigned full, int warp, int lane) {
    typedef BulkShape<Q, F, NT> SH;
    typedef typename Elem<F>::T T;
    constexpr int ES = SH::ES, TX = SH::TX, NW = NT / 32;
    constexpr int n_shift = (Q == 9 ? 6 : Q == 19 ? 10 : 18);               // directions with c_x != 0
    if (lane != 0) return;
    const bool single = g.tiles_per_row == 1;
    const TileCoord c = tile_coord(t, g, p);
    const int cells = c.rows * c.w;
    // single: the rows of the tile are one contiguous segment per direction; else the tile is part of one row and
    // the shifted directions get a 16-byte halo copy
    const int pitch = c.w * ES;
    if (warp == 0)
        mbar_arrive_expect_tx(full, (unsigned)(Q * cells * ES + cells + (single ? 0 : c.rows * n_shift * SH::PAD)));
    const long long own = (long long)p.nx * (c.y + (long long)p.ny * c.z);
    // tiles on a y or z face of the box pull some directions from the opposite face (R2): rare, row by row
    const bool face = c.y == 0 || c.y + c.rows == p.ny || c.z == 0 || c.z == p.nz - 1;
#pragma unroll 1
    for (int i = warp; i <= Q; i += NW) {
        if (i == Q) {                                                       // flag bytes, rows packed at pitch w
            if (single) bulk_g2s(stage + Q * SH::ROWB, p.flags + own, (unsigned)cells, full);
            else
                for (int r = 0; r < c.rows; ++r)
                    bulk_g2s(stage + Q * SH::ROWB + r * c.w, p.flags + own + (long long)r * p.nx + c.x0, (unsigned)c.w, full);
            break;
        }
        const int m = Q == 9 ? d2q9_members[i] : i;
        const int cx = c27_table[m][0];
        const unsigned dst = stage + i * SH::ROWB + SH::PAD;
        if (single && !face) {
            bulk_g2s(dst, A + own + g.src_off[i], (unsigned)(cells * ES), full);
            continue;
        }
        const int cy = c27_table[m][1], cz = c27_table[m][2];
        int zs = c.z - cz;
        zs = zs < 0 ? p.nz - 1 : zs >= p.nz ? 0 : zs;
#pragma unroll 1
        for (int r = 0; r < c.rows; ++r) {
            int ys = c.y + r - cy;
            ys = ys < 0 ? p.ny - 1 : ys >= p.ny ? 0 : ys;
            const T *src_row = A + (long long)i * p.N + (long long)p.nx * (ys + (long long)p.ny * zs);
            const unsigned d = dst + r * pitch;
            bulk_g2s(d, src_row + c.x0, (unsigned)(c.w * ES), full);
            if (!single && cx != 0) {
                if (cx > 0) {                                               // element x0 - 1: the chunk before x0
                    const int xs = (c.x0 == 0 ? p.nx : c.x0) - SH::HALO_ELEMS;
                    bulk_g2s(d - SH::PAD, src_row + xs, SH::PAD, full);
                } else {                                                    // element x0 + w: the chunk after the tile
                    const int xs = c.x0 + c.w == p.nx ? 0 : c.x0 + c.w;
                    bulk_g2s(d + c.w * ES, src_row + xs, SH::PAD, full);
                }
            }
        }
    }
}

// x 2^SC, exact (the staged kernel keeps FP16S / P16_0S values scaled, collide_bgk<.., SC>)
template <int SC>
__device__ __forceinline__ float scaled(float v) { return SC == 0 ? v : mul(v, pow2f(SC)); }

// Halfway bounce-back for one cell next to a wall (R3; moving wall R9).  f holds the q
// directions pulled as if every source were fluid; the links whose source is a wall cell -- one precomputed word per
// cell, written by lbm_set_flags -- are replaced by the cell's own opposite population, all loads independent of
// one another.  Wall velocities are loaded only for cells one of whose walls moves (bit 31, set by lbm_init).
// f is in the kernel's 2^SC scaling; the bounced values and the moving-wall term (evaluated as R9 states) are
// scaled exactly.
template <int Q, int F, int SC>
__device__ __forceinline__ void bounce_links(const typename Elem<F>::T *__restrict__ A, const Params &p, long long n, int x, int y,
                                             int z, unsigned m, float (&f)[Q]) {
    typedef Lat<Q> L;
    typedef Elem<F> E;
#pragma unroll
    for (int i = 1; i < Q; ++i)
        if ((m >> i) & 1u) f[i] = scaled<SC>(E::ld1(A + (long long)L::opp(i) * p.N + n));
    if (!(m >> 31)) return;
#pragma unroll
    for (int i = 1; i < Q; ++i) {                                               // static indices: f stays in registers
        if (!((m >> i) & 1u)) continue;
        int xs = x - L::c(i, 0), ys = y - L::c(i, 1), zs = z - L::c(i, 2);
        xs = xs < 0 ? p.nx - 1 : xs >= p.nx ? 0 : xs;
        ys = ys < 0 ? p.ny - 1 : ys >= p.ny ? 0 : ys;
        zs = zs < 0 ? p.nz - 1 : zs >= p.nz ? 0 : zs;
        const long long src = xs + (long long)p.nx * (ys + (long long)p.ny * zs);
        const float v[3] = {__ldg(p.u0 + src), __ldg(p.u0 + p.N + src), __ldg(p.u0 + 2 * p.N + src)};
        if (v[0] != 0.0f || v[1] != 0.0f || v[2] != 0.0f) {                     // rho_w = 1; a resting wall adds nothing
            float sdot = 0.0f;                                                  // c_i . u_w as cdot<Q, i> of lbm_lattice.cuh
            bool first = true;
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                if (L::c(i, a) == 0) continue;
                const float term = L::c(i, a) > 0 ? v[a] : -v[a];
                sdot = first ? term : add(sdot, term);
                first = false;
            }
            f[i] = add(f[i], scaled<SC>(mul(L::w6(i), sdot)));
        }
    }
}

template <int Q, int F, int NT, bool FORCE, int COLL = 0>
__global__ void __launch_bounds__(NT, 2)
stream_collide_bulk_kernel(const typename Elem<F>::T *__restrict__ A, typename Elem<F>::T *__restrict__ B, const Params p,
                           const BulkGeom g, const EncEntry *__restrict__ enc_table) {
    typedef BulkShape<Q, F, NT> SH;
    typedef Elem<F> E;
    typedef typename E::T T;
    constexpr int ES = SH::ES, TX = SH::TX, S = SH::S, NW = NT / 32;
    typedef PairCodec<F> PC;
    constexpr int SC = PC::SC;

    extern __shared__ __align__(128) char smem[];
    const unsigned smem_base = smem_addr(smem);
    const unsigned bar_full = smem_base + SH::BAR_OFF, bar_empty = bar_full + S * 8;
    const int tid = threadIdx.x, lane = tid & 31;
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);                  // warp-uniform by construction

    if (tid == 0) {
        for (int s = 0; s < S; ++s) {
            mbar_init(bar_full + s * 8, 1);                                  // warp 0's arrive.expect_tx
            mbar_init(bar_empty + s * 8, NW);                                // one arrival per warp
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        fence_async_smem();
    }
    const EncEntry *tab = reinterpret_cast<const EncEntry *>(smem + SH::TAB_OFF);
    if constexpr (PC::TABLE) {
        for (int i = tid; i < 512; i += NT)
            reinterpret_cast<uint4 *>(smem + SH::TAB_OFF)[i] = __ldg(reinterpret_cast<const uint4 *>(enc_table) + i);
    }
    __syncthreads();

    const bool single = g.tiles_per_row == 1;            // a tile spans its rows: x wraps inside the segment
    const int stride = gridDim.x;

#pragma unroll 1
    for (int s = 0; s < S; ++s) {                                            // prologue: fill every stage
        const long long t = (long long)blockIdx.x + (long long)s * stride;
        if (t < g.n_tiles) issue_tile_loads<Q, F, NT>(A, p, g, (int)t, smem_base + s * SH::STAGEB, bar_full + s * 8, warp, lane);
    }

    bool full_mode = false;                              // posits: this thread currently needs the full-range decoders
    int k = 0;
    for (int t = blockIdx.x; t < g.n_tiles; t += stride, ++k) {
        const int s = k % S;
        const unsigned ph = (unsigned)(k / S) & 1u;
        const TileCoord c = tile_coord(t, g, p);
        const int w = c.w, hw = w >> 1;
        const char *stage = smem + s * SH::STAGEB;
        const int pitch = w * ES;
        const int pairs = c.rows * hw;                                          // cell pairs of the tile
        const FastDiv by_hw = c.last ? g.by_hw_last : g.by_hw_full;

        mbar_wait(bar_full + s * 8, ph);
#pragma unroll 1
        // the pairs of a tile rotate through the warps from tile to tile: a pair that is always slow (row ends next to
        // walls) does not always burden the same warp
        const int tidr = (tid + 32 * (k % NW)) & (NT - 1);
        for (int it = 0, fp = tidr; it * NT < pairs; ++it, fp += NT) {          // same trip count for every thread
            const bool active = fp < pairs;
            const int r = hw == NT ? it : by_hw.div(fp);                        // row of the tile holding this cell pair
            const int xl = 2 * (fp - r * hw);
            const int el = xl - 1 + ((single && xl == 0) ? w : 0);              // element "xl - 1" of the row
            const int er = xl + 2 - ((single && xl + 2 == w) ? w : 0);          // element "xl + 2" of the row
            const int y = c.y + r, z = c.z;
            const long long own = (long long)p.nx * (y + (long long)p.ny * z) + c.x0 + xl;   // the thread's first cell
            unsigned fl = 0;
            if (active) fl = *reinterpret_cast<const unsigned short *>(stage + Q * SH::ROWB + r * w + xl);
            const bool fast = active && fl == 0;
            // near-wall cells: which links bounce (one word per cell, lbm_set_flags); loaded now, needed after the pull
            unsigned bm[2] = {0u, 0u};
            if (fl & FLAG_NEAR) bm[0] = __ldg(p.bounce + own);
            if (fl & (FLAG_NEAR << 8)) bm[1] = __ldg(p.bounce + own + 1);
            float f[2][Q];
            unsigned acc = 0;
            const char *base = stage + SH::PAD + r * pitch;
            bool warp_full = false;
            if constexpr (PC::CHECK != 0) warp_full = __any_sync(0xffffffffu, full_mode);   // one decoder per warp where possible
            if (active) {                                   // every direction from the stage, as if no wall were near
                if constexpr (PC::CHECK != 0) {
                    // posits: the cheap decoders cover a regime of zeros (|f| < 2^-7).  A thread that met other codes
                    // makes its warp pull with the full-range decoders until its pairs are free of such codes again
                    // (flows are smooth: the choice rarely changes from one pair to the next)
                    if (!warp_full) PullStaged<Q, F, NT, PC, 0>::run(base + xl * ES, base + el * ES, base + er * ES, f, acc);
                    if (warp_full || ((acc | (acc >> 16)) & PC::CHECK) != 0) {
                        acc = 0;
                        PullStaged<Q, F, NT, FullRange<F>, 0>::run(base + xl * ES, base + el * ES, base + er * ES, f, acc);
                    }
                    full_mode = ((acc | (acc >> 16)) & PC::CHECK) != 0;
                } else {
                    PullStaged<Q, F, NT, PC, 0>::run(base + xl * ES, base + el * ES, base + er * ES, f, acc);
                }
            }
            const bool slow = active && fl != 0;            // a fixed cell or a wall among the pull sources (below)
            if ((it + 1) * NT >= pairs) {                                       // last trip: the warp has its values in registers,
                __syncwarp();                                                   // the stage may be refilled
                if (lane == 0) mbar_arrive(bar_empty + s * 8);
            }
            if (slow) {
                // f holds every direction pulled from the stage as if there were no wall: a cell next to a wall replaces
                // its bounced links (R3, R9), all loads of both cells in flight together
#pragma unroll
                for (int j = 0; j < 2; ++j)
                    if (bm[j]) bounce_links<Q, F, SC>(A, p, own + j, c.x0 + xl + j, y, z, bm[j], f[j]);
            }
            if (active) {
                // one instruction stream for plain and flagged pairs (a fixed cell's values are computed and dropped)
                collide<COLL, Q, FORCE, SC>(f[0], p);
                collide<COLL, Q, FORCE, SC>(f[1], p);
                T *o = B + own;
                if (!slow) {
#pragma unroll
                    for (int i = 0; i < Q; ++i) {
                        if constexpr (ES == 4) *reinterpret_cast<float2 *>(o + (long long)i * p.N) = make_float2(f[0][i], f[1][i]);
                        else *reinterpret_cast<unsigned *>(o + (long long)i * p.N) = PC::enc2(f[0][i], f[1][i], tab);
                    }
                } else {
                    // fixed cells (wall, equilibrium boundary) are not written: PAPER.md:1017; R15
#pragma unroll
                    for (int j = 0; j < 2; ++j) {
                        if ((fl >> (8 * j)) & FLAG_FIXED) continue;
#pragma unroll
                        for (int i = 0; i < Q; ++i) {
                            if constexpr (ES == 4) o[(long long)i * p.N + j] = f[j][i];
                            else o[(long long)i * p.N + j] = (T)PC::enc1(f[j][i], tab);
                        }
                    }
                }
            }
        }
        // refill the stage just consumed with tile k+S, once every warp has taken its values out of it
        const long long tn = (long long)t + (long long)S * stride;
        if (tn < g.n_tiles) {
            mbar_wait(bar_empty + s * 8, ph);
            issue_tile_loads<Q, F, NT>(A, p, g, (int)tn, smem_base + s * SH::STAGEB, bar_full + s * 8, warp, lane);
        }
    }
}

}  // namespace lbmk
