// lbm_bulk.cuh -- building blocks of the shared-memory-staged stream-collide kernel (lbm_stage.cuh): the tile geometry
// (a tile = a run of consecutive cells: whole rows of a z-plane, or a segment of a long row), exact division by
// multiplication for tile -> (row, plane), and the PTX wrappers for mbarriers and cp.async.bulk (SASS UBLKCP).
//
// In a structure-of-arrays pull step every direction of a row of cells is ONE contiguous segment of ONE source row
// (eq (24)), so a tile needs q plain 1-D copies in and q out; once the segments sit in shared memory
// every address is "thread base + compile-time immediate".
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
    int tile_w;            // cells of a full tile row: min(nx, TC)
    int tiles_per_row;     // ceil(nx / tile_w)
    int rows_per_tile;     // TC / nx whole rows if a row is one tile (they are contiguous in memory), else 1
    int ytiles;            // ceil(ny / rows_per_tile)
    int n_tiles;           // tiles_per_row * ytiles * nz  (< 2^31)
    FastDiv by_tpr, by_ytiles;
    FastDiv by_hw_full, by_hw_last;   // division by half the width of a full tile / of a row's last tile
    // per direction i, in BYTES: src_boff = (i*N - nx*(c_iy + ny*c_iz)) * sizeof(element), the source row of direction i
    // relative to the own row (no wrap); dir_boff = i*N*sizeof(element).  The loader / storer warps add them to a tile's
    // base address with one uniform 64-bit add each (they sit in the kernel's constant bank).
    long long src_boff[27], dir_boff[27];
    int chunk_shift;       // a tile has 2^chunk_shift chunk ids (>= its chunks of 32 cell pairs, >= 8)
};

// c_i of the library's numbering for a run-time direction index (the collision uses Lat<Q>)
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
__device__ __forceinline__ void mbar_arrive_n(unsigned bar, unsigned count) {          // `count` arrivals at once
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(count) : "memory");
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

// decode policy of the full-range posit decoders: PairCodec<F>::Full, recording the codes it sees like PairCodec<F>
template <int F>
struct FullRange : PairCodec<F>::Full {
    static constexpr unsigned CHECK = PairCodec<F>::CHECK;
    static constexpr bool SEXT = PairCodec<F>::SEXT;     // (PositFull uses the low 16 bits only: either load will do)
};

// shared-memory access (addresses are "thread base + immediate")
__device__ __forceinline__ unsigned lds_u32(const char *p) { return *reinterpret_cast<const unsigned *>(p); }
__device__ __forceinline__ int lds_s16(const char *p) { return (int)*reinterpret_cast<const short *>(p); }
__device__ __forceinline__ int lds_u16(const char *p) { return (int)*reinterpret_cast<const unsigned short *>(p); }
__device__ __forceinline__ float lds_f32(const char *p) { return *reinterpret_cast<const float *>(p); }

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

}  // namespace lbmk
