// lbm_unit.cu -- one (velocity set, storage format) instantiation unit of the kernels in
// lbm_kernels.cuh.  Compiled once per pair with -DLBM_Q=<9|19|27> -DLBM_F=<0..6> (see build.py).
#include "lbm_internal.h"
#include "lbm_kernels.cuh"
#include "lbm_bulk.cuh"
#include "lbm_stage.cuh"

#include <mutex>

#ifndef LBM_Q
#error "compile with -DLBM_Q=<velocity set> -DLBM_F=<format>"
#endif

#define LBM_CAT_(a, b, c, d) a##b##c##d
#define LBM_CAT(a, b, c, d) LBM_CAT_(a, b, c, d)
#define LBM_UNIT_SYMBOL LBM_CAT(lbm_unit_q, LBM_Q, _f, LBM_F)
#define LBM_STR_(x) #x
#define LBM_STR(x) LBM_STR_(x)

namespace lbmk {
namespace {

constexpr int Q = LBM_Q, F = LBM_F;
typedef typename Elem<F>::T T;

template <int V, bool FORCE, int COLL = 0, bool SHIFT = true>
cudaError_t launch_sc(const void *A, void *B, const Params &p, cudaStream_t st) {
    const int tx = (p.nx + V - 1) / V;
    int bx = 1;
    while (bx < tx && bx < SC_THREADS) bx <<= 1;
    const int by = SC_THREADS / bx;
    const dim3 block(bx, by, 1);
    const dim3 grid((tx + bx - 1) / bx, (p.ny + by - 1) / by, p.nz);
    stream_collide_kernel<Q, F, V, FORCE, COLL, SHIFT><<<grid, block, 0, st>>>((const T *)A, (T *)B, p);
    count_launch();
    return cudaGetLastError();
}


// Resident CTAs of a persistent kernel on the CURRENT device (SMs x CTAs per SM), and the opt-in to its dynamic shared
// memory.  Both are per-device state: resolved once per device and kernel, under a lock.  `cache` is the calling
// launcher's own table (one per kernel instantiation).
struct CtaCache {
    std::mutex mu;
    int ctas[64] = {};
};
template <class K>
cudaError_t resident_ctas(K kern, int threads, int smem, int *out, CtaCache &cache) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(cache.mu);
    if (cache.ctas[dev] == 0) {
        if ((e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem)) != cudaSuccess) return e;
        int sms = 0, per_sm = 0;
        if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
        if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, threads, smem)) != cudaSuccess) return e;
        if (per_sm < 1) return cudaErrorLaunchOutOfResources;
        cache.ctas[dev] = sms * per_sm;
    }
    *out = cache.ctas[dev];
    return cudaSuccess;
}

// ---- the warp-specialised staged variant (lbm_stage.cuh) ----------------------------------------------
template <int ALT>
BulkGeom stage_geom_of(const Params &p, long long *tiles) {
    typedef StageShape<Q, F, ALT> SH;
    BulkGeom g;
    // a row longer than a tile is cut into EQUAL pieces (multiples of 16 cells; the last one may be shorter): 1280 cells
    // are 2 x 640, not 1024 + 256 -- a short tile costs the same per-tile work and leaves the stages half empty
    g.tiles_per_row = (p.nx + SH::TC - 1) / SH::TC;
    g.tile_w = p.nx <= SH::TC ? p.nx : ((p.nx + g.tiles_per_row - 1) / g.tiles_per_row + 15) / 16 * 16;
    g.rows_per_tile = g.tiles_per_row == 1 ? SH::TC / p.nx : 1;
    const int w_last = p.nx - (g.tiles_per_row - 1) * g.tile_w;
    g.by_hw_full = FastDiv::make(g.tile_w / 2);
    g.by_hw_last = FastDiv::make(w_last / 2);
    g.ytiles = (p.ny + g.rows_per_tile - 1) / g.rows_per_tile;
    *tiles = (long long)g.tiles_per_row * g.ytiles * p.nz;
    g.n_tiles = (int)(*tiles < 0x7FFFFFFFLL ? *tiles : 0x7FFFFFFFLL);
    g.by_tpr = FastDiv::make(g.tiles_per_row);
    g.by_ytiles = FastDiv::make(g.ytiles);
    for (int i = 0; i < 27; ++i) {
        g.src_boff[i] = i < Q ? ((long long)i * p.N - (long long)p.nx * (Lat<Q>::c(i, 1) + (long long)p.ny * Lat<Q>::c(i, 2))) * SH::ES : 0;
        g.dir_boff[i] = i < Q ? (long long)i * p.N * SH::ES : 0;
    }
    const int chunks_full = (g.rows_per_tile * (g.tile_w / 2) + 31) / 32;
    g.chunk_shift = 3;
    while ((1 << g.chunk_shift) < chunks_full) ++g.chunk_shift;
    return g;
}

// Which of the two compiled tile shapes (StageShape::HAS_ALT) a box runs with: the three-stage shape, unless the box's
// rows fill its smaller tile so badly that the two-stage shape's tiles hold at least 1.5 times the cells.  Measured, D3Q27
// FP16S cubes, fraction of the HBM roofline with the 768 x 3 | 1024 x 2 shape: 256^3 (768 | 1024 cells per tile) 0.85 |
// 0.75, 320^3 (640 | 960) 0.77 | 0.77, 384^3 (768 | 768) 0.86 | 0.73, 448^3 (448 | 896) 0.62 | 0.79, 512^3 (512 | 1024)
// 0.70 | 0.79.  One rule for the kernel launch and for the per-tile lists.
bool stage_alt(const Params &p) {
    if (!StageShape<Q, F, 0>::HAS_ALT) return false;
    long long t0 = 0, t1 = 0;
    const BulkGeom g0 = stage_geom_of<0>(p, &t0), g1 = stage_geom_of<1>(p, &t1);
    return 2LL * g1.rows_per_tile * g1.tile_w >= 3LL * g0.rows_per_tile * g0.tile_w;
}
BulkGeom stage_geom(const Params &p, long long *tiles) { return stage_alt(p) ? stage_geom_of<1>(p, tiles) : stage_geom_of<0>(p, tiles); }

template <bool FORCE, int COLL, int ALT>
cudaError_t launch_staged_shape(const void *A, void *B, const Params &p, cudaStream_t st) {
    typedef StageShape<Q, F, ALT> SH;
    auto kern = stream_collide_staged_kernel<Q, F, FORCE, COLL, ALT>;
    static CtaCache cache;
    int ctas = 0;
    if (cudaError_t e = resident_ctas(kern, SH::NT, SH::SMEM, &ctas, cache)) return e;
    long long tiles = 0;
    const BulkGeom g = stage_geom_of<ALT>(p, &tiles);
    if (p.nx % 16 != 0 || tiles >= 0x7FFFFFFFLL) return cudaErrorInvalidValue;
    const int grid = (int)(tiles < ctas ? tiles : ctas);
    const EncEntry *tab = nullptr;
    if (PairCodec<F>::TABLE) {
        cudaError_t e = enc_table(F, &tab, st);
        if (e != cudaSuccess) return e;
    }
    kern<<<grid, SH::NT, SH::SMEM, st>>>((const T *)A, (T *)B, p, g, tab);
    count_launch();
    return cudaGetLastError();
}
template <bool FORCE, int COLL = 0>
cudaError_t launch_staged(const void *A, void *B, const Params &p, cudaStream_t st) {
    if constexpr (StageShape<Q, F, 0>::HAS_ALT) {
        if (stage_alt(p)) return launch_staged_shape<FORCE, COLL, 1>(A, B, p, st);
    }
    return launch_staged_shape<FORCE, COLL, 0>(A, B, p, st);
}

// Per-tile lists of flagged cell pairs for this unit's tile geometry (lbm_aux.cu)
cudaError_t build_fix_lists(const Params &p, unsigned **off_out, uint2 **list_out, cudaStream_t st) {
    long long tiles = 0;
    const BulkGeom g = stage_geom(p, &tiles);
    if (p.nx % 16 != 0 || tiles >= 0x7FFFFFFFLL) return cudaErrorInvalidValue;
    return build_fix_lists_for(p, g, off_out, list_out, st);
}

cudaError_t stream_collide(const void *A, void *B, const Params &p_in, int V, int coll, bool force, cudaStream_t st) {
    Params p = p_in;
    if (force) guo_constants<Q>(p);                          // R10's per-direction constants (lbm_lattice.cuh)
    if (!p.shifted) {
        // R17, the paper's negative control (eqs (19)-(23)): the per-thread kernel, one cell per thread
        if (coll == 1) return force ? launch_sc<1, true, 1, false>(A, B, p, st) : launch_sc<1, false, 1, false>(A, B, p, st);
        return force ? launch_sc<1, true, 0, false>(A, B, p, st) : launch_sc<1, false, 0, false>(A, B, p, st);
    }
    if (V == VARIANT_STAGED) {
        if (coll == 1) return force ? launch_staged<true, 1>(A, B, p, st) : launch_staged<false, 1>(A, B, p, st);
        return force ? launch_staged<true>(A, B, p, st) : launch_staged<false>(A, B, p, st);
    }
    if (coll == 1) {
        // TRT (R13): the staged kernel, or the per-thread kernel with one, two or four cells per thread
        if (V == 4 && p.nx % 4 == 0) return force ? launch_sc<4, true, 1>(A, B, p, st) : launch_sc<4, false, 1>(A, B, p, st);
        if (V >= 2 && p.nx % 2 == 0) return force ? launch_sc<2, true, 1>(A, B, p, st) : launch_sc<2, false, 1>(A, B, p, st);
        return force ? launch_sc<1, true, 1>(A, B, p, st) : launch_sc<1, false, 1>(A, B, p, st);
    }
    switch (V * 2 + (force ? 1 : 0)) {
        case 2: return launch_sc<1, false>(A, B, p, st);
        case 3: return launch_sc<1, true>(A, B, p, st);
        case 4: return launch_sc<2, false>(A, B, p, st);
        case 5: return launch_sc<2, true>(A, B, p, st);
        case 8: return launch_sc<4, false>(A, B, p, st);
        case 9: return launch_sc<4, true>(A, B, p, st);
    }
    return cudaErrorInvalidValue;
}

int blocks_for(long long N) {
    long long b = (N + 255) / 256;
    const long long cap = 148LL * 64;   // grid-stride loops: a few waves over the 148 SMs
    return (int)(b < cap ? (b < 1 ? 1 : b) : cap);
}

cudaError_t init(void *A, void *B, const float *rho, const float *u, long long N, bool shifted, cudaStream_t st) {
    if (shifted) init_kernel<Q, F, true><<<blocks_for(N), 256, 0, st>>>((T *)A, (T *)B, rho, u, N);
    else init_kernel<Q, F, false><<<blocks_for(N), 256, 0, st>>>((T *)A, (T *)B, rho, u, N);
    count_launch();
    return cudaGetLastError();
}

cudaError_t init_generated(void *A, void *B, long long N, unsigned long long seed, cudaStream_t st) {
    init_generated_kernel<Q, F><<<blocks_for(N), 256, 0, st>>>((T *)A, (T *)B, N, seed);
    count_launch();
    return cudaGetLastError();
}

cudaError_t read(const void *A, const Params &p, bool force, float *rho, float *u, cudaStream_t st) {
    if (!p.shifted) {
        if (force) read_rho_u_kernel<Q, F, true, false><<<blocks_for(p.N), 256, 0, st>>>((const T *)A, p, rho, u);
        else read_rho_u_kernel<Q, F, false, false><<<blocks_for(p.N), 256, 0, st>>>((const T *)A, p, rho, u);
    } else if (force) read_rho_u_kernel<Q, F, true><<<blocks_for(p.N), 256, 0, st>>>((const T *)A, p, rho, u);
    else read_rho_u_kernel<Q, F, false><<<blocks_for(p.N), 256, 0, st>>>((const T *)A, p, rho, u);
    count_launch();
    return cudaGetLastError();
}

cudaError_t probe(const void *A, const Params &p, bool force, const long long *cells, int count, float *rho, float *u, cudaStream_t st) {
    const int blocks = (count + 127) / 128;
    if (!p.shifted) {
        if (force) probe_rho_u_kernel<Q, F, true, false><<<blocks, 128, 0, st>>>((const T *)A, p, cells, count, rho, u);
        else probe_rho_u_kernel<Q, F, false, false><<<blocks, 128, 0, st>>>((const T *)A, p, cells, count, rho, u);
    } else if (force) probe_rho_u_kernel<Q, F, true><<<blocks, 128, 0, st>>>((const T *)A, p, cells, count, rho, u);
    else probe_rho_u_kernel<Q, F, false><<<blocks, 128, 0, st>>>((const T *)A, p, cells, count, rho, u);
    count_launch();
    return cudaGetLastError();
}

const char *name(int V, int coll, bool force) {
    // (the unshifted control, Params::shifted == 0, always runs stream_collide_kernel<V=1,...,SHIFT=0>)
#define LBM_KNAME(kernel, extra) kernel "<Q=" LBM_STR(LBM_Q) ",F=" LBM_STR(LBM_F) extra ">"
    if (V == VARIANT_STAGED) {
        if (coll == 1) return force ? LBM_KNAME("stream_collide_staged_kernel", ",FORCE=1,COLL=TRT") : LBM_KNAME("stream_collide_staged_kernel", ",FORCE=0,COLL=TRT");
        return force ? LBM_KNAME("stream_collide_staged_kernel", ",FORCE=1") : LBM_KNAME("stream_collide_staged_kernel", ",FORCE=0");
    }
    if (coll == 1) {
        if (V == 4) return force ? LBM_KNAME("stream_collide_kernel", ",V=4,FORCE=1,COLL=TRT") : LBM_KNAME("stream_collide_kernel", ",V=4,FORCE=0,COLL=TRT");
        if (V >= 2) return force ? LBM_KNAME("stream_collide_kernel", ",V=2,FORCE=1,COLL=TRT") : LBM_KNAME("stream_collide_kernel", ",V=2,FORCE=0,COLL=TRT");
        return force ? LBM_KNAME("stream_collide_kernel", ",V=1,FORCE=1,COLL=TRT") : LBM_KNAME("stream_collide_kernel", ",V=1,FORCE=0,COLL=TRT");
    }
    if (V == 4) return force ? LBM_KNAME("stream_collide_kernel", ",V=4,FORCE=1") : LBM_KNAME("stream_collide_kernel", ",V=4,FORCE=0");
    if (V == 2) return force ? LBM_KNAME("stream_collide_kernel", ",V=2,FORCE=1") : LBM_KNAME("stream_collide_kernel", ",V=2,FORCE=0");
    return force ? LBM_KNAME("stream_collide_kernel", ",V=1,FORCE=1") : LBM_KNAME("stream_collide_kernel", ",V=1,FORCE=0");
#undef LBM_KNAME
}

int staged_tile_cells() { return StageShape<Q, F, 0>::TC; }       // (the smaller of the two shapes' tiles: the tile-count bound of pick_variant)

}  // namespace

extern const UnitOps LBM_UNIT_SYMBOL;
const UnitOps LBM_UNIT_SYMBOL = {stream_collide, init, read, name, probe, nullptr, staged_tile_cells, build_fix_lists, init_generated};

}  // namespace lbmk
