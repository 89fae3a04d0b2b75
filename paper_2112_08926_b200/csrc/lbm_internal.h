// lbm_internal.h -- host-side glue between the C ABI (lbm_api.cu) and the kernel translation units.
// One translation unit per (velocity set, storage format) pair is compiled from lbm_unit.cu with
// -DLBM_Q=<q> -DLBM_F=<fmt> (lbm_unit64.cu for the FP64-arithmetic formats 7 and 8); each exports the launchers
// below under a suffixed name.
#pragma once
#include <cuda_runtime.h>

#include "lbm_lattice.cuh"

namespace lbmk {

constexpr int VARIANT_STAGED = 32;    // LBM_VARIANT_STAGED of include/lbm.h

struct UnitOps {
    // stream_collide: V = cells per thread (1, 2 or 4; nx % V == 0) of the per-thread kernel, or VARIANT_STAGED
    // = the shared-memory-staged kernel (nx % 16 == 0); force = Guo term compiled in
    cudaError_t (*stream_collide)(const void *A, void *B, const Params &p, int V, int coll, bool force, cudaStream_t st);
    cudaError_t (*init)(void *A, void *B, const float *rho, const float *u, long long N, bool shifted, cudaStream_t st);
    cudaError_t (*read)(const void *A, const Params &p, bool force, float *rho, float *u, cudaStream_t st);
    const char *(*name)(int V, int coll, bool force);
    cudaError_t (*probe)(const void *A, const Params &p, bool force, const long long *cells, int count, float *rho, float *u,
                         cudaStream_t st);
    // FP64-arithmetic units only (lbm_unit64.cu), else null: read-out in double
    cudaError_t (*read64)(const void *A, const Params &p, bool force, double *rho, double *u, cudaStream_t st);
    // warp-specialised staged kernel (lbm_stage.cuh; null in the FP64-arithmetic units): cells per tile, and the
    // builder of the per-tile flagged-pair lists (Params::fix_off / fix_cells; the caller cudaFrees both)
    int (*staged_tile_cells)();
    cudaError_t (*build_fix_lists)(const Params &p, unsigned **off, uint2 **list, cudaStream_t st);
    // init from the counter-based generator of lbm_kernels.cuh (null in the FP64-arithmetic units)
    cudaError_t (*init_generated)(void *A, void *B, long long N, unsigned long long seed, cudaStream_t st);
};

const UnitOps *unit_ops(int q, int fmt);   // lbm_units.cu (table of all compiled units)

// lbm_aux.cu
cudaError_t launch_mark_near(int q, const unsigned char *in, unsigned char *out, unsigned *bounce, int nx, int ny, int nz,
                             cudaStream_t st);
cudaError_t launch_mark_moving(int q, unsigned *bounce, const float *u0, int nx, int ny, int nz, cudaStream_t st);
cudaError_t launch_codec(int fmt, bool encode, const void *in, void *out, long long count, cudaStream_t st);
struct EncEntry;
cudaError_t enc_table(int fmt, const EncEntry **out, cudaStream_t st);   // device pointer to the format's encoder table (built on first use)
cudaError_t launch_pair_selftest(int fmt, unsigned long long *mismatches_dev, cudaStream_t st);
cudaError_t launch_div_selftest(unsigned long long *mismatches_dev, cudaStream_t st);
struct BulkGeom;
cudaError_t build_fix_lists_for(const Params &p, const BulkGeom &g, unsigned **off, uint2 **list, cudaStream_t st);

void count_launch(long long n = 1);

}  // namespace lbmk
