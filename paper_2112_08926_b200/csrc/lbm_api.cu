// lbm_api.cu -- the C ABI of include/lbm.h.  Host logic only: argument checks, device memory, the
// A/B buffer swap and kernel dispatch.  Every step of the path itself runs in the CUDA kernels of
// lbm_kernels.cuh; there is no CPU implementation of any of it in this library.
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <string>

#include "../../include/lbm.h"
#include "lbm_internal.h"

namespace lbmk {
long long launches();
}

using lbmk::Params;
using lbmk::UnitOps;

struct lbm {
    int nx, ny, nz, q, fmt, collision;
    long long N;
    float tau, omega;
    double trt_lambda;         // TRT magic parameter Lambda (R13), default 3/16
    float force[3];
    bool has_force;
    int device;
    cudaStream_t stream;
    unsigned char *flags;      // device, N bytes, bit 0 = wall, bit 7 = FLAG_NEAR
    bool has_walls;
    void *ddf[2];              // device, SoA [q][N]
    bool owns_ddf, bound;
    int cur;                   // index of the buffer holding the current state
    float *rho0, *u0;          // device copies of the init fields, kept only when the box has walls
    unsigned *bounce;          // device, N words: which directions bounce (lbm_lattice.cuh), only when the box has walls
    unsigned *fix_off;         // device: per-tile lists of flagged cell pairs for the staged kernel (lbm_stage.cuh), built on
    uint2 *fix_cells; // first use after lbm_set_flags, only when the box has flagged cells
    cudaGraphExec_t gexec[2];  // lbm_step on small boxes: GRAPH_STEPS launches captured once, starting from buffer 0 / 1
    bool graphs;               // lbm_set_graphs
    bool shifted;              // lbm_set_shifting (default true)
    void *scratch;             // device staging area of the host-pointer calls (lbm_init, lbm_read_rho_u*), kept between calls
    size_t scratch_bytes;
    long long steps;
    bool inited;
    int V;                     // stream_collide variant in use: 1, 2, 4 cells per thread or LBM_VARIANT_STAGED
    int V_request;             // LBM_VARIANT_AUTO = automatic
    const UnitOps *ops;
};

namespace {

thread_local std::string g_err;

int fail(int code, const std::string &msg) {
    g_err = msg;
    return code;
}

#define LBM_CUDA_TRY(expr)                                                                              \
    do {                                                                                                \
        cudaError_t e_ = (expr);                                                                        \
        if (e_ != cudaSuccess) {                                                                        \
            (void)cudaGetLastError();                                                                   \
            return fail(e_ == cudaErrorMemoryAllocation ? LBM_E_NOMEM : LBM_E_CUDA,                     \
                        std::string(#expr) + ": " + cudaGetErrorString(e_));                            \
        }                                                                                               \
    } while (0)

int elem_size(int fmt) { return fmt == LBM_FP64 ? 8 : (fmt == LBM_FP32 || fmt == LBM_FP64_FP32) ? 4 : 2; }
bool arith64(int fmt) { return fmt == LBM_FP64 || fmt == LBM_FP64_FP32; }
bool valid_velset(int v) { return v == LBM_D2Q9 || v == LBM_D3Q19 || v == LBM_D3Q27; }
bool valid_format(int f) { return f >= LBM_FP32 && f <= LBM_FP64_FP32; }

Params make_params(const lbm *h) {
    Params p = {};
    p.nx = h->nx; p.ny = h->ny; p.nz = h->nz;
    p.N = h->N;
    p.omega = h->omega;
    p.one_m_omega = 1.0f - h->omega;
    // R13: Lambda = (1/omega+ - 1/2)(1/omega- - 1/2), evaluated in FP32 like omega
    p.omega_minus = 1.0f / (0.5f + (float)h->trt_lambda / (h->tau - 0.5f));
    p.one_m_omega_minus = 1.0f - p.omega_minus;
    p.trt_lambda = h->trt_lambda;
    p.fx = h->force[0]; p.fy = h->force[1]; p.fz = h->force[2];
    p.flags = h->flags;
    p.rho0 = h->rho0;
    p.u0 = h->u0;
    p.bounce = h->bounce;
    p.tau = h->tau;
    p.fix_off = h->fix_off;
    p.fix_cells = h->fix_cells;
    p.shifted = h->shifted ? 1 : 0;
    return p;
}

int enter(lbm *h) {
    if (!h) return fail(LBM_E_INVAL, "null handle");
    LBM_CUDA_TRY(cudaSetDevice(h->device));
    return LBM_OK;
}

// One staging buffer per handle for the calls that take host pointers: allocated at the first such call, grown when a
// later call needs more, freed by lbm_destroy (a cudaMalloc / cudaFree pair of gigabytes per call costs milliseconds
// and synchronises the device).
// Small boxes are launch-bound (BASELINE configs 1 and 2: 32 768 and 16 384 cells, a kernel of a few microseconds): lbm_step
// captures GRAPH_STEPS consecutive launches (an even number: the A/B buffers end where they started) into a CUDA graph
// once and replays it.  Anything that changes a kernel argument drops the graphs.
constexpr int GRAPH_STEPS = 32;
constexpr long long GRAPH_MAX_CELLS = 1LL << 23;
void drop_graphs(lbm *h) {
    for (int b = 0; b < 2; ++b)
        if (h->gexec[b]) { cudaGraphExecDestroy(h->gexec[b]); h->gexec[b] = nullptr; }
}

int ensure_scratch(lbm *h, size_t bytes) {
    if (h->scratch_bytes >= bytes) return LBM_OK;
    if (h->scratch) { cudaFree(h->scratch); h->scratch = nullptr; h->scratch_bytes = 0; }
    LBM_CUDA_TRY(cudaMalloc(&h->scratch, bytes));
    h->scratch_bytes = bytes;
    return LBM_OK;
}

int ensure_ddf(lbm *h) {
    if (h->ddf[0]) return LBM_OK;
    const long long bytes = lbm_ddf_buffer_bytes(h->nx, h->ny, h->nz, h->q, h->fmt);
    for (int b = 0; b < 2; ++b) {
        cudaError_t e = cudaMalloc(&h->ddf[b], (size_t)bytes);
        if (e != cudaSuccess) {
            (void)cudaGetLastError();
            if (b == 1) { cudaFree(h->ddf[0]); }
            h->ddf[0] = h->ddf[1] = nullptr;
            return fail(LBM_E_NOMEM, std::string("cudaMalloc of a DDF buffer: ") + cudaGetErrorString(e));
        }
    }
    h->owns_ddf = true;
    return LBM_OK;
}

// Kernel variant.  Automatic choice, from the sweeps recorded in DESIGN.md section 6:
//   * FP64 arithmetic: one kernel, one cell per thread (lbm_fp64.cuh);
//   * rows 16-cell aligned and >= 64 cells, box >= 2^20 cells (2^19 with flagged cells), and either a 16-bit format or a box
//     with flagged cells:
//     the warp-specialised staged kernel (lbm_stage.cuh) -- it lifts the 16-bit formats out of the issue bound and
//     handles flagged cells in a compacted list pass instead of a divergent slow path;
//   * FP32 storage without flagged cells: the per-thread kernel, which runs at the HBM roofline;
//   * everything else (ragged rows, small L2-resident / launch-bound boxes): the per-thread kernel, 4 cells per thread
//     for D2Q9 16-bit, else 2.
int pick_variant(const lbm *h) {
    if (arith64(h->fmt) || !h->shifted) return 1;            // (the unshifted control: one kernel, one cell per thread)
    int want = h->V_request;
    const bool staged_ok = h->nx % 16 == 0 && (long long)((h->nx + h->ops->staged_tile_cells() - 1) / h->ops->staged_tile_cells()) * h->ny * h->nz < 0x7FFFFFFFLL;
    if (want == LBM_VARIANT_STAGED && staged_ok) return LBM_VARIANT_STAGED;
    // (boxes with flagged cells: from 2^19 cells -- the per-thread kernel's wall path is 1.1-1.6 times slower there already)
    if (want == 0 && staged_ok && (h->fmt != LBM_FP32 || h->has_walls) && h->nx >= 64 && h->N >= (h->has_walls ? (1LL << 19) : (1LL << 20)))
        return LBM_VARIANT_STAGED;
    if (want != 1 && want != 2 && want != 4) want = (h->q == LBM_D2Q9 && h->fmt != LBM_FP32) ? 4 : 2;
    while (want > 1 && h->nx % want != 0) want >>= 1;
    return want;
}

}  // namespace

extern "C" {

const char *lbm_last_error(void) { return g_err.c_str(); }

long long lbm_launch_count(void) { return lbmk::launches(); }

long long lbm_ddf_buffer_bytes(int nx, int ny, int nz, int velset, int ddf_format) {
    if (nx < 1 || ny < 1 || nz < 1 || !valid_velset(velset) || !valid_format(ddf_format)) return -1;
    const long long bytes = (long long)nx * ny * nz * velset * elem_size(ddf_format);
    return (bytes + 255) / 256 * 256;
}

long long lbm_bytes_per_cell(int velset, int ddf_format) {
    if (!valid_velset(velset) || !valid_format(ddf_format)) return -1;
    return 2LL * velset * elem_size(ddf_format) + 1;
}

int lbm_create(lbm_t **out, int nx, int ny, int nz, int velset, int collision, int ddf_format, float tau,
               const float *force) {
    if (!out) return fail(LBM_E_INVAL, "lbm_create: out is NULL");
    *out = nullptr;
    if (nx < 1 || ny < 1 || nz < 1) return fail(LBM_E_INVAL, "lbm_create: nx, ny, nz must be >= 1");
    if (ny > 65535 || nz > 65535) return fail(LBM_E_INVAL, "lbm_create: ny and nz must be <= 65535 (CUDA grid limit)");
    if (!valid_velset(velset)) return fail(LBM_E_INVAL, "lbm_create: velset must be 9, 19 or 27");
    if (velset == LBM_D2Q9 && nz != 1) return fail(LBM_E_INVAL, "lbm_create: D2Q9 needs nz == 1");
    if (!valid_format(ddf_format)) return fail(LBM_E_INVAL, "lbm_create: unknown ddf_format");
    if (collision != LBM_BGK && collision != LBM_TRT) return fail(LBM_E_INVAL, "lbm_create: unknown collision operator");
    if (!(tau > 0.5f)) return fail(LBM_E_INVAL, "lbm_create: tau must be > 0.5 (PAPER.md:79)");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        (void)cudaGetLastError();
        return fail(LBM_E_CUDA, "lbm_create: no CUDA device (this library has no CPU fallback)");
    }
    lbm *h = new (std::nothrow) lbm();
    if (!h) return fail(LBM_E_NOMEM, "lbm_create: out of host memory");
    std::memset(h, 0, sizeof *h);
    h->nx = nx; h->ny = ny; h->nz = nz; h->q = velset; h->fmt = ddf_format; h->collision = collision;
    h->N = (long long)nx * ny * nz;
    h->tau = tau;
    h->omega = 1.0f / tau;
    h->trt_lambda = 3.0 / 16.0;
    h->graphs = true;
    h->shifted = true;
    for (int a = 0; a < 3; ++a) {
        h->force[a] = force ? force[a] : 0.0f;
        if (h->force[a] != 0.0f) h->has_force = true;
    }
    h->ops = lbmk::unit_ops(velset, ddf_format);
    if (!h->ops) { delete h; return fail(LBM_E_UNSUPPORTED, "lbm_create: no kernel unit for this velset/format"); }
    cudaError_t e = cudaGetDevice(&h->device);
    if (e == cudaSuccess) e = cudaMalloc((void **)&h->flags, (size_t)h->N);
    if (e == cudaSuccess) e = cudaMemset(h->flags, 0, (size_t)h->N);
    if (e != cudaSuccess) {
        (void)cudaGetLastError();
        if (h->flags) cudaFree(h->flags);
        delete h;
        return fail(e == cudaErrorMemoryAllocation ? LBM_E_NOMEM : LBM_E_CUDA, std::string("lbm_create: ") + cudaGetErrorString(e));
    }
    *out = h;
    return LBM_OK;
}

int lbm_bind(lbm_t *h, void *ddf_a, void *ddf_b, void *cuda_stream) {
    if (int rc = enter(h)) return rc;
    if (h->inited) return fail(LBM_E_STATE, "lbm_bind: must be called before lbm_init");
    if ((ddf_a == nullptr) != (ddf_b == nullptr)) return fail(LBM_E_INVAL, "lbm_bind: bind both DDF buffers or neither");
    if (ddf_a) {
        if (((size_t)ddf_a | (size_t)ddf_b) & 15) return fail(LBM_E_INVAL, "lbm_bind: DDF buffers must be 16-byte aligned");
        const long long need = lbm_ddf_buffer_bytes(h->nx, h->ny, h->nz, h->q, h->fmt);
        const char *pa = (const char *)ddf_a, *pb = (const char *)ddf_b;
        if ((pa <= pb ? pb - pa : pa - pb) < need) return fail(LBM_E_INVAL, "lbm_bind: the two DDF buffers overlap");
        if (h->owns_ddf) { cudaFree(h->ddf[0]); cudaFree(h->ddf[1]); h->owns_ddf = false; }
        h->ddf[0] = ddf_a;
        h->ddf[1] = ddf_b;
    }
    drop_graphs(h);
    h->stream = (cudaStream_t)cuda_stream;
    h->bound = true;
    return LBM_OK;
}

int lbm_set_variant(lbm_t *h, int v) {
    if (int rc = enter(h)) return rc;
    if (v == LBM_VARIANT_BULK) v = LBM_VARIANT_STAGED;           // the first staged kernel's name, kept for callers
    if (v != LBM_VARIANT_AUTO && v != 1 && v != 2 && v != 4 && v != LBM_VARIANT_STAGED)
        return fail(LBM_E_INVAL, "lbm_set_variant: 0 (auto), 1, 2, 4 (cells per thread) or LBM_VARIANT_STAGED");
    if ((v == 2 || v == 4) && h->nx % v != 0) return fail(LBM_E_INVAL, "lbm_set_variant: nx must be a multiple of the cells per thread");
    const bool staged = v == LBM_VARIANT_STAGED;
    if (staged && h->nx % 16 != 0) return fail(LBM_E_INVAL, "lbm_set_variant: the staged kernel needs nx to be a multiple of 16");
    if (staged && arith64(h->fmt)) return fail(LBM_E_UNSUPPORTED, "lbm_set_variant: the FP64-arithmetic formats have no staged kernel");
    drop_graphs(h);
    h->V_request = v;
    h->V = pick_variant(h);
    if (staged && h->V != v) return fail(LBM_E_INVAL, "lbm_set_variant: box too large for the staged kernel's tile index");
    return LBM_OK;
}

int lbm_set_trt_lambda(lbm_t *h, double lambda) {
    if (int rc = enter(h)) return rc;
    if (h->collision != LBM_TRT) return fail(LBM_E_STATE, "lbm_set_trt_lambda: the handle was not created with LBM_TRT");
    if (!(lambda > 0.0) || !(lambda < 1e30)) return fail(LBM_E_INVAL, "lbm_set_trt_lambda: Lambda must be positive and finite");
    // FP32 arithmetic sees the FP32 value of Lambda, FP64 arithmetic the double as given
    drop_graphs(h);
    h->trt_lambda = arith64(h->fmt) ? lambda : (double)(float)lambda;
    return LBM_OK;
}

int lbm_set_cells_per_thread(lbm_t *h, int v) {
    if (v != 0 && v != 1 && v != 2 && v != 4) return fail(LBM_E_INVAL, "lbm_set_cells_per_thread: 0 (auto), 1, 2 or 4");
    return lbm_set_variant(h, v);
}

int lbm_set_flags(lbm_t *h, const unsigned char *flags) {
    if (int rc = enter(h)) return rc;
    if (!flags) return fail(LBM_E_INVAL, "lbm_set_flags: flags is NULL");
    if (h->inited) return fail(LBM_E_STATE, "lbm_set_flags: must be called before lbm_init");
    bool walls = false;
    for (long long n = 0; n < h->N; ++n) {
        if (flags[n] & ~(LBM_FLAG_WALL | LBM_FLAG_EQ | LBM_FLAG_OUT)) return fail(LBM_E_INVAL, "lbm_set_flags: unknown flag bit set");
        if (flags[n] & (flags[n] - 1)) return fail(LBM_E_INVAL, "lbm_set_flags: a cell is a wall, an equilibrium boundary or an outflow cell, not several");
        walls |= flags[n] != 0;
    }
    h->has_walls = walls;
    drop_graphs(h);
    if (h->fix_off) { cudaFree(h->fix_off); h->fix_off = nullptr; }       // the lists belong to the old flags
    if (h->fix_cells) { cudaFree(h->fix_cells); h->fix_cells = nullptr; }
    if (!walls) {
        LBM_CUDA_TRY(cudaMemsetAsync(h->flags, 0, (size_t)h->N, h->stream));
        LBM_CUDA_TRY(cudaStreamSynchronize(h->stream));
        return LBM_OK;
    }
    unsigned char *tmp = nullptr;
    if (!h->bounce) LBM_CUDA_TRY(cudaMalloc((void **)&h->bounce, (size_t)h->N * 4));
    LBM_CUDA_TRY(cudaMalloc((void **)&tmp, (size_t)h->N));
    cudaError_t e = cudaMemcpyAsync(tmp, flags, (size_t)h->N, cudaMemcpyHostToDevice, h->stream);
    if (e == cudaSuccess) e = lbmk::launch_mark_near(h->q, tmp, h->flags, h->bounce, h->nx, h->ny, h->nz, h->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
    cudaFree(tmp);
    LBM_CUDA_TRY(e);
    return LBM_OK;
}

static int init_from_device(lbm *h, const float *rho_dev, const float *u_dev) {
    if (int rc = ensure_ddf(h)) return rc;
    drop_graphs(h);
    if (h->fix_off) { cudaFree(h->fix_off); h->fix_off = nullptr; }       // the lists carry the "wall moves" bits of the old fields
    if (h->fix_cells) { cudaFree(h->fix_cells); h->fix_cells = nullptr; }
    const float *r = rho_dev, *u = u_dev;
    if (h->has_walls) {                          // wall velocity (R9) and wall read-out (R12) need the init fields later
        if (!h->rho0) LBM_CUDA_TRY(cudaMalloc((void **)&h->rho0, (size_t)h->N * 4));
        if (!h->u0) LBM_CUDA_TRY(cudaMalloc((void **)&h->u0, (size_t)h->N * 12));
        if (h->rho0 != rho_dev) LBM_CUDA_TRY(cudaMemcpyAsync(h->rho0, rho_dev, (size_t)h->N * 4, cudaMemcpyDeviceToDevice, h->stream));
        if (h->u0 != u_dev) LBM_CUDA_TRY(cudaMemcpyAsync(h->u0, u_dev, (size_t)h->N * 12, cudaMemcpyDeviceToDevice, h->stream));
        r = h->rho0;
        u = h->u0;
        LBM_CUDA_TRY(lbmk::launch_mark_moving(h->q, h->bounce, h->u0, h->nx, h->ny, h->nz, h->stream));
    }
    LBM_CUDA_TRY(h->ops->init(h->ddf[0], h->ddf[1], r, u, h->N, h->shifted, h->stream));
    h->cur = 0;
    h->steps = 0;
    h->inited = true;
    h->V = pick_variant(h);
    return LBM_OK;
}

int lbm_init_device(lbm_t *h, const float *rho_dev, const float *u_dev) {
    if (int rc = enter(h)) return rc;
    if (!rho_dev || !u_dev) return fail(LBM_E_INVAL, "lbm_init_device: rho and u must not be NULL");
    return init_from_device(h, rho_dev, u_dev);
}

int lbm_init_generated(lbm_t *h, unsigned long long seed) {
    if (int rc = enter(h)) return rc;
    if (arith64(h->fmt) || !h->ops->init_generated) return fail(LBM_E_UNSUPPORTED, "lbm_init_generated: not for the FP64-arithmetic formats");
    if (h->has_walls) return fail(LBM_E_STATE, "lbm_init_generated: the box has flagged cells (their fields must be given: lbm_init)");
    if (!h->shifted) return fail(LBM_E_UNSUPPORTED, "lbm_init_generated: with DDF-shifting only");
    if (int rc = ensure_ddf(h)) return rc;
    drop_graphs(h);
    LBM_CUDA_TRY(h->ops->init_generated(h->ddf[0], h->ddf[1], h->N, seed, h->stream));
    h->cur = 0;
    h->steps = 0;
    h->inited = true;
    h->V = pick_variant(h);
    return LBM_OK;
}

int lbm_init(lbm_t *h, const float *rho, const float *u) {
    if (int rc = enter(h)) return rc;
    if (!rho || !u) return fail(LBM_E_INVAL, "lbm_init: rho and u must not be NULL");
    float *r = nullptr, *v = nullptr;
    if (h->has_walls) {
        if (!h->rho0) LBM_CUDA_TRY(cudaMalloc((void **)&h->rho0, (size_t)h->N * 4));
        if (!h->u0) LBM_CUDA_TRY(cudaMalloc((void **)&h->u0, (size_t)h->N * 12));
        r = h->rho0;
        v = h->u0;
    } else {
        if (int rc = ensure_scratch(h, (size_t)h->N * 16)) return rc;
        r = (float *)h->scratch;
        v = r + h->N;
    }
    cudaError_t e = cudaMemcpyAsync(r, rho, (size_t)h->N * 4, cudaMemcpyHostToDevice, h->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(v, u, (size_t)h->N * 12, cudaMemcpyHostToDevice, h->stream);
    int rc = LBM_OK;
    if (e == cudaSuccess) rc = init_from_device(h, r, v);
    cudaError_t e2 = cudaStreamSynchronize(h->stream);
    LBM_CUDA_TRY(e);
    if (rc) return rc;
    LBM_CUDA_TRY(e2);
    return LBM_OK;
}

static int step_plain(lbm *h, const Params &p, int n) {
    for (int k = 0; k < n; ++k) {
        LBM_CUDA_TRY(h->ops->stream_collide(h->ddf[h->cur], h->ddf[1 - h->cur], p, h->V, h->collision, h->has_force, h->stream));
        h->cur = 1 - h->cur;
        h->steps += 1;
    }
    return LBM_OK;
}

int lbm_step(lbm_t *h, int n) {
    if (int rc = enter(h)) return rc;
    if (n < 0) return fail(LBM_E_INVAL, "lbm_step: n must be >= 0");
    if (!h->inited) return fail(LBM_E_STATE, "lbm_step: call lbm_init first");
    if (h->V == LBM_VARIANT_STAGED && h->has_walls && !h->fix_off && n > 0)
        LBM_CUDA_TRY(h->ops->build_fix_lists(make_params(h), &h->fix_off, &h->fix_cells, h->stream));
    const Params p = make_params(h);
    if (h->graphs && h->N <= GRAPH_MAX_CELLS && n >= 2 + GRAPH_STEPS) {
        cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
        if (cudaStreamIsCapturing(h->stream, &cs) == cudaSuccess && cs == cudaStreamCaptureStatusNone) {
            if (!h->gexec[h->cur]) {
                // both directions once outside the capture (first launches set function attributes, build tables)
                if (int rc = step_plain(h, p, 2)) return rc;
                n -= 2;
                cudaGraph_t graph = nullptr;
                const long long steps0 = h->steps;
                const int cur0 = h->cur;
                cudaError_t e = cudaStreamBeginCapture(h->stream, cudaStreamCaptureModeThreadLocal);
                int rc = LBM_OK;
                if (e == cudaSuccess) {
                    rc = step_plain(h, p, GRAPH_STEPS);
                    e = cudaStreamEndCapture(h->stream, &graph);
                }
                h->steps = steps0;                              // captured, not executed
                h->cur = cur0;
                lbmk::count_launch(-(long long)GRAPH_STEPS);
                if (rc == LBM_OK && e == cudaSuccess && graph) e = cudaGraphInstantiate(&h->gexec[cur0], graph, 0);
                if (graph) cudaGraphDestroy(graph);
                if (rc != LBM_OK || e != cudaSuccess) {          // no graph: plain launches below
                    (void)cudaGetLastError();
                    h->gexec[cur0] = nullptr;
                }
            }
            while (h->gexec[h->cur] && n >= GRAPH_STEPS) {
                LBM_CUDA_TRY(cudaGraphLaunch(h->gexec[h->cur], h->stream));
                lbmk::count_launch(GRAPH_STEPS);
                h->steps += GRAPH_STEPS;
                n -= GRAPH_STEPS;
            }
        }
    }
    return step_plain(h, p, n);
}

int lbm_set_shifting(lbm_t *h, int on) {
    if (int rc = enter(h)) return rc;
    if (h->inited) return fail(LBM_E_STATE, "lbm_set_shifting: must be called before lbm_init");
    if (!on && arith64(h->fmt)) return fail(LBM_E_UNSUPPORTED, "lbm_set_shifting: the FP64-arithmetic formats run with DDF-shifting only");
    h->shifted = on != 0;
    drop_graphs(h);
    return LBM_OK;
}

int lbm_set_graphs(lbm_t *h, int enable) {
    if (int rc = enter(h)) return rc;
    h->graphs = enable != 0;
    if (!h->graphs) drop_graphs(h);
    return LBM_OK;
}

int lbm_read_rho_u_device(lbm_t *h, float *rho_dev, float *u_dev) {
    if (int rc = enter(h)) return rc;
    if (!h->inited) return fail(LBM_E_STATE, "lbm_read_rho_u: call lbm_init first");
    if (!rho_dev && !u_dev) return LBM_OK;
    LBM_CUDA_TRY(h->ops->read(h->ddf[h->cur], make_params(h), h->has_force, rho_dev, u_dev, h->stream));
    return LBM_OK;
}

int lbm_read_rho_u(lbm_t *h, float *rho, float *u) {
    if (int rc = enter(h)) return rc;
    if (!h->inited) return fail(LBM_E_STATE, "lbm_read_rho_u: call lbm_init first");
    if (!rho && !u) return LBM_OK;
    if (int rc = ensure_scratch(h, (size_t)h->N * 16)) return rc;
    float *d = (float *)h->scratch;
    cudaError_t e = h->ops->read(h->ddf[h->cur], make_params(h), h->has_force, rho ? d : nullptr, u ? d + h->N : nullptr, h->stream);
    if (e == cudaSuccess && rho) e = cudaMemcpyAsync(rho, d, (size_t)h->N * 4, cudaMemcpyDeviceToHost, h->stream);
    if (e == cudaSuccess && u) e = cudaMemcpyAsync(u, d + h->N, (size_t)h->N * 12, cudaMemcpyDeviceToHost, h->stream);
    cudaError_t e2 = cudaStreamSynchronize(h->stream);
    LBM_CUDA_TRY(e);
    LBM_CUDA_TRY(e2);
    return LBM_OK;
}

int lbm_read_rho_u_f64(lbm_t *h, double *rho, double *u) {
    if (int rc = enter(h)) return rc;
    if (!h->inited) return fail(LBM_E_STATE, "lbm_read_rho_u_f64: call lbm_init first");
    if (!h->ops->read64) return fail(LBM_E_UNSUPPORTED, "lbm_read_rho_u_f64: FP64-arithmetic formats only (LBM_FP64, LBM_FP64_FP32)");
    if (!rho && !u) return LBM_OK;
    if (int rc = ensure_scratch(h, (size_t)h->N * 32)) return rc;
    double *d = (double *)h->scratch;
    cudaError_t e = h->ops->read64(h->ddf[h->cur], make_params(h), h->has_force, rho ? d : nullptr, u ? d + h->N : nullptr, h->stream);
    if (e == cudaSuccess && rho) e = cudaMemcpyAsync(rho, d, (size_t)h->N * 8, cudaMemcpyDeviceToHost, h->stream);
    if (e == cudaSuccess && u) e = cudaMemcpyAsync(u, d + h->N, (size_t)h->N * 24, cudaMemcpyDeviceToHost, h->stream);
    cudaError_t e2 = cudaStreamSynchronize(h->stream);
    LBM_CUDA_TRY(e);
    LBM_CUDA_TRY(e2);
    return LBM_OK;
}

int lbm_read_rho_u_at(lbm_t *h, const long long *cells, int count, float *rho, float *u) {
    if (int rc = enter(h)) return rc;
    if (!h->inited) return fail(LBM_E_STATE, "lbm_read_rho_u_at: call lbm_init first");
    if (count < 0 || (count > 0 && (!cells || !rho || !u))) return fail(LBM_E_INVAL, "lbm_read_rho_u_at: bad arguments");
    if (count == 0) return LBM_OK;
    for (int k = 0; k < count; ++k)
        if (cells[k] < 0 || cells[k] >= h->N) return fail(LBM_E_INVAL, "lbm_read_rho_u_at: cell index out of range");
    const size_t cb = (size_t)count * 8, fb = (size_t)count * 16;
    if (int rc = ensure_scratch(h, cb + fb)) return rc;
    char *d = (char *)h->scratch;
    float *df = (float *)(d + cb);
    cudaError_t e = cudaMemcpyAsync(d, cells, cb, cudaMemcpyHostToDevice, h->stream);
    if (e == cudaSuccess) e = h->ops->probe(h->ddf[h->cur], make_params(h), h->has_force, (const long long *)d, count, df, df + count, h->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(rho, df, (size_t)count * 4, cudaMemcpyDeviceToHost, h->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(u, df + count, (size_t)count * 12, cudaMemcpyDeviceToHost, h->stream);
    cudaError_t e2 = cudaStreamSynchronize(h->stream);
    LBM_CUDA_TRY(e);
    LBM_CUDA_TRY(e2);
    return LBM_OK;
}

}  // extern "C"

// ---- lbm_read_rho_u_at_static: the probe read-out for callers that must not allocate ---------------------------
// The scratch of lbm_read_rho_u_at (the cell indices on the device + the kernel's outputs) comes from the handle's
// staging buffer, i.e. from cudaMalloc at the first call and whenever a call needs more.  Here it is a fixed array in the
// library's image: 24 bytes per probe (8-byte cell index | rho | ux | uy | uz), LBM_STATIC_PROBES_MAX probes, 96 KiB
// that every GPU which loads the library holds until the process exits.
// In host code the array's NAME is a host-side stand-in, not a device address: its address comes from
// cudaGetSymbolAddress, asked once per device with that device current (the array exists once per device).
static __device__ __align__(256) unsigned char g_static_probe_scratch[LBM_STATIC_PROBES_MAX * 24];

namespace {
int static_probe_scratch(int device, unsigned char **out) {          // the caller has made `device` current (enter())
    static std::mutex mu;
    static unsigned char *addr[64];
    if (device < 0 || device >= 64) return fail(LBM_E_INVAL, "lbm_read_rho_u_at_static: device ordinal out of range");
    std::lock_guard<std::mutex> lock(mu);
    if (!addr[device]) {
        void *ptr = nullptr;
        LBM_CUDA_TRY(cudaGetSymbolAddress(&ptr, g_static_probe_scratch));
        addr[device] = (unsigned char *)ptr;
    }
    *out = addr[device];
    return LBM_OK;
}
}  // namespace

extern "C" {

int lbm_read_rho_u_at_static(lbm_t *h, const long long *cells, int count, float *rho, float *u) {
    if (int rc = enter(h)) return rc;
    if (!h->inited) return fail(LBM_E_STATE, "lbm_read_rho_u_at_static: call lbm_init first");
    if (count < 0 || (count > 0 && (!cells || !rho || !u))) return fail(LBM_E_INVAL, "lbm_read_rho_u_at_static: bad arguments");
    if (count > LBM_STATIC_PROBES_MAX)
        return fail(LBM_E_INVAL, "lbm_read_rho_u_at_static: count = " + std::to_string(count) + " exceeds LBM_STATIC_PROBES_MAX = " +
                                     std::to_string(LBM_STATIC_PROBES_MAX) + " (the fixed scratch array; use lbm_read_rho_u_at)");
    if (count == 0) return LBM_OK;
    for (int k = 0; k < count; ++k)
        if (cells[k] < 0 || cells[k] >= h->N) return fail(LBM_E_INVAL, "lbm_read_rho_u_at_static: cell index out of range");
    unsigned char *d = nullptr;
    if (int rc = static_probe_scratch(h->device, &d)) return rc;
    // layout: count cell indices, then rho [count], then u [3][count].  The array keeps the last call's contents; nothing
    // here must start at zero: the copy below and the kernel overwrite every byte that is read afterwards.
    const size_t cb = (size_t)count * 8;
    float *df = (float *)(d + cb);
    cudaError_t e = cudaMemcpyAsync(d, cells, cb, cudaMemcpyHostToDevice, h->stream);
    if (e == cudaSuccess) e = h->ops->probe(h->ddf[h->cur], make_params(h), h->has_force, (const long long *)d, count, df, df + count, h->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(rho, df, (size_t)count * 4, cudaMemcpyDeviceToHost, h->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(u, df + count, (size_t)count * 12, cudaMemcpyDeviceToHost, h->stream);
    cudaError_t e2 = cudaStreamSynchronize(h->stream);
    LBM_CUDA_TRY(e);
    LBM_CUDA_TRY(e2);
    return LBM_OK;
}

int lbm_read_ddf(lbm_t *h, int i, void *out) {
    if (int rc = enter(h)) return rc;
    if (!h->inited) return fail(LBM_E_STATE, "lbm_read_ddf: call lbm_init first");
    if (i < 0 || i >= h->q || !out) return fail(LBM_E_INVAL, "lbm_read_ddf: bad direction or NULL pointer");
    const size_t es = (size_t)elem_size(h->fmt);
    LBM_CUDA_TRY(cudaMemcpyAsync(out, (const char *)h->ddf[h->cur] + (size_t)i * h->N * es, (size_t)h->N * es,
                                 cudaMemcpyDeviceToHost, h->stream));
    LBM_CUDA_TRY(cudaStreamSynchronize(h->stream));
    return LBM_OK;
}

int lbm_sync(lbm_t *h) {
    if (int rc = enter(h)) return rc;
    LBM_CUDA_TRY(cudaStreamSynchronize(h->stream));
    return LBM_OK;
}

long long lbm_steps_done(const lbm_t *h) { return h ? h->steps : -1; }

const char *lbm_kernel_name(const lbm_t *h) {
    if (!h || !h->inited) return "";
    return h->ops->name(h->V, h->collision, h->has_force);
}

int lbm_destroy(lbm_t *h) {
    if (!h) return LBM_OK;
    cudaSetDevice(h->device);
    cudaStreamSynchronize(h->stream);
    drop_graphs(h);
    if (h->owns_ddf) { cudaFree(h->ddf[0]); cudaFree(h->ddf[1]); }
    if (h->flags) cudaFree(h->flags);
    if (h->rho0) cudaFree(h->rho0);
    if (h->u0) cudaFree(h->u0);
    if (h->bounce) cudaFree(h->bounce);
    if (h->fix_off) cudaFree(h->fix_off);
    if (h->fix_cells) cudaFree(h->fix_cells);
    if (h->scratch) cudaFree(h->scratch);
    (void)cudaGetLastError();
    delete h;
    return LBM_OK;
}

// ---- codecs -------------------------------------------------------------------------------------
int lbm_codec_encode_device(int ddf_format, const float *x_dev, unsigned short *codes_dev, long long count, void *cuda_stream) {
    if (ddf_format < LBM_FP16S || ddf_format > LBM_FP16) return fail(LBM_E_INVAL, "lbm_codec_encode: 16-bit formats only");
    if (count < 0 || (count > 0 && (!x_dev || !codes_dev))) return fail(LBM_E_INVAL, "lbm_codec_encode: bad arguments");
    if (count == 0) return LBM_OK;
    LBM_CUDA_TRY(lbmk::launch_codec(ddf_format, true, x_dev, codes_dev, count, (cudaStream_t)cuda_stream));
    return LBM_OK;
}

int lbm_codec_decode_device(int ddf_format, const unsigned short *codes_dev, float *x_dev, long long count, void *cuda_stream) {
    if (ddf_format < LBM_FP16S || ddf_format > LBM_FP16) return fail(LBM_E_INVAL, "lbm_codec_decode: 16-bit formats only");
    if (count < 0 || (count > 0 && (!x_dev || !codes_dev))) return fail(LBM_E_INVAL, "lbm_codec_decode: bad arguments");
    if (count == 0) return LBM_OK;
    LBM_CUDA_TRY(lbmk::launch_codec(ddf_format, false, codes_dev, x_dev, count, (cudaStream_t)cuda_stream));
    return LBM_OK;
}

static int codec_host(int fmt, bool encode, const void *in, void *out, long long count) {
    if (fmt < LBM_FP16S || fmt > LBM_FP16) return fail(LBM_E_INVAL, "lbm_codec: 16-bit formats only");
    if (count < 0 || (count > 0 && (!in || !out))) return fail(LBM_E_INVAL, "lbm_codec: bad arguments");
    if (count == 0) return LBM_OK;
    const size_t in_b = (size_t)count * (encode ? 4 : 2), out_b = (size_t)count * (encode ? 2 : 4);
    void *din = nullptr, *dout = nullptr;
    LBM_CUDA_TRY(cudaMalloc(&din, in_b));
    cudaError_t e = cudaMalloc(&dout, out_b);
    if (e == cudaSuccess) e = cudaMemcpy(din, in, in_b, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = lbmk::launch_codec(fmt, encode, din, dout, count, 0);
    if (e == cudaSuccess) e = cudaMemcpy(out, dout, out_b, cudaMemcpyDeviceToHost);
    cudaFree(din);
    if (dout) cudaFree(dout);
    LBM_CUDA_TRY(e);
    return LBM_OK;
}

int lbm_codec_encode(int ddf_format, const float *x, unsigned short *codes, long long count) {
    return codec_host(ddf_format, true, x, codes, count);
}
int lbm_codec_decode(int ddf_format, const unsigned short *codes, float *x, long long count) {
    return codec_host(ddf_format, false, codes, x, count);
}

int lbm_codec_pair_selftest(int ddf_format, long long *mismatches) {
    if (ddf_format < LBM_FP16S || ddf_format > LBM_FP16 || !mismatches) return fail(LBM_E_INVAL, "lbm_codec_pair_selftest: bad arguments");
    unsigned long long *d = nullptr, hval = 0;
    LBM_CUDA_TRY(cudaMalloc((void **)&d, 8));
    cudaError_t e = cudaMemset(d, 0, 8);
    if (e == cudaSuccess) e = lbmk::launch_pair_selftest(ddf_format, d, 0);
    if (e == cudaSuccess) e = cudaMemcpy(&hval, d, 8, cudaMemcpyDeviceToHost);
    cudaFree(d);
    LBM_CUDA_TRY(e);
    *mismatches = (long long)hval;
    return LBM_OK;
}

int lbm_div_selftest(long long *mismatches) {
    if (!mismatches) return fail(LBM_E_INVAL, "lbm_div_selftest: mismatches is NULL");
    unsigned long long *d = nullptr, hval = 0;
    LBM_CUDA_TRY(cudaMalloc((void **)&d, 8));
    cudaError_t e = cudaMemset(d, 0, 8);
    if (e == cudaSuccess) e = lbmk::launch_div_selftest(d, 0);
    if (e == cudaSuccess) e = cudaMemcpy(&hval, d, 8, cudaMemcpyDeviceToHost);
    cudaFree(d);
    LBM_CUDA_TRY(e);
    *mismatches = (long long)hval;
    return LBM_OK;
}

}  // extern "C"