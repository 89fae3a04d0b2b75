/* include/lbm.h -- C ABI of liblbm_b200.so: the fused LBM stream-collide time step with decoupled
 * arithmetic (FP32) and storage (FP32 / 16-bit) precision, for one NVIDIA B200 (sm_100a).
 *
 * The method is the one of Lehmann et al., arXiv 2112.08926 ("PAPER.md" below = the paper text,
 * cited as PAPER.md:<line>); every reading of a silent / garbled passage is listed in DESIGN.md
 * section 3 ("R<n>").  Nothing here is torch-typed: plain pointers and sizes.  Each pointer argument
 * says whether it is a HOST or a DEVICE pointer.
 *
 * Conventions
 *   - every function returns an int status: LBM_OK (0) or a negative LBM_E_* code; no C++ exception
 *     crosses the boundary; lbm_last_error() gives a thread-local human-readable message.
 *   - cell index n = x + nx*(y + ny*z); N = nx*ny*nz.
 *   - DDF buffers are structure-of-arrays [q][N], element = float (LBM_FP32, LBM_FP64_FP32),
 *     double (LBM_FP64) or uint16 (all other formats); the library keeps two of them (A-B / one-step pull).
 *     The stored quantity is the SHIFTED DDF f_i - w_i.
 *   - rho is float [N]; u is float [3][N] (ux | uy | uz).
 *   - flags are 1 byte per cell; bit LBM_FLAG_WALL (TYPE_W) marks a halfway
 *     bounce-back wall cell.  The u entries of a wall cell are the wall velocity (moving wall, R9).
 *   - all faces are periodic; solid boundaries exist only as wall cells.
 *   - a handle is bound to the CUDA device that was current at lbm_create and to one stream; calls on
 *     one handle must not race.  lbm_step is asynchronous on that stream; everything that returns data
 *     to the host synchronises the stream.
 *   - there is NO CPU fallback: without a usable CUDA device lbm_create fails with LBM_E_CUDA.
 */
#ifndef LBM_B200_H
#define LBM_B200_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lbm lbm_t; /* opaque, owned by the library, freed by lbm_destroy */

/* velocity sets (R1: D3Q19 numbering from PAPER.md:955-959, 1029-1031; D2Q9 needs nz == 1) */
enum { LBM_D2Q9 = 9, LBM_D3Q19 = 19, LBM_D3Q27 = 27 };
/* collision operators.  BGK = eq (28).  TRT is named but never
 * defined by the paper; LBM_TRT is the textbook two-relaxation-time operator (R13): per opposite pair
 * (i, i') the symmetric part (f_i + f_i')/2 relaxes towards its equilibrium with omega+ = 1/tau, the antisymmetric
 * part (f_i - f_i')/2 with omega-, where Lambda = (1/omega+ - 1/2)(1/omega- - 1/2) (see lbm_set_trt_lambda); the
 * Guo source term splits the same way.  Same memory traffic as BGK. */
enum { LBM_BGK = 0, LBM_TRT = 1 };
/* DDF storage formats (Table 2, 152-178, 201-219; Listing 1) */
enum {
    LBM_FP32 = 0,   /* IEEE binary32, identity load/store                        */
    LBM_FP16S = 1,  /* IEEE binary16 of x*2^15, round-to-nearest-even   */
    LBM_FP16C = 2,  /* custom 1-4-11, bias 15, no Inf/NaN, saturating   */
    LBM_P16_0S = 3, /* posit<16,0>, sign-magnitude, scaled by 2^7      */
    LBM_P16_1S = 4, /* posit<16,1>, sign-magnitude, scaled by 2^7  */
    LBM_P16_2C = 5, /* one-sided regime, 2 exponent bits, unscaled */
    LBM_FP16 = 6,   /* plain IEEE binary16 (Table 2 row 139)                          */
    /* The two formats below also switch the ARITHMETIC to IEEE binary64 (the paper's "FP64/FP64" and "FP64/FP32"
     * columns, arithmetic / storage; Tables 3-5): same path, same operation order,
     * omega = 1 / (double)tau, weights and 1/sqrt(3) in double.  rho, u, force and the wall velocity stay float at
     * this boundary and are widened exactly; lbm_read_rho_u rounds the double results to float,
     * lbm_read_rho_u_f64 returns them unrounded. */
    LBM_FP64 = 7,     /* element = double, identity load/store                                      */
    LBM_FP64_FP32 = 8 /* element = float: load widens, store rounds to nearest even                 */
};
/* LBM_FLAG_WALL: halfway bounce-back wall cell (TYPE_W), optionally moving (its u).
 * LBM_FLAG_EQ:   equilibrium boundary cell (TYPE_E; "equilibrium boundaries"; R15): it keeps
 *                the DDFs lbm_init gave it -- the shifted equilibrium of its rho, u -- for ever; its neighbours pull
 *                from it as from a fluid cell (inflow / outflow / free-stream perimeter).
 * Neither kind of cell is written by lbm_step; lbm_read_rho_u returns for them the fields given to lbm_init.
 * LBM_FLAG_OUT:  zero-gradient outflow cell (BASELINE configs[3] "zero-gradient outflow"; NOT in the paper: DESIGN.md R18):
 *                every step it takes the shifted equilibrium of the density and velocity of its upstream neighbour, the
 *                cell at x - 1 (periodic), as that neighbour's stored DDFs give them (local moments, u = (j - F/2) / rho).
 *                Neighbours pull from it as from a fluid cell; lbm_read_rho_u reads it like a fluid cell.
 * A cell carries at most one of the three bits. */
enum { LBM_FLAG_WALL = 0x01, LBM_FLAG_EQ = 0x02, LBM_FLAG_OUT = 0x04 };
enum {
    LBM_OK = 0,
    LBM_E_INVAL = -1,       /* bad argument                                   */
    LBM_E_UNSUPPORTED = -2, /* valid request the library does not implement   */
    LBM_E_NOMEM = -3,       /* device or host allocation failed               */
    LBM_E_CUDA = -4,        /* CUDA runtime error (message in lbm_last_error) */
    LBM_E_STATE = -5        /* call sequence violated                         */
};

/* Create a simulation.  nx, ny, nz >= 1 (nz == 1 for LBM_D2Q9); tau > 0.5 (omega = 1/tau,
 * PAPER.md:707); force: HOST pointer to 3 floats (uniform body force, Guo forcing R10) or NULL.
 * Allocates the flags (all fluid) but no DDF memory: that happens at the first lbm_bind / lbm_init.
 * On success *out is the new handle. */
int lbm_create(lbm_t **out, int nx, int ny, int nz, int velset, int collision, int ddf_format, float tau,
               const float *force);

/* Optional: run on caller-owned device memory and/or a caller-owned stream (e.g. torch tensors and
 * torch's current stream).  ddf_a, ddf_b: DEVICE pointers, each at least lbm_ddf_buffer_bytes() bytes,
 * 16-byte aligned, must outlive the handle; both NULL = library allocates.  cuda_stream: a cudaStream_t
 * cast to void* (NULL = the legacy default stream).  Must be called before lbm_init. */
int lbm_bind(lbm_t *h, void *ddf_a, void *ddf_b, void *cuda_stream);

/* Tuning knob: which stream_collide kernel runs.  The result of a run does not depend on it (tests check that
 * bit for bit).
 *   LBM_VARIANT_AUTO   the library chooses;
 *   1, 2, 4            the per-thread kernel with that many cells per thread along x (nx a multiple of it);
 *   LBM_VARIANT_STAGED the shared-memory-staged kernel: persistent CTAs, one loader and one storer warp move every
 *                      DDF with cp.async.bulk, the other warps only compute (nx a multiple of 16).
 *                      LBM_VARIANT_BULK is the same kernel (the name of its first version).
 * lbm_set_cells_per_thread(h, v) = lbm_set_variant(h, v) restricted to v in {0, 1, 2, 4}. */
enum { LBM_VARIANT_AUTO = 0, LBM_VARIANT_BULK = 16, LBM_VARIANT_STAGED = 32 };
int lbm_set_variant(lbm_t *h, int variant);
int lbm_set_cells_per_thread(lbm_t *h, int v);

/* LBM_TRT handles only (else LBM_E_STATE): the magic parameter Lambda > 0 (else LBM_E_INVAL), default 3/16 (the
 * halfway bounce-back wall of a Poiseuille channel then sits exactly half a cell outside the last fluid node).
 * Lambda = (tau - 1/2)^2 makes omega- = omega+.  The FP32-arithmetic formats use the value rounded to FP32.  May be
 * called at any time between steps; takes effect from the next lbm_step. */
int lbm_set_trt_lambda(lbm_t *h, double lambda);

/* The paper's negative control (eqs (19)-(23); dashed curves of PAPER.md:265, 316): on = 0 stores f_i
 * instead of f_i - w_i, sums rho without the "+1" and takes f^eq from eq (22) (R17).  Default on = 1.  Before
 * lbm_init (else LBM_E_STATE); not for the FP64-arithmetic formats (LBM_E_UNSUPPORTED).  The control runs on the
 * per-thread kernel with one cell per thread: it exists to show what DDF-shifting buys, not to be fast. */
int lbm_set_shifting(lbm_t *h, int on);

/* Set the cell flags.  flags: HOST pointer, N bytes, copied.  One of LBM_FLAG_WALL, LBM_FLAG_EQ, LBM_FLAG_OUT per cell, or none
 * (else LBM_E_INVAL).  Must precede lbm_init (LBM_E_STATE otherwise).  Synchronises the stream. */
int lbm_set_flags(lbm_t *h, const unsigned char *flags);

/* Initialise every cell, walls included, in both DDF buffers with the shifted equilibrium
 * f_i^eq(rho[n], u[n]) of eq (3) (R11) and reset the step counter.
 * rho: N floats, u: 3N floats (SoA).  lbm_init takes HOST pointers (copied, synchronous);
 * lbm_init_device takes DEVICE pointers read asynchronously on the handle's stream. */
int lbm_init(lbm_t *h, const float *rho, const float *u);
int lbm_init_device(lbm_t *h, const float *rho_dev, const float *u_dev);
/* The same with the fields of BASELINE configs[4] drawn cell by cell from a counter-based generator instead of read from
 * memory ("random-perturbed equilibrium init (rho = 1 + N(0, 1e-3), |u| <= 0.05 from seed)"): for boxes whose input
 * fields (16 bytes per cell) do not fit beside the DDFs -- the largest cubes of the bandwidth sweep.  The recipe
 * (splitmix64 of seed and cell index; rho = 1 + sqrt(3) 1e-3 (a0 + a1 + a2 + a3 - 2), u = (2 a - 1) 0.05 / sqrt(3), a_k
 * 22-bit uniforms) is stated in csrc/lbm_kernels.cuh and typed a second time, in numpy, in workloads.generated_fields.
 * Boxes without flagged cells only (LBM_E_STATE); not for the FP64-arithmetic formats (LBM_E_UNSUPPORTED).
 * Asynchronous on the handle's stream. */
int lbm_init_generated(lbm_t *h, unsigned long long seed);

/* Advance n >= 0 time steps: n launches of the fused stream-collide kernel (Listing 2,
 * PAPER.md:1014-1042; eqs (24)-(28)), alternating the two buffers.
 * Asynchronous on the handle's stream.  On boxes of up to 2^23 cells, where a launch costs as much as the kernel, runs of
 * 32 launches are captured into a CUDA graph once and replayed (same kernels, same arguments, same results);
 * lbm_set_graphs(h, 0) turns that off (for before / after measurements), lbm_set_graphs(h, 1) on again (default). */
int lbm_step(lbm_t *h, int n);
int lbm_set_graphs(lbm_t *h, int enable);

/* Density and velocity "after the steps done so far" = local moments of the current buffer (R12;
 * PAPER.md:428, 951-968); wall cells return the values given to lbm_init.  Either pointer may be NULL.
 * lbm_read_rho_u: HOST pointers, synchronises.  lbm_read_rho_u_device: DEVICE pointers, asynchronous. */
int lbm_read_rho_u(lbm_t *h, float *rho, float *u);
int lbm_read_rho_u_device(lbm_t *h, float *rho_dev, float *u_dev);
/* The same read-out in double, for the FP64-arithmetic formats (LBM_FP64, LBM_FP64_FP32; LBM_E_UNSUPPORTED for the
 * others): rho = HOST N doubles, u = HOST 3N doubles, either may be NULL.  Synchronises. */
int lbm_read_rho_u_f64(lbm_t *h, double *rho, double *u);

/* The same read-out at `count` selected cells (probes of a long run): cells = HOST array of cell indices n,
 * rho = HOST count floats, u = HOST 3*count floats (ux of all probes | uy | uz).  Synchronises. */
int lbm_read_rho_u_at(lbm_t *h, const long long *cells, int count, float *rho, float *u);

/* lbm_read_rho_u_at for callers that must not allocate device memory (code near a CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): same arguments, same results, but the scratch the read-out needs on the
 * device (the cell indices and the kernel's outputs, 24 bytes per probe) is a fixed array inside the library --
 * LBM_STATIC_PROBES_MAX probes, 96 KiB per GPU that loads the library, held until the process exits -- instead of the
 * handle's staging buffer.  The call makes no cudaMalloc / cudaFree and calls no allocating routine.
 * count > LBM_STATIC_PROBES_MAX: LBM_E_INVAL, nothing is done (use lbm_read_rho_u_at, or several calls).
 * ALL handles and threads of a process share the one array per GPU: calls that overlap on the GPU (two handles on
 * different streams, two host threads) race on it -- serialise them.  The array keeps the last call's contents; no call
 * depends on them.  HOST pointers; synchronises the handle's stream. */
#define LBM_STATIC_PROBES_MAX 4096
int lbm_read_rho_u_at_static(lbm_t *h, const long long *cells, int count, float *rho, float *u);

/* Copy direction i (0 <= i < q) of the current DDF buffer, as stored (N elements of 2, 4 or 8 bytes),
 * to a HOST pointer.  Synchronises.  For bit-level parity tests. */
int lbm_read_ddf(lbm_t *h, int i, void *out);

/* Block until all work queued on the handle's stream has finished. */
int lbm_sync(lbm_t *h);
/* Steps done since the last lbm_init. */
long long lbm_steps_done(const lbm_t *h);
/* Free the handle and everything the library allocated for it (not caller-bound memory). */
int lbm_destroy(lbm_t *h);

/* Message of the last failing call on this thread ("" if none). */
const char *lbm_last_error(void);

/* ---- storage-format codecs, exposed for bit-level parity tests and micro-benchmarks ------------
 * store(): FP32 -> 16-bit code; load(): code -> FP32.  ddf_format in
 * LBM_FP16S..LBM_FP16.  *_device variants take DEVICE pointers and run asynchronously on `cuda_stream`
 * (cudaStream_t as void*, NULL = default stream); the plain variants take HOST pointers. */
int lbm_codec_encode(int ddf_format, const float *x, unsigned short *codes, long long count);
int lbm_codec_decode(int ddf_format, const unsigned short *codes, float *x, long long count);
int lbm_codec_encode_device(int ddf_format, const float *x_dev, unsigned short *codes_dev, long long count,
                            void *cuda_stream);
int lbm_codec_decode_device(int ddf_format, const unsigned short *codes_dev, float *x_dev, long long count,
                            void *cuda_stream);

/* Device self-check of the staged kernel's pair converters against the scalar converters above: all 65 536 codes
 * through the pair decoders and all 2^32 FP32 bit patterns through the pair encoder, compared bit for bit (NaN
 * inputs excepted).  *mismatches (HOST) receives the number of differences (0 = identical).  Synchronous. */
int lbm_codec_pair_selftest(int ddf_format, long long *mismatches);

/* Device self-check of the staged kernel's velocity division (u = j / rho with one shared reciprocal, lbm_lattice.cuh
 * div3) against the IEEE division it replaces: about 10^8 (numerator, denominator) pairs incl. zero numerators of both
 * signs, compared bit for bit.  *mismatches (HOST) receives the number of differences (0 = identical).  Synchronous. */
int lbm_div_selftest(long long *mismatches);

/* ---- sizes -------------------------------------------------------------------------------------*/
/* bytes of ONE DDF buffer: q * N * sizeof(element), rounded up to a multiple of 256 */
long long lbm_ddf_buffer_bytes(int nx, int ny, int nz, int velset, int ddf_format);
/* algorithmic DRAM traffic of one cell update: 2*q*sizeof(element) + 1 flag byte */
long long lbm_bytes_per_cell(int velset, int ddf_format);
/* name of the stream_collide kernel variant the handle dispatches to (for profiles), "" before init */
const char *lbm_kernel_name(const lbm_t *h);
/* number of kernels this library has launched in this process (all handles), for bench accounting */
long long lbm_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* LBM_B200_H */
