/* oracle/oracle.h -- C ABI of the CPU oracle.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * `--impl reference` legs may load this library.  It shares no code with the CUDA path under
 * paper_2112_08926_b200/ (no common header, table, constant generator or helper): everything here is
 * typed in from the paper (/root/reference/PAPER.md, cited per function as PAPER.md:<line>) and from
 * the readings listed in DESIGN.md section 3.
 *
 * The oracle is deliberately plain and slow: value tables + binary search for the codecs, one
 * triple loop per time step for the LBM, no blocking, fusion or reordering beyond what the cited
 * passage states.
 */
#ifndef LBM_ORACLE_H
#define LBM_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* storage formats (same numbering as the product header, typed in independently) */
enum { ORC_FP32 = 0, ORC_FP16S = 1, ORC_FP16C = 2, ORC_P16_0S = 3, ORC_P16_1S = 4, ORC_P16_2C = 5,
       ORC_FP16 = 6, ORC_FP64 = 7 /* oracle only: raw doubles, needs arith = 1 */ };
enum { ORC_ARITH_F32 = 0, ORC_ARITH_F64 = 1 };
enum { ORC_BGK = 0, ORC_TRT = 1 /* textbook two-relaxation-time operator, NOT defined by the paper (R13) */ };
enum { ORC_FLAG_WALL = 0x01, ORC_FLAG_EQ = 0x02 /* equilibrium boundary cell: keeps its init DDFs (R15) */,
       ORC_FLAG_OUT = 0x04 /* zero-gradient outflow cell: equilibrium of its upstream (x - 1) neighbour's rho, u (R18) */ };

/* ---- codecs (16-bit formats only, fmt in 1..6) ------------------------------------------------ */
/* unscaled table value V(mag) of the 15-bit magnitude field, as a double (Inf/NaN for FP16 e=31) */
double orc_table_value(int fmt, unsigned mag);
/* power-of-two scale the format applies on store (load applies 1/scale): 2^15, 2^7 or 1 */
double orc_scale(int fmt);
/* load(): code -> FP32 value the collision sees (table value / scale, exact in FP32) */
int orc_decode(int fmt, const uint16_t *codes, float *out, long n);
/* store(): FP32 value -> code (rule U / IEEE RNE, see codecs.cpp) */
int orc_encode(int fmt, const float *x, uint16_t *out, long n);

/* ---- LBM -------------------------------------------------------------------------------------- */
typedef struct orc_sim orc_sim;
orc_sim *orc_create(int nx, int ny, int nz, int velset, int fmt, int arith, double tau, const double force[3]);
void orc_destroy(orc_sim *s);
/* collision operator (default ORC_BGK) and, for ORC_TRT, the magic parameter Lambda (default 3/16); before orc_step */
int  orc_set_collision(orc_sim *s, int collision, double lambda);
/* DDF-shifting on (default) / off: off = eqs (19)-(23), the paper's negative control (R17); before orc_init */
int  orc_set_shifting(orc_sim *s, int on);
int  orc_set_flags(orc_sim *s, const uint8_t *flags);                 /* N bytes */
int  orc_init(orc_sim *s, const float *rho, const float *u);         /* N, 3N (SoA) */
int  orc_init_f64(orc_sim *s, const double *rho, const double *u);   /* arith = f64 only */
int  orc_step(orc_sim *s, int n);
int  orc_read_rho_u(orc_sim *s, float *rho, float *u);
int  orc_read_rho_u_f64(orc_sim *s, double *rho, double *u);
/* raw stored DDFs of the current buffer, direction i: N elements of 2 / 4 / 8 bytes */
int  orc_read_ddf(orc_sim *s, int i, void *out);
/* sum over all cells and directions of the decoded shifted DDFs, accumulated in long double */
double orc_sum_ddf(orc_sim *s);
int  orc_set_threads(int n);                                          /* OpenMP threads; returns the count in use */
/* velocity-set tables, for the tests: c[q][3], w[q] (double), opp[q] */
int  orc_velocity_set(int velset, int *c, double *w, int *opp);
/* shifted equilibrium of one cell in double or float arithmetic (R7), for the tests */
int  orc_equilibrium(int velset, int arith, double rho, double ux, double uy, double uz, double *feq);

#ifdef __cplusplus
}
#endif
#endif
