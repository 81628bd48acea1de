/* ozfft_oracle.h -- C interface of the CPU oracle (TEST INFRASTRUCTURE, not product).
 * See ozfft_oracle.c for what each function follows in PAPER.md. 128-bit values
 * cross the boundary as {lo, hi} uint64 pairs (two's complement). */
#ifndef OZFFT_ORACLE_H
#define OZFFT_ORACLE_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif
void oz_init(void);
void oz_select_modset(int which);            /* 0 = Rev-34, 1 = Rev-33 (regression) */
int oz_num_moduli(void);
int oz_modulus(int k);
void oz_get_M(uint64_t out[2]);
void oz_get_u(int k, uint64_t out[2]);
int oz_get_t(int k);
uint64_t oz_get_w(int k);
int oz_num_slices(void);
int oz_get_uslice(int k, int s);
int oz_get_wslice(int k, int s);
void oz_twiddle(int t, int64_t *c, int64_t *s);
uint64_t oz_twiddle_checksum(void);
long oz_capacity_violations(void);
void oz_reset_capacity_violations(void);
int oz_column_top(const uint64_t *bits, int n, int *Tmax);
int64_t oz_quantise(uint64_t bits, int Tmax);
uint64_t oz_pack(uint64_t lo, uint64_t hi, int g);
void oz_residues(uint64_t lo, uint64_t hi, int *v);
void oz_crt(const int *v, int route, uint64_t out[2]); /* 0 Alg.2, 1 plain, 2 Garner, 3/4 Alg.2 one-sided upper/lower */
void oz_phaseA(const int *v, int32_t *P, int32_t *Z);
void oz_kulisch_deposit(const int32_t *P, int S, uint32_t *W);
int oz_stage(int K, int Rr, const uint64_t *x, const int *tidx, int sign, uint64_t *y, int route);
void oz_factor(int n, int *p, int *q);
int oz_fft1d(int n, int batch, int sign, const double *in, double *out, int route);
int oz_fft3d(int nx, int ny, int nz, int sign, const double *in, double *out, int route);
int oz_fft1d_strided(int n, int sign, const double *in, long in_stride, double *out, long out_stride, int route);
double oz_relerr_1d_f128(int n, int batch, int sign, const double *x, const double *y);
double oz_relerr_3d_f128(int nx, int ny, int nz, int sign, const double *x, const long *idx, int nsamp, const double *ysamp);
int oz_num_threads(void);
#ifdef __cplusplus
}
#endif
#endif
