/*
 * ozfft_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * Plain, slow, obviously-correct CPU oracle for the emulated-fp64 FFT of
 * arxiv/paper_2606_23698 ("FP8 is All You Need, Part 2").  It shares no code
 * with the CUDA path under paper_2606_23698_b200/csrc and neither includes the
 * other.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load it.
 *
 * What it computes (all citations are PAPER.md lines; readings S1..S19 are
 * listed in DESIGN.md):
 *   - Rev-34 modulus set, M, CRT idempotents u_k, byte slices, lift
 *     fractions w_k.
 *   - per-column power-of-two quantisation to 53-bit signed integers
 *     ("round(s_A A)", 218 shared column scale; reading S2-S4).
 *   - one Bailey stage as an exact integer DFT-by-matrix in two routes that
 *     must agree: (a) the plain definition in __int128; (b) the paper's
 *     step-by-step residue route: residues mod m_i, complex Karatsuba D,E,F
 *     (PAPER.md:113, 225-228, 275), canonicalise, Phase A slice sums
 *     (Eq. 17-20), Algorithm 2 Kulisch radix-28 deposits,
 *     fractional lift and two-sided correction.
 *   - the single correctly-rounded pack to fp64, integer only.
 *   - 1-D Bailey six-step with twiddle-fused second stage (PAPER.md:115-122,
 *     210-214 Eq. 6) and the 3-D transform as three axis passes.
 *   - an O(N^2) DFT in __float128 for accuracy pins.
 *
 * Pins: tests/test_oracle_*.py (constants the paper prints, Python big-int
 * CRT, Fraction-rounded pack, mpmath DFT, closed forms, symmetries).
 * Parity unpinned: the "10 units above a rounding boundary" figure of
 * PAPER.md:370 (not reproducible without verify.py; the invariant it
 * illustrates is tested instead).
 */
#include "ozfft_oracle.h"

#include <math.h>
#include <quadmath.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef __int128 i128;
typedef unsigned __int128 u128;

#define R_MOD 12
#define MAXS 16
#define SFRAC 6
#define FBITS 48
#define TABLE_N 1024

/* ---------------------------------------------------------------- modsets */

typedef struct {
    int m[R_MOD];
    u128 M, Mhalf;
    u128 u[R_MOD];
    int t[R_MOD];             /* (M/m_k)^-1 mod m_k */
    int S;                    /* byte slices of u_k: ceil(bitlen(M)/8) */
    uint8_t uslice[R_MOD][MAXS];
    uint64_t w[R_MOD];        /* round(2^48 u_k / M) */
    uint8_t wslice[R_MOD][SFRAC];
    int pow256[R_MOD][8];     /* 2^(8k) mod m_i, k<7 */
} modset_t;

/* PAPER.md:101 (Rev-34) and PAPER.md:111 (Rev-33 had 509,503,499). */
static const int REV34[R_MOD] = {2039, 2029, 2027, 1089, 1024, 961, 841, 625, 529, 511, 491, 487};
static const int REV33[R_MOD] = {509, 503, 499, 1089, 1024, 961, 841, 625, 529, 511, 491, 487};

static modset_t g_sets[2];
static int residue_i64(const modset_t *ms, int k, __int128 x);
static int g_cur = 0;
static int g_init = 0;
static long g_capacity_violations = 0;

static int bitlen128(u128 a) {
    int n = 0;
    while (a) { n++; a >>= 1; }
    return n;
}

static int inv_mod(int a, int m) { /* brute force: m < 2048 */
    a %= m;
    for (int x = 1; x < m; x++)
        if ((a * x) % m == 1) return x;
    return 0;
}

static void build_set(modset_t *ms, const int *mods) {
    memcpy(ms->m, mods, sizeof(int) * R_MOD);
    ms->M = 1;
    for (int k = 0; k < R_MOD; k++) ms->M *= (u128)mods[k];
    ms->Mhalf = ms->M / 2;
    ms->S = (bitlen128(ms->M) + 7) / 8;
    for (int k = 0; k < R_MOD; k++) {
        u128 Mk = ms->M / (u128)mods[k];
        int r = (int)(Mk % (u128)mods[k]);
        ms->t[k] = inv_mod(r, mods[k]);
        ms->u[k] = Mk * (u128)ms->t[k]; /* Eq. 17; < M */
        for (int s = 0; s < MAXS; s++) ms->uslice[k][s] = (uint8_t)((ms->u[k] >> (8 * s)) & 0xFF);
        /* w_k = floor(2^48 u_k / M + 1/2) by binary long division (reading S10) */
        u128 rem = ms->u[k];
        uint64_t w = 0;
        for (int b = 0; b < FBITS; b++) {
            rem <<= 1;
            w <<= 1;
            if (rem >= ms->M) { rem -= ms->M; w |= 1; }
        }
        if (2 * rem >= ms->M) w += 1;
        ms->w[k] = w;
        for (int s = 0; s < SFRAC; s++) ms->wslice[k][s] = (uint8_t)((w >> (8 * s)) & 0xFF);
        int p = 1 % mods[k];
        for (int b = 0; b < 8; b++) { ms->pow256[k][b] = p; p = (p * 256) % mods[k]; }
    }
}

/* ---------------------------------------------------------------- twiddles */

static int64_t g_tc[TABLE_N], g_ts[TABLE_N];
static int g_tcres[2][R_MOD][TABLE_N], g_tsres[2][R_MOD][TABLE_N]; /* canonical residues of the table */

/* Reading S5: RN(2^53 cos), RN(2^53 sin) of 2*pi*t/1024 from quad precision on
 * the first octant, the rest by symmetry. */
static void build_twiddles(void) {
    const __float128 two53 = 9007199254740992.0Q;
    for (int t = 0; t <= 128; t++) {
        __float128 th = 2.0Q * M_PIq * (__float128)t / 1024.0Q;
        g_tc[t] = (int64_t)llrintq(two53 * cosq(th));
        g_ts[t] = (int64_t)llrintq(two53 * sinq(th));
    }
    for (int t = 129; t <= 256; t++) { g_tc[t] = g_ts[256 - t]; g_ts[t] = g_tc[256 - t]; }
    for (int t = 257; t <= 512; t++) { g_tc[t] = -g_tc[512 - t]; g_ts[t] = g_ts[512 - t]; }
    for (int t = 513; t < 1024; t++) { g_tc[t] = g_tc[1024 - t]; g_ts[t] = -g_ts[1024 - t]; }
}

void oz_init(void) {
    if (g_init) return;
    build_set(&g_sets[0], REV34);
    build_set(&g_sets[1], REV33);
    build_twiddles();
    for (int w = 0; w < 2; w++)
        for (int i = 0; i < R_MOD; i++)
            for (int t = 0; t < TABLE_N; t++) {
                g_tcres[w][i][t] = residue_i64(&g_sets[w], i, g_tc[t]);
                g_tsres[w][i][t] = residue_i64(&g_sets[w], i, g_ts[t]);
            }
    g_init = 1;
}

void oz_select_modset(int which) { oz_init(); g_cur = which ? 1 : 0; }
static const modset_t *cur(void) { oz_init(); return &g_sets[g_cur]; }

/* ------------------------------------------------------- constant getters */

static void split128(u128 v, uint64_t out[2]) { out[0] = (uint64_t)v; out[1] = (uint64_t)(v >> 64); }

int oz_num_moduli(void) { return R_MOD; }
int oz_modulus(int k) { return cur()->m[k]; }
void oz_get_M(uint64_t out[2]) { split128(cur()->M, out); }
void oz_get_u(int k, uint64_t out[2]) { split128(cur()->u[k], out); }
int oz_get_t(int k) { return cur()->t[k]; }
uint64_t oz_get_w(int k) { return cur()->w[k]; }
int oz_num_slices(void) { return cur()->S; }
int oz_get_uslice(int k, int s) { return cur()->uslice[k][s]; }
int oz_get_wslice(int k, int s) { return cur()->wslice[k][s]; }
void oz_twiddle(int t, int64_t *c, int64_t *s) { oz_init(); *c = g_tc[t & (TABLE_N - 1)]; *s = g_ts[t & (TABLE_N - 1)]; }
long oz_capacity_violations(void) { return g_capacity_violations; }
void oz_reset_capacity_violations(void) { g_capacity_violations = 0; }

uint64_t oz_twiddle_checksum(void) { /* FNV-1a over (c,s) little-endian */
    oz_init();
    uint64_t h = 1469598103934665603ULL;
    for (int t = 0; t < TABLE_N; t++) {
        int64_t v[2] = {g_tc[t], g_ts[t]};
        const unsigned char *p = (const unsigned char *)v;
        for (int i = 0; i < 16; i++) { h ^= p[i]; h *= 1099511628211ULL; }
    }
    return h;
}

/* ------------------------------------------------------------ quantisation */

/* Appendix A.1: decode; returns 0 zero, 1 finite nonzero, 2 non-finite. */
static int decode(uint64_t b, int *sgn, uint64_t *m, int *E) {
    *sgn = (int)(b >> 63);
    int ef = (int)((b >> 52) & 0x7FF);
    uint64_t fr = b & ((1ULL << 52) - 1);
    if (ef == 0x7FF) return 2;
    if (ef == 0) { *m = fr; *E = -1074; }
    else { *m = fr | (1ULL << 52); *E = ef - 1075; }
    return *m ? 1 : 0;
}

static int bitlen64(uint64_t a) { return a ? 64 - __builtin_clzll(a) : 0; }

/* A.2: floor(log2 |x|) over the nonzero entries; returns 0 all-zero, 1 ok, 2 non-finite */
int oz_column_top(const uint64_t *bits, int n, int *Tmax) {
    int have = 0, T = 0;
    for (int i = 0; i < n; i++) {
        int s, E; uint64_t m;
        int c = decode(bits[i], &s, &m, &E);
        if (c == 2) return 2;
        if (c == 0) continue;
        int Ti = E + bitlen64(m) - 1;
        if (!have || Ti > T) { T = Ti; have = 1; }
    }
    *Tmax = T;
    return have;
}

/* A.3: RNE(x * 2^(52 - Tmax)) with integer shifts only. */
int64_t oz_quantise(uint64_t b, int Tmax) {
    int s, E; uint64_t m;
    if (decode(b, &s, &m, &E) != 1) return 0;
    int sh = Tmax - 52 - E; /* x*2^(52-Tmax) = m * 2^-sh */
    uint64_t q;
    if (sh <= 0) q = m << (-sh);
    else if (sh >= 64) q = 0;
    else {
        q = m >> sh;
        uint64_t rem = m & ((1ULL << sh) - 1), half = 1ULL << (sh - 1);
        if (rem > half || (rem == half && (q & 1))) q++;
    }
    return s ? -(int64_t)q : (int64_t)q;
}

/* --------------------------------------------------------------------- pack */

/* A.6: RNE_fp64(R * 2^-g), integer only. */
static uint64_t pack128(i128 R, int g) {
    uint64_t sgn = R < 0 ? 1ULL << 63 : 0;
    u128 a = R < 0 ? (u128)(-R) : (u128)R;
    if (a == 0) return 0;
    int L = bitlen128(a);
    int X = L - 1 - g;
    if (X >= -1022) {
        uint64_t q;
        if (L > 53) {
            int d = L - 53;
            q = (uint64_t)(a >> d);
            u128 rem = a & (((u128)1 << d) - 1), half = (u128)1 << (d - 1);
            if (rem > half || (rem == half && (q & 1))) q++;
            if (q == (1ULL << 53)) { q >>= 1; X++; }
        } else q = (uint64_t)(a << (53 - L));
        if (X > 1023) return sgn | 0x7FF0000000000000ULL;
        return sgn | ((uint64_t)(X + 1023) << 52) | (q - (1ULL << 52));
    }
    int d = g - 1074; /* grid unit 2^-1074: q = RNE(a * 2^-d) */
    uint64_t q;
    if (d <= 0) q = (uint64_t)(a << (-d));
    else if (d > 127) q = 0;
    else {
        q = (uint64_t)(a >> d);
        u128 rem = a & (((u128)1 << d) - 1), half = (u128)1 << (d - 1);
        if (rem > half || (rem == half && (q & 1))) q++;
    }
    return sgn | q;
}

uint64_t oz_pack(uint64_t lo, uint64_t hi, int g) {
    i128 R = (i128)(((u128)hi << 64) | lo);
    return pack128(R, g);
}

/* ---------------------------------------------------------------- residues */

/* A.4 / PAPER.md:190: byte-plane route, canonical residue of a signed integer. */
static int residue_i64(const modset_t *ms, int k, i128 x) {
    int neg = x < 0;
    u128 a = neg ? (u128)(-x) : (u128)x;
    int m = ms->m[k];
    long acc = 0;
    int p = 1 % m;
    while (a) { /* sum_b byte_b * (256^b mod m) */
        acc += (long)(a & 0xFF) * p;
        p = (p * 256) % m;
        a >>= 8;
    }
    int r = (int)(acc % m);
    return (neg && r) ? m - r : r;
}

void oz_residues(uint64_t lo, uint64_t hi, int *v) {
    const modset_t *ms = cur();
    i128 C = (i128)(((u128)hi << 64) | lo);
    for (int k = 0; k < R_MOD; k++) v[k] = residue_i64(ms, k, C);
}

/* --------------------------------------------------- CRT, three routes */

/* Phase A: P_s = sum_k v_k u_k^(s), Z_t = sum_k v_k w_k^(t). */
static void phaseA(const modset_t *ms, const int *v, int32_t *P, int32_t *Z) {
    for (int s = 0; s < ms->S; s++) {
        long a = 0;
        for (int k = 0; k < R_MOD; k++) a += (long)v[k] * ms->uslice[k][s];
        P[s] = (int32_t)a;
    }
    for (int t = 0; t < SFRAC; t++) {
        long a = 0;
        for (int k = 0; k < R_MOD; k++) a += (long)v[k] * ms->wslice[k][t];
        Z[t] = (int32_t)a;
    }
}

/* Algorithm 2 lines 1-5 (Appendix A.7): biased deposits into
 * six radix-28 words, one carry sweep.  W holds the biased total. */
void oz_kulisch_deposit(const int32_t *P, int S, uint32_t *W) {
    for (int w = 0; w < 6; w++) W[w] = 0;
    for (int s = 0; s < S; s++) {
        uint32_t d = (uint32_t)(P[s] + (1 << 23)); /* biased, 24-bit non-negative */
        int w0 = (8 * s) / 28, o = (8 * s) % 28;
        W[w0] += (d << o) & 0x0FFFFFFFu;
        if (w0 + 1 < 6) W[w0 + 1] += (o ? d >> (28 - o) : 0);
    }
    for (int w = 0; w < 5; w++) { uint32_t c = W[w] >> 28; W[w] &= 0x0FFFFFFFu; W[w + 1] += c; }
}

/* Algorithm 2 lines 5-8: subtract bias and zhat*M, centre.  sides=1 or 2
 * reproduces the one-sided defect the paper describes. */
static int64_t zhat_of(const int32_t *Z) { /* A.8: floor(2^-48 z_acc + 1/2), signed */
    int64_t zacc = 0;
    for (int t = 0; t < SFRAC; t++) zacc += (int64_t)Z[t] * ((int64_t)1 << (8 * t));
    return (zacc + ((int64_t)1 << (FBITS - 1))) >> FBITS;
}

/* sides: bit0 = apply "R >= M/2 -> R - M", bit1 = apply "R < -M/2 -> R + M" */
static i128 centre(const modset_t *ms, i128 R, int sides) {
    i128 Mh = (i128)ms->Mhalf, Mi = (i128)ms->M;
    if ((sides & 1) && R >= Mh) R -= Mi;
    if ((sides & 2) && R < -Mh) R += Mi;
    return R;
}

static i128 alg2_finish(const modset_t *ms, const uint32_t *W, int S, const int32_t *Z, int sides) {
    int64_t zhat = zhat_of(Z);
    int64_t V[6];
    for (int w = 0; w < 6; w++) V[w] = W[w];
    for (int s = 0; s < S; s++) { /* B_tot = sum_s 2^23 * 256^s */
        int bit = 8 * s + 23;
        V[bit / 28] -= (int64_t)1 << (bit % 28);
    }
    for (int w = 0; w < 5; w++) { /* zhat * M in radix 28 */
        int64_t Mw = (int64_t)((ms->M >> (28 * w)) & 0x0FFFFFFFu);
        V[w] -= zhat * Mw;
    }
    for (int w = 0; w < 5; w++) { /* signed carry normalise */
        int64_t c = V[w] >> 28;
        V[w] -= c << 28;
        V[w + 1] += c;
    }
    /* |R| < 2^119, so the top word is pure sign and the value is its low 128 bits */
    u128 lo = 0;
    for (int w = 0; w < 5; w++) lo += (u128)(uint64_t)V[w] << (28 * w);
    if (!(V[5] == 0 || V[5] == -1)) g_capacity_violations++;
    return centre(ms, (i128)lo, sides);
}

static i128 crt_alg2(const modset_t *ms, const int *v, int sides) {
    int32_t P[MAXS], Z[SFRAC];
    uint32_t W[6];
    phaseA(ms, v, P, Z);
    oz_kulisch_deposit(P, ms->S, W);
    i128 R = alg2_finish(ms, W, ms->S, Z, sides);
    /* Appendix A.7 cross-check: the same value by wrapping 128-bit arithmetic */
    u128 chk = 0;
    for (int s = 0; s < ms->S; s++) chk += (u128)(i128)P[s] << (8 * s);
    chk -= (u128)(i128)zhat_of(Z) * ms->M;
    if (centre(ms, (i128)chk, sides) != R) g_capacity_violations += 1000000;
    return R;
}

/* Plain definition: sum v_k u_k mod M, centred to [-M/2, M/2). */
static i128 crt_plain(const modset_t *ms, const int *v) {
    u128 acc = 0;
    for (int k = 0; k < R_MOD; k++) {
        u128 term = (ms->M / (u128)ms->m[k]) * (u128)((v[k] * ms->t[k]) % ms->m[k]); /* < M */
        acc += term;
        if (acc >= ms->M) acc -= ms->M;
    }
    i128 R = (i128)acc;
    if (acc >= ms->Mhalf) R -= (i128)ms->M;
    return R;
}

/* Garner mixed radix, independent third route. */
static i128 crt_garner(const modset_t *ms, const int *v) {
    int a[R_MOD];
    for (int k = 0; k < R_MOD; k++) {
        int m = ms->m[k];
        long x = v[k] % m;
        for (int j = 0; j < k; j++) { /* x = (x - a_j) * m_j^-1 mod m_k */
            x = ((x - a[j]) % m + m) % m;
            x = (x * inv_mod(ms->m[j] % m, m)) % m;
        }
        a[k] = (int)x;
    }
    u128 acc = 0, base = 1;
    for (int k = 0; k < R_MOD; k++) { acc += base * (u128)a[k]; base *= (u128)ms->m[k]; }
    i128 R = (i128)acc;
    if (acc >= ms->Mhalf) R -= (i128)ms->M;
    return R;
}

void oz_crt(const int *v, int route, uint64_t out[2]) {
    const modset_t *ms = cur();
    i128 R;
    switch (route) {
    case 0: R = crt_alg2(ms, v, 3); break;
    case 1: R = crt_plain(ms, v); break;
    case 2: R = crt_garner(ms, v); break;
    case 3: R = crt_alg2(ms, v, 1); break;  /* one-sided, upper test only (defective by design) */
    default: R = crt_alg2(ms, v, 2); break; /* one-sided, lower test only (defective by design) */
    }
    split128((u128)R, out);
}

void oz_phaseA(const int *v, int32_t *P, int32_t *Z) { phaseA(cur(), v, P, Z); }

/* ---------------------------------------------------------------- one stage */

/* Exact integer stage (SURVEY 8(c) definition):
 *   x: K complex fp64 (bit patterns, re/im interleaved); tidx[k*K+j]: index of
 *   the coefficient in the omega_1024 table; sign: -1 forward, +1 inverse;
 *   y: Rr complex fp64 bit patterns.  route 0: __int128 definition;
 *   route 1: residue/Karatsuba/Phase A/Algorithm 2; route 2: both, asserted equal. */
int oz_stage(int K, int Rr, const uint64_t *x, const int *tidx, int sign, uint64_t *y, int route) {
    const modset_t *ms = cur();
    int Tmax, st = oz_column_top(x, 2 * K, &Tmax);
    if (st == 2) { for (int i = 0; i < 2 * Rr; i++) y[i] = 0x7FF8000000000000ULL; return 0; }
    if (st == 0) { for (int i = 0; i < 2 * Rr; i++) y[i] = 0; return 0; }
    int64_t xr[32], xi[32];
    for (int j = 0; j < K; j++) { xr[j] = oz_quantise(x[2 * j], Tmax); xi[j] = oz_quantise(x[2 * j + 1], Tmax); }
    int g = 53 + (52 - Tmax);
    int bad = 0;
    int xres[R_MOD][32][2];
    if (route != 0)
        for (int i = 0; i < R_MOD; i++)
            for (int j = 0; j < K; j++) { xres[i][j][0] = residue_i64(ms, i, xr[j]); xres[i][j][1] = residue_i64(ms, i, xi[j]); }
    for (int k = 0; k < Rr; k++) {
        i128 Rd = 0, Id = 0;
        if (route != 1) {
            for (int j = 0; j < K; j++) {
                int64_t ar = g_tc[tidx[k * K + j]], ai = sign * g_ts[tidx[k * K + j]];
                Rd += (i128)ar * xr[j] - (i128)ai * xi[j];
                Id += (i128)ar * xi[j] + (i128)ai * xr[j];
            }
            i128 Mh = (i128)ms->Mhalf;
            if (Rd >= Mh || Rd < -Mh || Id >= Mh || Id < -Mh) g_capacity_violations++;
        }
        i128 Rp = 0, Ip = 0;
        if (route != 0) {
            int vr[R_MOD], vi[R_MOD];
            for (int i = 0; i < R_MOD; i++) {
                int m = ms->m[i];
                long D = 0, E = 0, F = 0;
                for (int j = 0; j < K; j++) {
                    int t = tidx[k * K + j];
                    int a_r = g_tcres[g_cur][i][t];
                    int a_i = sign > 0 ? g_tsres[g_cur][i][t] : (m - g_tsres[g_cur][i][t]) % m;
                    int x_r = xres[i][j][0], x_i = xres[i][j][1];
                    int a_s = a_r + a_i; if (a_s >= m) a_s -= m; /* Karatsuba operands */
                    int x_s = x_r + x_i; if (x_s >= m) x_s -= m;
                    D += (long)a_r * x_r; E += (long)a_i * x_i; F += (long)a_s * x_s;
                }
                int d = (int)(D % m), e = (int)(E % m), f = (int)(F % m);
                int re = d - e, im = f - d - e;
                re %= m; if (re < 0) re += m;             /* canonicalise */
                im %= m; if (im < 0) im += m;
                vr[i] = re; vi[i] = im;
            }
            Rp = crt_alg2(ms, vr, 3);
            Ip = crt_alg2(ms, vi, 3);
            if (route == 2 && (Rp != Rd || Ip != Id)) bad++;
        }
        if (route == 1) { Rd = Rp; Id = Ip; }
        y[2 * k] = pack128(Rd, g);
        y[2 * k + 1] = pack128(Id, g);
    }
    return bad;
}

/* ------------------------------------------------------------------ 1-D FFT */

/* Reading S7: n <= 32 single stage; else q = 32 first stage, p = n/32 second. */
void oz_factor(int n, int *p, int *q) { if (n <= 32) { *p = 1; *q = n; } else { *q = 32; *p = n / 32; } }

/* PAPER.md:115-122 + Eq. 6.  x, y: n complex (bit patterns),
 * stride in complex elements.  Returns the number of route mismatches. */
static int fft1d(int n, int sign, const uint64_t *x, long xs, uint64_t *y, long ys, int route) {
    int p, q;
    oz_factor(n, &p, &q);
    int bad = 0;
    uint64_t col[64], res[64];
    int tidx[32 * 32];
    if (p == 1) {
        for (int j = 0; j < n; j++) { col[2 * j] = x[2 * j * xs]; col[2 * j + 1] = x[2 * j * xs + 1]; }
        for (int k = 0; k < n; k++)
            for (int j = 0; j < n; j++) tidx[k * n + j] = (int)(((long)(TABLE_N / n) * j * k) % TABLE_N);
        bad += oz_stage(n, n, col, tidx, sign, res, route);
        for (int k = 0; k < n; k++) { y[2 * k * ys] = res[2 * k]; y[2 * k * ys + 1] = res[2 * k + 1]; }
        return bad;
    }
    uint64_t *Y1 = (uint64_t *)malloc(sizeof(uint64_t) * 2 * n); /* Y'[j1][k2] */
    for (int k2 = 0; k2 < q; k2++)
        for (int j2 = 0; j2 < q; j2++) tidx[k2 * q + j2] = (int)(((long)(TABLE_N / q) * j2 * k2) % TABLE_N);
    for (int j1 = 0; j1 < p; j1++) { /* stage 1: columns over j2 at fixed j1, matrix F_q */
        for (int j2 = 0; j2 < q; j2++) {
            long j = j1 + (long)p * j2;
            col[2 * j2] = x[2 * j * xs]; col[2 * j2 + 1] = x[2 * j * xs + 1];
        }
        bad += oz_stage(q, q, col, tidx, sign, res, route);
        for (int k2 = 0; k2 < q; k2++) { Y1[2 * (j1 * q + k2)] = res[2 * k2]; Y1[2 * (j1 * q + k2) + 1] = res[2 * k2 + 1]; }
    }
    for (int k2 = 0; k2 < q; k2++) { /* stage 2: columns over j1 at fixed k2, fused matrix F_p^(k2) */
        for (int j1 = 0; j1 < p; j1++) { col[2 * j1] = Y1[2 * (j1 * q + k2)]; col[2 * j1 + 1] = Y1[2 * (j1 * q + k2) + 1]; }
        for (int k1 = 0; k1 < p; k1++)
            for (int j1 = 0; j1 < p; j1++)
                tidx[k1 * p + j1] = (int)(((long)(TABLE_N / n) * j1 * (k2 + (long)q * k1)) % TABLE_N);
        bad += oz_stage(p, p, col, tidx, sign, res, route);
        for (int k1 = 0; k1 < p; k1++) {
            long k = k2 + (long)q * k1;
            y[2 * k * ys] = res[2 * k1]; y[2 * k * ys + 1] = res[2 * k1 + 1];
        }
    }
    free(Y1);
    return bad;
}

int oz_fft1d(int n, int batch, int sign, const double *in, double *out, int route) {
    oz_init();
    int bad = 0;
#pragma omp parallel for reduction(+ : bad) schedule(static)
    for (int b = 0; b < batch; b++)
        bad += fft1d(n, sign, (const uint64_t *)in + 2L * n * b, 1, (uint64_t *)out + 2L * n * b, 1, route);
    return bad;
}

/* 3-D: passes over z, then y, then x (reading S8); row-major, z fastest. */
int oz_fft3d(int nx, int ny, int nz, int sign, const double *in, double *out, int route) {
    oz_init();
    long tot = (long)nx * ny * nz;
    uint64_t *A = (uint64_t *)malloc(sizeof(uint64_t) * 2 * tot);
    uint64_t *B = (uint64_t *)out;
    int bad = 0;
    /* z pass: in -> A */
#pragma omp parallel for reduction(+ : bad) schedule(static)
    for (long r = 0; r < (long)nx * ny; r++)
        bad += fft1d(nz, sign, (const uint64_t *)in + 2 * r * nz, 1, A + 2 * r * nz, 1, route);
    /* y pass: A -> B */
#pragma omp parallel for reduction(+ : bad) schedule(static)
    for (long r = 0; r < (long)nx * nz; r++) {
        long x = r / nz, z = r % nz;
        long base = (x * ny) * nz + z;
        bad += fft1d(ny, sign, A + 2 * base, nz, B + 2 * base, nz, route);
    }
    /* x pass: B -> A, then copy */
#pragma omp parallel for reduction(+ : bad) schedule(static)
    for (long r = 0; r < (long)ny * nz; r++)
        bad += fft1d(nx, sign, B + 2 * r, (long)ny * nz, A + 2 * r, (long)ny * nz, route);
    memcpy(out, A, sizeof(uint64_t) * 2 * tot);
    free(A);
    return bad;
}

/* one pencil of a 3-D array along one axis (for the sampled-pencil check P13) */
int oz_fft1d_strided(int n, int sign, const double *in, long in_stride, double *out, long out_stride, int route) {
    oz_init();
    return fft1d(n, sign, (const uint64_t *)in, in_stride, (uint64_t *)out, out_stride, route);
}

/* ------------------------------------------------- __float128 reference DFT */

/* ||y - DFT(x)||_2 / ||DFT(x)||_2 with the O(n^2) DFT in __float128. */
double oz_relerr_1d_f128(int n, int batch, int sign, const double *x, const double *y) {
    __float128 *wr = (__float128 *)malloc(sizeof(__float128) * n), *wi = (__float128 *)malloc(sizeof(__float128) * n);
    for (int t = 0; t < n; t++) {
        __float128 th = 2.0Q * M_PIq * (__float128)t / (__float128)n;
        wr[t] = cosq(th); wi[t] = (__float128)sign * sinq(th);
    }
    __float128 num = 0, den = 0;
#pragma omp parallel for reduction(+ : num, den) schedule(static)
    for (long bk = 0; bk < (long)batch * n; bk++) {
        long b = bk / n; int k = (int)(bk % n);
        const double *xb = x + 2L * n * b;
        __float128 sr = 0, si = 0;
        for (int j = 0; j < n; j++) {
            int t = (int)(((long)j * k) % n);
            __float128 a = xb[2 * j], c = xb[2 * j + 1];
            sr += a * wr[t] - c * wi[t];
            si += a * wi[t] + c * wr[t];
        }
        __float128 dr = (__float128)y[2 * bk] - sr, di = (__float128)y[2 * bk + 1] - si;
        num += dr * dr + di * di;
        den += sr * sr + si * si;
    }
    free(wr); free(wi);
    return (double)sqrtq(num / den);
}

/* Same for nsamp sampled outputs idx[] (flat row-major) of a 3-D transform. */
double oz_relerr_3d_f128(int nx, int ny, int nz, int sign, const double *x, const long *idx, int nsamp, const double *ysamp) {
    __float128 num = 0, den = 0;
#pragma omp parallel for reduction(+ : num, den) schedule(dynamic)
    for (int s = 0; s < nsamp; s++) {
        long f = idx[s];
        int kz = (int)(f % nz), ky = (int)((f / nz) % ny), kx = (int)(f / ((long)nz * ny));
        __float128 *zr = (__float128 *)malloc(sizeof(__float128) * nz), *zi = (__float128 *)malloc(sizeof(__float128) * nz);
        __float128 *yr = (__float128 *)malloc(sizeof(__float128) * ny), *yi = (__float128 *)malloc(sizeof(__float128) * ny);
        for (int t = 0; t < nz; t++) { __float128 th = 2.0Q * M_PIq * (__float128)(((long)t * kz) % nz) / nz; zr[t] = cosq(th); zi[t] = sign * sinq(th); }
        for (int t = 0; t < ny; t++) { __float128 th = 2.0Q * M_PIq * (__float128)(((long)t * ky) % ny) / ny; yr[t] = cosq(th); yi[t] = sign * sinq(th); }
        __float128 sr = 0, si = 0;
        for (int ix = 0; ix < nx; ix++) {
            __float128 th = 2.0Q * M_PIq * (__float128)(((long)ix * kx) % nx) / nx;
            __float128 wxr = cosq(th), wxi = sign * sinq(th);
            __float128 pr = 0, pi = 0;
            for (int iy = 0; iy < ny; iy++) {
                const double *row = x + 2 * (((long)ix * ny + iy) * nz);
                __float128 qr = 0, qi = 0;
                for (int iz = 0; iz < nz; iz++) {
                    __float128 a = row[2 * iz], c = row[2 * iz + 1];
                    qr += a * zr[iz] - c * zi[iz];
                    qi += a * zi[iz] + c * zr[iz];
                }
                pr += qr * yr[iy] - qi * yi[iy];
                pi += qr * yi[iy] + qi * yr[iy];
            }
            sr += pr * wxr - pi * wxi;
            si += pr * wxi + pi * wxr;
        }
        free(zr); free(zi); free(yr); free(yi);
        __float128 dr = (__float128)ysamp[2 * s] - sr, di = (__float128)ysamp[2 * s + 1] - si;
        num += dr * dr + di * di;
        den += sr * sr + si * si;
    }
    return (double)sqrtq(num / den);
}

int oz_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
