// tables.cuh -- plan-time HOST generation of every integer constant the kernels use.
//   * Rev-34 modulus set, M, CRT idempotents u_k, lift fractions w_k
//   * omega_1024 table (RN(2^53 cos), RN(2^53 sin)) in double-double arithmetic (reading S5)
//   * per-stage DFT / twiddle-fused matrices reduced mod m_i                  (Eq. 6)
// Independent of oracle/: the oracle uses libquadmath; this file uses its own double-double Taylor series.
#pragma once
#include <cmath>
#include <cstdint>
#include <vector>

namespace oz {

constexpr int R_MOD = 12;
constexpr int TABLE_N = 1024;
static const int kModuli[R_MOD] = {2039, 2029, 2027, 1089, 1024, 961, 841, 625, 529, 511, 491, 487};

typedef unsigned __int128 u128;

// ------------------------------------------------------------------ double-double
struct dd {
    double hi, lo;
};
static inline dd dd_two_sum(double a, double b) {
    double s = a + b, bb = s - a;
    return {s, (a - (s - bb)) + (b - bb)};
}
static inline dd dd_add(dd a, dd b) {
    dd s = dd_two_sum(a.hi, b.hi);
    dd t = dd_two_sum(a.lo, b.lo);
    s.lo += t.hi;
    s = dd_two_sum(s.hi, s.lo);
    s.lo += t.lo;
    return dd_two_sum(s.hi, s.lo);
}
static inline dd dd_mul(dd a, dd b) {
    double p = a.hi * b.hi;
    double e = std::fma(a.hi, b.hi, -p);
    e += a.hi * b.lo + a.lo * b.hi;
    return dd_two_sum(p, e);
}
static inline dd dd_div_int(dd a, double n) {  // n a small exact integer
    double q1 = a.hi / n;
    double r = std::fma(-q1, n, a.hi);  // exact remainder of the high part
    double q2 = (r + a.lo) / n;
    return dd_two_sum(q1, q2);
}

// sin and cos of theta (|theta| <= pi/4) by Taylor series in double-double (~2^-104 relative)
static inline void dd_sincos(dd th, dd &s, dd &c) {
    dd t2 = dd_mul(th, th);
    dd term = th;  // sin series term
    s = th;
    for (int n = 1; n < 16; n++) {
        term = dd_div_int(dd_mul(term, t2), (double)((2 * n) * (2 * n + 1)));
        term.hi = -term.hi;
        term.lo = -term.lo;
        s = dd_add(s, term);
    }
    term = {1.0, 0.0};
    c = term;
    for (int n = 1; n < 16; n++) {
        term = dd_div_int(dd_mul(term, t2), (double)((2 * n - 1) * (2 * n)));
        term.hi = -term.hi;
        term.lo = -term.lo;
        c = dd_add(c, term);
    }
}

static inline int64_t dd_round_scaled(dd v) {  // nearest integer of v * 2^53 (no tie occurs in this table)
    double hi = std::ldexp(v.hi, 53), lo = std::ldexp(v.lo, 53);
    double n = std::nearbyint(hi);
    double rem = (hi - n) + lo;
    int64_t r = (int64_t)n;
    if (rem > 0.5) r++;
    if (rem < -0.5) r--;
    return r;
}

struct Twiddles {
    int64_t c[TABLE_N], s[TABLE_N];
};

// T[t] = (RN(2^53 cos(2 pi t/1024)), RN(2^53 sin(2 pi t/1024))): first octant computed, rest by symmetry.
static inline void build_twiddles(Twiddles &T) {
    const dd pi = {3.141592653589793116e+00, 1.224646799147353207e-16};
    for (int t = 0; t <= 128; t++) {
        dd th = dd_div_int(dd_mul(pi, dd{(double)t, 0.0}), 512.0);
        dd s, c;
        dd_sincos(th, s, c);
        T.c[t] = dd_round_scaled(c);
        T.s[t] = dd_round_scaled(s);
    }
    for (int t = 129; t <= 256; t++) { T.c[t] = T.s[256 - t]; T.s[t] = T.c[256 - t]; }
    for (int t = 257; t <= 512; t++) { T.c[t] = -T.c[512 - t]; T.s[t] = T.s[512 - t]; }
    for (int t = 513; t < 1024; t++) { T.c[t] = T.c[1024 - t]; T.s[t] = -T.s[1024 - t]; }
}

static inline uint64_t twiddle_fnv(const Twiddles &T) {  // FNV-1a over (c, s) little-endian, t = 0..1023
    uint64_t h = 1469598103934665603ULL;
    for (int t = 0; t < TABLE_N; t++) {
        int64_t v[2] = {T.c[t], T.s[t]};
        const unsigned char *p = (const unsigned char *)v;
        for (int i = 0; i < 16; i++) { h ^= p[i]; h *= 1099511628211ULL; }
    }
    return h;
}

// ------------------------------------------------------------------ CRT constants
struct CrtConsts {
    u128 M, Mhalf;
    u128 u[R_MOD];      // idempotents (Eq. 17)
    uint64_t w[R_MOD];  // round(2^48 u_k / M)
};

static inline int mod_inverse(int a, int m) {  // extended Euclid
    long r0 = m, r1 = a % m, s0 = 0, s1 = 1;
    while (r1) {
        long q = r0 / r1, t = r0 - q * r1;
        r0 = r1; r1 = t;
        t = s0 - q * s1; s0 = s1; s1 = t;
    }
    return (int)((s0 % m + m) % m);
}

static inline void build_crt(CrtConsts &C) {
    C.M = 1;
    for (int k = 0; k < R_MOD; k++) C.M *= (u128)kModuli[k];
    C.Mhalf = C.M >> 1;
    for (int k = 0; k < R_MOD; k++) {
        u128 Mk = C.M / (u128)kModuli[k];
        int t = mod_inverse((int)(Mk % (u128)kModuli[k]), kModuli[k]);
        C.u[k] = Mk * (u128)t;
        // w = floor(2^48 u / M + 1/2): schoolbook division, one base-256 quotient digit at a time
        // (u < M < 2^118, so rem << 8 stays below 2^126)
        u128 rem = C.u[k];
        uint64_t q = 0;
        for (int d = 0; d < 6; d++) {
            rem <<= 8;
            q = (q << 8) | (uint64_t)(rem / C.M);
            rem %= C.M;
        }
        if (rem * 2 >= C.M) q++;
        C.w[k] = q;
    }
}

static inline int residue_of(int64_t x, int m) {
    int64_t r = x % m;
    return (int)(r < 0 ? r + m : r);
}

}  // namespace oz
