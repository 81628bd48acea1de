// arith.cuh -- integer-only device arithmetic of the hot path (no fp64 instruction anywhere):
//   decode / column exponent / quantise   ("round(s_A A)", 218; DESIGN.md A.1-A.3)
//   residues mod m_i
//   Barrett canonicalisation
//   correctly rounded pack                 (DESIGN.md A.6)
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace oz {

struct DevConsts {
    uint32_t m[12];      // moduli
    uint32_t mu[12];     // floor(2^32 / m)
    uint32_t c16[12];    // 2^16 mod m
    uint32_t c32[12];    // 2^32 mod m
    uint32_t c48[12];    // 2^48 mod m
    uint32_t off28[12];  // smallest multiple of m that is >= 2^28 (makes signed accumulators non-negative)
    uint32_t offtc[12];  // same, >= 2^25 (tensor-core digit recombination stays below 2^25 in magnitude)
    uint32_t u[12][4];   // CRT idempotents, 32-bit limbs (u_k < 2^118)
    uint32_t wlo[12], whi[12];  // w_k = round(2^48 u_k / M), split 32 + 16 bits
    uint32_t M[4];       // M limbs
    uint32_t Mh[4];      // M/2 limbs
    uint32_t c18[12];    // 2^18 mod m
    uint32_t c36[12];    // 2^36 mod m
    uint32_t m2[12];     // 2 m
    uint32_t zC;         // round(2^149 / M): zhat = (umulhi(E >> 104, zC) + 2^12) >> 13
    uint32_t m2m2[12];   // 2m in both half-words
    uint32_t off30[12];  // smallest multiple of m >= 2^30: makes the signed plane sum of the deconstruction positive
    uint32_t phaseA[128];  // Phase-A constant matrix: 16 slice rows x 32 bytes in MMA operand order
    // ablation rungs only (PAPER.md:260-273 Garner, 340-345 naive fp64 Phase B)
    uint16_t gprod[12][12];  // gprod[j][k] = (m_0 ... m_{j-1}) mod m_k  (Eq. 10)
    uint16_t ginv[12];       // (m_0 ... m_{k-1})^-1 mod m_k
    uint8_t uslice[12][16];  // byte s of u_k (Eq. 18)
};

// the same constants in the constant bank (uniform operands, no shared-memory loads); set by stage_tc_prepare
__constant__ DevConsts kc;

// [ledger: a2 column exponent]
// value class of an fp64 bit pattern; T = floor(log2 |x|) for finite nonzero x
enum { CLS_ZERO = 0, CLS_FINITE = 1, CLS_NONFINITE = 2 };

__device__ __forceinline__ int classify_top(uint64_t b, int &T) {
    const uint32_t hi = (uint32_t)(b >> 32);
    const int ef = (hi >> 20) & 0x7FF;
    if (ef == 0x7FF) return CLS_NONFINITE;
    if (ef) { T = ef - 1023; return CLS_FINITE; }
    const uint64_t fr = b & 0xFFFFFFFFFFFFFull;
    if (!fr) return CLS_ZERO;
    T = -1074 + (63 - __clzll((long long)fr));
    return CLS_FINITE;
}

// [ledger: a3 deconstruction: quantise, offset, byte planes]
// |RNE(x * 2^(52 - Tmax))| as an integer < 2^53; sign returned separately (bit 63 of b)
__device__ __forceinline__ uint64_t quantise_mag(uint64_t b, int Tmax) {
    const int ef = (int)((b >> 52) & 0x7FF);
    uint64_t mant = b & 0xFFFFFFFFFFFFFull;
    int E = -1074;
    if (ef) { mant |= 1ull << 52; E = ef - 1075; }
    if (!mant) return 0;
    const int sh = Tmax - 52 - E;  // x * 2^(52-Tmax) = mant * 2^-sh
    if (sh <= 0) return mant << (-sh);
    if (sh >= 64) return 0;
    uint64_t q = mant >> sh;
    const uint64_t rem = mant & ((1ull << sh) - 1), half = 1ull << (sh - 1);
    if (rem > half || (rem == half && (q & 1))) q++;
    return q;
}

// out-of-line copies of the rare paths: keeps the unrolled hot loops small enough for the instruction cache
__device__ __noinline__ uint64_t quantise_mag_slow(uint64_t b, int Tmax) { return quantise_mag(b, Tmax); }

// same value as quantise_mag; normal numbers (the usual case) take a short branch-free path:
// q = mant >> sh, the dropped bits left-aligned give the guard bit and the sticky flag
__device__ __forceinline__ uint64_t quantise_mag_fast(uint64_t b, int Tmax) {
    const int ef = (int)((b >> 52) & 0x7FF);
    if (ef == 0) return quantise_mag_slow(b, Tmax);  // zero or subnormal
    const uint64_t mant = (b & 0xFFFFFFFFFFFFFull) | (1ull << 52);
    const int sh = Tmax + 1023 - ef;  // >= 0 because Tmax is the column maximum
    if (sh == 0) return mant;
    if (sh < 32) {  // elements within 2^32 of the column maximum: the dropped bits come from the low word only
        const uint32_t lo = (uint32_t)mant, hi = (uint32_t)(mant >> 32);
        const uint32_t qlo = __funnelshift_r(lo, hi, sh), qhi = hi >> sh, dropped = lo << (32 - sh);
        const uint32_t up = (dropped >> 31) & ((uint32_t)((dropped << 1) != 0) | qlo);
        return (((uint64_t)qhi << 32) | qlo) + up;  // qlo + 1 cannot carry: q < 2^53 means qhi:qlo + 1 fits
    }
    return quantise_mag_slow(b, Tmax);  // more than 2^32 below the column maximum
}

// [ledger: a3/a5 residues: plane dot, Barrett, digit packing]
// r in [0, 2^32) -> r mod m by Barrett with mu = floor(2^32/m): one multiply-high, one conditional subtract
__device__ __forceinline__ uint32_t barrett(uint32_t r, uint32_t m, uint32_t mu) {
    uint32_t q = __umulhi(r, mu);
    r -= q * m;  // in [0, 2m)
    return r >= m ? r - m : r;
}

// r < 2^32 -> a representative of r mod m in [0, 2m): q = mulhi(r, floor(2^32/m)), r + q * (-m); two instructions
// (inline PTX so the compiler keeps the multiply-add form with the negated modulus as an operand)
__device__ __forceinline__ uint32_t barrett_lazy(uint32_t r, uint32_t mu, uint32_t negm) {
    uint32_t o;
    asm("{\n\t.reg .u32 q;\n\tmul.hi.u32 q, %1, %2;\n\tmad.lo.u32 %0, q, %3, %1;\n\t}" : "=r"(o) : "r"(r), "r"(mu), "r"(negm));
    return o;
}

// a + b on the ALU pipe (VIADDMNMX): the integer multiplier pipe is the busier one in the stage kernel, so plain
// adds and packs are steered away from IMAD forms
__device__ __forceinline__ uint32_t add_alu(uint32_t a, uint32_t b) { return __viaddmax_u32(a, b, 0u); }
// (lo & 0xFFFF) | (hi << 16) as one PRMT (ALU pipe)
__device__ __forceinline__ uint32_t pack16(uint32_t lo, uint32_t hi) { return __byte_perm(lo, hi, 0x5410); }

// canonical residue of a 53-bit magnitude (PAPER.md:190 with 16-bit planes: sum_k limb_k * (2^16k mod m))
__device__ __forceinline__ uint32_t residue53(uint64_t a, int i, const DevConsts &c) {
    const uint32_t lo = (uint32_t)a, hi = (uint32_t)(a >> 32);
    uint32_t r = (lo & 0xFFFF) + (lo >> 16) * c.c16[i] + (hi & 0xFFFF) * c.c32[i] + (hi >> 16) * c.c48[i];
    return barrett(r, c.m[i], c.mu[i]);
}

// [ledger: a9 pack]
typedef unsigned __int128 u128;
typedef __int128 i128;

__device__ __forceinline__ int bitlen128(u128 a) {
    const uint64_t hi = (uint64_t)(a >> 64), lo = (uint64_t)a;
    return hi ? 128 - __clzll((long long)hi) : 64 - __clzll((long long)lo);
}

// RNE_fp64(R * 2^-g) as a bit pattern, integer only (DESIGN.md A.6). R != 0 handled; R == 0 -> +0.0.
__device__ __forceinline__ uint64_t pack_rne(i128 R, int g) {
    if (R == 0) return 0;
    const uint64_t sgn = R < 0 ? 1ull << 63 : 0;
    const u128 a = R < 0 ? (u128)(-R) : (u128)R;
    const int L = bitlen128(a);
    int X = L - 1 - g;
    if (X >= -1022) {
        uint64_t q;
        if (L > 53) {
            const int d = L - 53;
            q = (uint64_t)(a >> d);
            const u128 rem = a & (((u128)1 << d) - 1), half = (u128)1 << (d - 1);
            if (rem > half || (rem == half && (q & 1))) q++;
            if (q >> 53) { q >>= 1; X++; }
        } else {
            q = (uint64_t)a << (53 - L);
        }
        if (X > 1023) return sgn | 0x7FF0000000000000ull;
        return sgn | ((uint64_t)(X + 1023) << 52) | (q & 0xFFFFFFFFFFFFFull);
    }
    const int d = g - 1074;  // subnormal result: one rounding straight onto the 2^-1074 grid
    uint64_t q;
    if (d <= 0) q = (uint64_t)a << (-d);
    else if (d > 127) q = 0;
    else {
        q = (uint64_t)(a >> d);
        const u128 rem = a & (((u128)1 << d) - 1), half = (u128)1 << (d - 1);
        if (rem > half || (rem == half && (q & 1))) q++;
    }
    return sgn | q;
}

__device__ __noinline__ uint64_t pack_rne_slow(uint32_t r0, uint32_t r1, uint32_t r2, uint32_t r3, int g) {
    return pack_rne((i128)(((u128)r3 << 96) | ((u128)r2 << 64) | ((u128)r1 << 32) | r0), g);
}

// [ledger: a8 lift: quotient, E - zM, centring, offset constant]
// Exact CRT of 12 canonical residues to the centred representative in [-M/2, M/2)
// (PAPER.md:316-329 direct CRT with idempotents; 370-373 fractional lift and two-sided correction).
// Plain multiword form used by the SIMT reference kernel: all sums are taken mod 2^128, which is exact
// because the centred result has fewer than 119 bits.
__device__ __forceinline__ i128 crt_centre(const uint32_t *v, const DevConsts &c) {
    u128 E = 0;
    uint64_t zacc = 0;
#pragma unroll
    for (int k = 0; k < 12; k++) {
        const u128 uk = ((u128)c.u[k][3] << 96) | ((u128)c.u[k][2] << 64) | ((u128)c.u[k][1] << 32) | c.u[k][0];
        E += uk * v[k];
        zacc += (((uint64_t)c.whi[k] << 32) | c.wlo[k]) * v[k];
    }
    const uint64_t zhat = (zacc + (1ull << 47)) >> 48;
    const u128 M = ((u128)c.M[3] << 96) | ((u128)c.M[2] << 64) | ((u128)c.M[1] << 32) | c.M[0];
    const i128 Mh = (i128)(M >> 1);
    i128 R = (i128)(E - M * zhat);
    if (R >= Mh) R -= (i128)M;
    if (R < -Mh) R += (i128)M;
    return R;
}

// ---------------------------------------------------------------------------------------------------
// 32-bit limb forms used by the tensor-core kernel (same integers as crt_centre / pack_rne above).

// r = a - b over four 32-bit limbs (mod 2^128), one borrow chain
__device__ __forceinline__ void sub128(uint32_t *r, uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t b0,
                                       uint32_t b1, uint32_t b2, uint32_t b3) {
    asm("sub.cc.u32 %0, %4, %8;\n\tsubc.cc.u32 %1, %5, %9;\n\tsubc.cc.u32 %2, %6, %10;\n\tsubc.u32 %3, %7, %11;"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3])
        : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1), "r"(b2), "r"(b3));
}
// [ledger: a9 pack]
// |x| of a two's-complement 128-bit value: (x ^ sm) + (sm & 1) with sm = sign mask, one carry chain
__device__ __forceinline__ void abs128(uint32_t *a, const uint32_t *x, uint32_t sm) {
    asm("add.cc.u32 %0, %4, %8;\n\taddc.cc.u32 %1, %5, 0;\n\taddc.cc.u32 %2, %6, 0;\n\taddc.u32 %3, %7, 0;"
        : "=r"(a[0]), "=r"(a[1]), "=r"(a[2]), "=r"(a[3])
        : "r"(x[0] ^ sm), "r"(x[1] ^ sm), "r"(x[2] ^ sm), "r"(x[3] ^ sm), "r"(sm & 1));
}

// [ledger: a8 lift: quotient, E - zM, centring, offset constant]
// Direct CRT E = sum_k v_k u_k (Eq. 17) on residues that need not be canonical (v_k < 2^13, any
// representative: m_k u_k == 0 mod M), quotient zhat = round(E/M) read off the top 30 bits of E (the lift of
// PAPER.md:370 with the fraction taken from E itself), R = E - zhat M, two-sided centring.
// r[0..3]: two's-complement limbs of R in [-M/2, M/2).
__device__ __forceinline__ void crt_from_E(uint32_t e0, uint32_t e1, uint32_t e2, uint32_t e3, uint32_t e4, uint32_t *r);

// two-sided centring of a value already within one M of the centred range; out of line: in a
// transform |R| <= 2^112.5 and the caller's top-limb test never sends it here (tests/test_gpu_crt.py does)
__device__ __noinline__ uint4 centre_two_sided(uint32_t r0, uint32_t r1, uint32_t r2, uint32_t r3) {
    const u128 M = ((u128)kc.M[3] << 96) | ((u128)kc.M[2] << 64) | ((u128)kc.M[1] << 32) | kc.M[0];
    i128 R = (i128)(((u128)r3 << 96) | ((u128)r2 << 64) | ((u128)r1 << 32) | r0);
    const i128 Mh = (i128)(M >> 1);
    if (R >= Mh) R -= (i128)M;
    if (R < -Mh) R += (i128)M;
    return make_uint4((uint32_t)R, (uint32_t)((u128)R >> 32), (uint32_t)((u128)R >> 64), (uint32_t)((u128)R >> 96));
}

__device__ __forceinline__ void crt_limbs(const uint32_t *v, uint32_t *r) {
    uint64_t a0 = 0, a1 = 0, a2 = 0, a3 = 0;
#pragma unroll
    for (int k = 0; k < 12; k++) {
        a0 += (uint64_t)v[k] * kc.u[k][0];
        a1 += (uint64_t)v[k] * kc.u[k][1];
        a2 += (uint64_t)v[k] * kc.u[k][2];
        a3 += (uint64_t)v[k] * kc.u[k][3];
    }
    a1 += a0 >> 32;
    a2 += a1 >> 32;
    a3 += a2 >> 32;
    crt_from_E((uint32_t)a0, (uint32_t)a1, (uint32_t)a2, (uint32_t)a3, (uint32_t)(a3 >> 32), r);
}

// [ledger: a7 Phase B deposits (TMEM loads, slice sums -> E)]
// Phase B (Alg. 2): deposit the 16 Phase-A slice sums P_s (each < 2^21) at byte offsets
// 8s -- four 64-bit words of four slices each, one carry sweep -- giving E = sum_s P_s 256^s in 32-bit limbs.
__device__ __forceinline__ void deposit_slices(const uint32_t *P, uint32_t *r) {
    uint64_t w[4];
#pragma unroll
    for (int j = 0; j < 4; j++) {  // three multiply-adds per word: 32-bit, then two 32 x 32 + 64 -> 64
        w[j] = (uint64_t)P[4 * j + 2] * 65536u + (P[4 * j] + P[4 * j + 1] * 256u);
        w[j] = (uint64_t)P[4 * j + 3] * 16777216u + w[j];
    }
    const uint64_t t1 = (w[0] >> 32) + w[1], t2 = (t1 >> 32) + w[2], t3 = (t2 >> 32) + w[3];
    crt_from_E((uint32_t)w[0], (uint32_t)t1, (uint32_t)t2, (uint32_t)t3, (uint32_t)(t3 >> 32), r);
}

// the same deposits, returning the five limbs of E (the byte-fed kernel lifts later, after freeing its TMEM slot)
__device__ __forceinline__ void slices_to_E(const uint32_t *P, uint32_t *e) {
    uint64_t w[4];
#pragma unroll
    for (int j = 0; j < 4; j++) {
        w[j] = (uint64_t)P[4 * j + 2] * 65536u + (P[4 * j] + P[4 * j + 1] * 256u);
        w[j] = (uint64_t)P[4 * j + 3] * 16777216u + w[j];
    }
    const uint64_t t1 = (w[0] >> 32) + w[1], t2 = (t1 >> 32) + w[2], t3 = (t2 >> 32) + w[3];
    e[0] = (uint32_t)w[0]; e[1] = (uint32_t)t1; e[2] = (uint32_t)t2; e[3] = (uint32_t)t3; e[4] = (uint32_t)(t3 >> 32);
}

// [ledger: a8 lift: quotient, E - zM, centring, offset constant]
// lift and centring from the limbs of E (< 2^134): see crt_limbs
__device__ __forceinline__ void crt_from_E(uint32_t e0, uint32_t e1, uint32_t e2, uint32_t e3, uint32_t e4, uint32_t *r) {
    const uint32_t T = __funnelshift_r(e3, e4, 8);  // E >> 104
    const uint32_t z = (__umulhi(T, kc.zC) + (1u << 12)) >> 13;
    uint64_t p0 = (uint64_t)z * kc.M[0];
    uint64_t p1 = (uint64_t)z * kc.M[1] + (p0 >> 32);
    uint64_t p2 = (uint64_t)z * kc.M[2] + (p1 >> 32);
    uint64_t p3 = (uint64_t)z * kc.M[3] + (p2 >> 32);
    sub128(r, e0, e1, e2, e3, (uint32_t)p0, (uint32_t)p1, (uint32_t)p2, (uint32_t)p3);
    // |R| can reach M/2 only if the top limb does; everything else skips the exact comparison
    if ((uint32_t)(r[3] + kc.Mh[3]) >= 2 * kc.Mh[3]) {
        const uint4 c = centre_two_sided(r[0], r[1], r[2], r[3]);
        r[0] = c.x; r[1] = c.y; r[2] = c.z; r[3] = c.w;
    }
}

// [ledger: a9 pack]
// RNE_fp64(R * 2^-g) from two's-complement limbs (DESIGN.md A.6); normal-range results take the limb path,
// zero / subnormal / overflowing ones the generic pack_rne.
__device__ __forceinline__ uint64_t pack_limbs(const uint32_t *r, int g) {
    const uint32_t sm = (uint32_t)((int32_t)r[3] >> 31);  // all ones if negative
    uint32_t av[4];
    abs128(av, r, sm);
    uint32_t a0 = av[0], a1 = av[1], a2 = av[2], a3 = av[3];
    int s;
    if (a3) {  // the usual case in a transform: |R| >= 2^96
        s = __clz((int)a3);
    } else {
        const uint64_t hi = a2, lo = ((uint64_t)a1 << 32) | a0;
        s = hi ? 32 + __clz((int)a2) : 64 + __clzll((long long)lo);  // 128 for R = 0
        if (s & 64) { a3 = a1; a2 = a0; a1 = 0; a0 = 0; }
        if (s & 32) { a3 = a2; a2 = a1; a1 = a0; a0 = 0; }
    }
    const int X = 127 - s - g;
    if ((uint32_t)(X + 1022) > 2045u || s >= 128) {  // zero, subnormal or overflowing result: generic path
        return pack_rne_slow(r[0], r[1], r[2], r[3], g);
    }
    const int bs = s & 31;
    const uint32_t m3 = __funnelshift_l(a2, a3, bs), m2 = __funnelshift_l(a1, a2, bs), m1 = __funnelshift_l(a0, a1, bs), m0 = a0 << bs;
    // top 53 bits = m3 : m2[31:11]; round bit m2[10]; sticky = rest
    const uint32_t qhi = m3 >> 11, qlo = __funnelshift_r(m2, m3, 11);
    const uint32_t sticky = ((m2 & 0x3FF) | m1 | m0) != 0;
    const uint32_t inc = (m2 >> 10) & (sticky | qlo) & 1;
    // exponent field X+1023 enters as (X+1022) << 52 plus the hidden bit; a mantissa carry bumps it by itself
    const uint32_t lo32 = qlo + inc;
    const uint32_t hi32 = qhi + ((uint32_t)(X + 1022) << 20) + (lo32 < inc) + (sm & 0x80000000u);
    return ((uint64_t)hi32 << 32) | lo32;
}

}  // namespace oz
