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
};

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

// r in [0, 2^32) -> r mod m by Barrett with mu = floor(2^32/m): one multiply-high, one conditional subtract
__device__ __forceinline__ uint32_t barrett(uint32_t r, uint32_t m, uint32_t mu) {
    uint32_t q = __umulhi(r, mu);
    r -= q * m;  // in [0, 2m)
    return r >= m ? r - m : r;
}

// canonical residue of a 53-bit magnitude (PAPER.md:190 with 16-bit planes: sum_k limb_k * (2^16k mod m))
__device__ __forceinline__ uint32_t residue53(uint64_t a, int i, const DevConsts &c) {
    const uint32_t lo = (uint32_t)a, hi = (uint32_t)(a >> 32);
    uint32_t r = (lo & 0xFFFF) + (lo >> 16) * c.c16[i] + (hi & 0xFFFF) * c.c32[i] + (hi >> 16) * c.c48[i];
    return barrett(r, c.m[i], c.mu[i]);
}

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

}  // namespace oz
