// stage_simt.cuh -- all-SIMT stage kernel: the simplest correct form of one Bailey stage, kept as the
// in-library cross-check for the tensor-core kernel (selected with OZFFT_VARIANT=simt).
// Steps (Alg. 1, 220-241): load -> column exponent -> quantise -> residues mod m_i ->
// residue DFT (direct 4-product complex form, IMAD) -> canonicalise -> exact CRT + lift -> pack.
#pragma once
#include "arith.cuh"
#include "stage.cuh"

namespace oz {

constexpr int SIMT_THREADS = 256;
constexpr int SIMT_KG = SIMT_THREADS / 32;

// Reconstruction of one output from its 12 canonical residues.
//   RECON 0: direct CRT with idempotents, fractional lift, two-sided centring -- the product form.
//   RECON 1 (ablation): recursive Garner, Eq. (9)-(10) of PAPER.md:262-267: mixed-radix digits
//            v_k = (v'_k - sum_{j<k} v_j prod_{i<j} m_i) (prod_{i<k} m_i)^-1 mod m_k, then the positional sum (Eq. 9).  Exact.
//   RECON 2 (ablation): tc-CRT slice sums P_s followed by the NAIVE fp64 Phase B of PAPER.md:340-345 (Eq. 21):
//            sum_s P_s c_s accumulated in fp64, rounding at every step.  The paper's naive form has no lift at all; to get a
//            comparable output the quotient is taken in fp64 as well (rint(E/M)).  NOT exact: it is the accuracy-and-speed
//            baseline, the only code in the library that uses fp64 arithmetic, excluded from the SASS hygiene test by name.
template <int RECON> __device__ __forceinline__ uint64_t simt_reconstruct(const uint32_t *v, const DevConsts &c, int gexp) {
    if constexpr (RECON == 0) {
        return pack_rne(crt_centre(v, c), gexp);
    } else if constexpr (RECON == 1) {
        uint32_t d[12];
#pragma unroll
        for (int k = 0; k < 12; k++) {
            const uint32_t m = c.m[k], mu = c.mu[k];
            uint32_t acc = 0;  // sum_{j<k} d_j * gprod[j][k] mod m_k, one multiply-add-reduce per earlier digit (Eq. 10)
#pragma unroll
            for (int j = 0; j < k; j++) acc = barrett(acc + d[j] * (uint32_t)c.gprod[j][k], m, mu);
            const uint32_t diff = v[k] >= acc ? v[k] - acc : v[k] + m - acc;
            d[k] = barrett(diff * (uint32_t)c.ginv[k], m, mu);
        }
        u128 a = d[11];
#pragma unroll
        for (int k = 10; k >= 0; k--) a = a * c.m[k] + d[k];  // Eq. (9), Horner form
        const u128 M = ((u128)c.M[3] << 96) | ((u128)c.M[2] << 64) | ((u128)c.M[1] << 32) | c.M[0];
        i128 R = (i128)a;
        if (a >= (M >> 1)) R -= (i128)M;
        return pack_rne(R, gexp);
    } else {
        double e = 0.0;
#pragma unroll
        for (int s = 14; s >= 0; s--) {  // P_s = sum_k v_k byte_s(u_k) (Eq. 18-19), then sum_s P_s 256^s in fp64
            uint32_t P = 0;
#pragma unroll
            for (int k = 0; k < 12; k++) P += v[k] * (uint32_t)c.uslice[k][s];
            e = fma((double)P, exp2((double)(8 * s)), e);
        }
        const u128 M = ((u128)c.M[3] << 96) | ((u128)c.M[2] << 64) | ((u128)c.M[1] << 32) | c.M[0];
        const double Md = (double)(uint64_t)(M >> 64) * 18446744073709551616.0 + (double)(uint64_t)M;
        const double z = rint(e / Md);
        const double r = fma(-z, Md, e);
        return (uint64_t)__double_as_longlong(ldexp(r, -gexp));
    }
}

// dynamic smem: bits[K][32] (16 B each) | xres[12][K][32] ushort2
template <int RECON>
__device__ __forceinline__ void stage_simt_body(const StageGeom &g, const ulonglong2 *__restrict__ in, ulonglong2 *__restrict__ out,
                                                const ushort2 *__restrict__ mat, const DevConsts *__restrict__ cptr) {
    extern __shared__ __align__(16) uint8_t smem_raw[];
    __shared__ int s_tmax[32];
    __shared__ int s_flag[32];  // bit0: some nonzero finite, bit1: non-finite
    __shared__ DevConsts c;
    const int K = g.K;
    ulonglong2 *s_bits = (ulonglong2 *)smem_raw;
    ushort2 *s_x = (ushort2 *)(smem_raw + (size_t)K * 32 * 16);
    const int tid = threadIdx.x, lane = tid & 31, grp = tid >> 5;

    for (int i = tid; i < (int)(sizeof(DevConsts) / 4); i += SIMT_THREADS) ((uint32_t *)&c)[i] = ((const uint32_t *)cptr)[i];
    if (tid < 32) { s_tmax[tid] = -100000; s_flag[tid] = 0; }
    __syncthreads();

    int tb, ts, to;
    tile_coords(g, blockIdx.x, g.nb, tb, ts, to);
    const long long ibase = tb * g.ib + ts * g.is + to * g.io + lane * g.lane;
    const long long obase = tb * g.ob + ts * g.os + to * g.oo + lane * g.olane;
    const int mid = g.matsel ? ts : 0;
    const bool valid = tb * 32 + lane < g.ncols;  // masked tail block

    // ---- load + column exponent (a1, a2)
    for (int j = grp; j < K; j += SIMT_KG) {
        const ulonglong2 v = valid ? in[ibase + j * g.ji] : make_ulonglong2(0, 0);
        s_bits[j * 32 + lane] = v;
        int T, cls, fl = 0, tm = -100000;
        cls = classify_top(v.x, T);
        if (cls == CLS_FINITE) { fl |= 1; tm = T; }
        if (cls == CLS_NONFINITE) fl |= 2;
        cls = classify_top(v.y, T);
        if (cls == CLS_FINITE) { fl |= 1; tm = max(tm, T); }
        if (cls == CLS_NONFINITE) fl |= 2;
        if (fl & 1) atomicMax(&s_tmax[lane], tm);
        if (fl) atomicOr(&s_flag[lane], fl);
    }
    __syncthreads();
    const int Tmax = s_tmax[lane], flag = s_flag[lane];

    // ---- quantise + residues (a3)
    for (int j = grp; j < K; j += SIMT_KG) {
        const ulonglong2 v = s_bits[j * 32 + lane];
        const uint64_t ar = (flag == 1) ? quantise_mag(v.x, Tmax) : 0, ai = (flag == 1) ? quantise_mag(v.y, Tmax) : 0;
        const bool nr = v.x >> 63, ni = v.y >> 63;
#pragma unroll
        for (int i = 0; i < 12; i++) {
            uint32_t rr = residue53(ar, i, c), ri = residue53(ai, i, c);
            if (nr && rr) rr = c.m[i] - rr;
            if (ni && ri) ri = c.m[i] - ri;
            s_x[(i * K + j) * 32 + lane] = make_ushort2((unsigned short)rr, (unsigned short)ri);
        }
    }
    __syncthreads();

    // ---- residue DFT + reconstruction, one (column, k) per thread iteration (a4-a9)
    const int gexp = 53 + 52 - Tmax;
    for (int k = grp; k < K; k += SIMT_KG) {
        ulonglong2 y;
        if (flag & 2) {
            y.x = y.y = 0x7FF8000000000000ull;
        } else if (flag == 0) {
            y.x = y.y = 0;
        } else {
            uint32_t vr[12], vi[12];
#pragma unroll
            for (int i = 0; i < 12; i++) {
                const ushort2 *arow = mat + (((size_t)mid * 12 + i) * K + k) * K;
                int re = 0, im = 0;
                for (int j = 0; j < K; j++) {
                    const ushort2 a = __ldg(arow + j);
                    const ushort2 x = s_x[(i * K + j) * 32 + lane];
                    re += (int)a.x * (int)x.x - (int)a.y * (int)x.y;
                    im += (int)a.x * (int)x.y + (int)a.y * (int)x.x;
                }
                vr[i] = barrett((uint32_t)(re + (int)c.off28[i]), c.m[i], c.mu[i]);
                vi[i] = barrett((uint32_t)(im + (int)c.off28[i]), c.m[i], c.mu[i]);
            }
            y.x = simt_reconstruct<RECON>(vr, c, gexp);
            y.y = simt_reconstruct<RECON>(vi, c, gexp);
        }
        if (valid) out[obase + k * g.ko] = y;
    }
}

__global__ void __launch_bounds__(SIMT_THREADS) stage_simt_kernel(StageGeom g, const ulonglong2 *__restrict__ in, ulonglong2 *__restrict__ out,
                                                                  const ushort2 *__restrict__ mat, const DevConsts *__restrict__ cptr) {
    stage_simt_body<0>(g, in, out, mat, cptr);
}
__global__ void __launch_bounds__(SIMT_THREADS) stage_garner_kernel(StageGeom g, const ulonglong2 *__restrict__ in, ulonglong2 *__restrict__ out,
                                                                    const ushort2 *__restrict__ mat, const DevConsts *__restrict__ cptr) {
    stage_simt_body<1>(g, in, out, mat, cptr);
}
__global__ void __launch_bounds__(SIMT_THREADS) stage_fp64sum_kernel(StageGeom g, const ulonglong2 *__restrict__ in, ulonglong2 *__restrict__ out,
                                                                     const ushort2 *__restrict__ mat, const DevConsts *__restrict__ cptr) {
    stage_simt_body<2>(g, in, out, mat, cptr);
}

}  // namespace oz
