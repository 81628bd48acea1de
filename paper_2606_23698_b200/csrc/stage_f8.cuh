// stage_f8.cuh -- the paper's titular rung as a measured variant (OZFFT_VARIANT=fp8): one Bailey stage with the residue
// DFT on tcgen05 kind::f8f6f4 (E4M3 operands, fp32 accumulation) and the 3-GEMM complex Karatsuba combine carried in the
// residue domain (Alg. 1 lines 3-6, 252-258 Eq. 8, 275).
//
// Plane layout (the paper gives none, "no exact three-plane layout is proven"): E4M3 holds
// the integers 0..16 exactly, so a canonical residue v < 2^12 is three hex digits v = v0 + 16 v1 + 256 v2
// and a matrix residue a enters as the hex digits of a 16^e mod m (e = 0, 1, 2):
//     a v == sum_f 16^f sum_e v_e hexdigit_f(a 16^e mod m)   (mod m),
// i.e. per modulus and real GEMM 3 data planes x 3 matrix planes feeding 3 fp32 accumulators P_f <= 96 * 225 < 2^15
// (exact; silicon contract in tests/test_gpu_silicon.py).  alpha = 9 plane products per modulus and real GEMM,
// alpha_C = 3 (D, E, F) x 9 x 12 = 324 against the paper's 111 (138 conservative) -- the number PAPER.md:113 could not state.
// Karatsuba: D = A_R X_R, E = A_I X_I, F = (A_R + A_I)(X_R + X_I) as three MMA chains with three data operands and
// three matrix operands; Re = D - E, Im = F - D - E on the recombined integers, one canonicalisation each.
//
// Deliberately simple: tile = 64 columns (MMA rows 64..127 repeat rows 0..63 so that every TMEM lane quarter has work in
// the epilogue), one modulus at a time, single-buffered operands, residues parked in shared memory, reconstruction
// (direct CRT in 32-bit limbs + lift + pack, arith.cuh) on the SIMT pipe.  It exists to be MEASURED against the
// kind::i8 kernels (profiles/r2_configs.md), not to be fast.
#pragma once
#include <vector>

#include "arith.cuh"
#include "stage.cuh"
#include "tables.cuh"
#include "tc.cuh"

namespace oz {

constexpr int F8_THREADS = 256;
__host__ __device__ constexpr int f8_kb(int K) { return ((3 * K + 31) / 32) * 32; }   // operand bytes per row: kappa = 3 j + e
__host__ __device__ constexpr int f8_np(int K) { return ((3 * K + 15) / 16) * 16; }   // MMA N: n = 3 k + f, padded
__host__ __device__ constexpr int f8_mat_bytes(int K) { return f8_np(K) * f8_kb(K); } // one of A_R, A_I, A_S of one modulus
__host__ __device__ constexpr size_t f8_smem_bytes(int K) {
    return (size_t)K * 64 * 16 + 3 * (size_t)128 * f8_kb(K) + 3 * (size_t)f8_mat_bytes(K) + (size_t)12 * 2 * K * 64 * 2;
}
static const uint8_t kE4M3[16] = {0x00, 0x38, 0x40, 0x44, 0x48, 0x4A, 0x4C, 0x4E, 0x50, 0x51, 0x52, 0x53, 0x54, 0x55, 0x56, 0x57};

// host: E4M3 hex-digit planes [mid][i][g = R, I, S][kappa/16][n][16 B]
inline void build_mat_f8(std::vector<uint8_t> &h, int K, int fusedN, int sign, const Twiddles &T) {
    const int nmat = fusedN ? 32 : 1, KB = f8_kb(K), NP = f8_np(K), MB = f8_mat_bytes(K);
    h.assign((size_t)nmat * 12 * 3 * MB, 0);
    for (int mid = 0; mid < nmat; mid++)
        for (int i = 0; i < 12; i++) {
            const int m = kModuli[i];
            for (int k = 0; k < K; k++)
                for (int j = 0; j < K; j++) {
                    const int t = fusedN ? (int)(((long)(TABLE_N / fusedN) * j * (mid + 32L * k)) % TABLE_N) : (int)(((long)(TABLE_N / K) * j * k) % TABLE_N);
                    const int aR = residue_of(T.c[t], m), aI = residue_of((int64_t)sign * T.s[t], m);
                    const int a[3] = {aR, aI, (aR + aI) % m};
                    for (int g = 0; g < 3; g++) {
                        uint8_t *dst = h.data() + (((size_t)mid * 12 + i) * 3 + g) * MB;
                        int v = a[g];
                        for (int e = 0; e < 3; e++) {  // v = a 16^e mod m
                            const int kap = 3 * j + e;
                            for (int f = 0; f < 3; f++)
                                dst[(kap / 16) * (NP * 16) + (3 * k + f) * 16 + kap % 16] = kE4M3[(v >> (4 * f)) & 15];
                            v = (v * 16) % m;
                        }
                    }
                }
        }
}

__device__ __forceinline__ uint32_t e4m3_of_hex(uint32_t n) {  // E4M3 byte of the integer n in 0..15
    const uint64_t lut = n & 8 ? 0x5756555453525150ull : 0x4E4C4A4844403800ull;
    return (uint32_t)(lut >> (8 * (n & 7))) & 0xFF;
}

__global__ void __launch_bounds__(F8_THREADS, 1) stage_f8_kernel(StageGeom g, const uint4 *__restrict__ in, uint4 *__restrict__ out,
                                                                const uint8_t *__restrict__ mat, long long ntiles) {
    extern __shared__ __align__(128) uint8_t smem[];
    __shared__ __align__(8) uint64_t bar_mat, bar_mma;
    __shared__ uint32_t s_tmem;
    __shared__ int s_tmax[64], s_flag[64];
    const int K = g.K, KB = f8_kb(K), NP = f8_np(K), MB = f8_mat_bytes(K);
    longlong2 *s_q = (longlong2 *)smem;                         // [K][64] quantised (re, im); raw bits before that
    uint8_t *sA = smem + (size_t)K * 64 * 16;                   // [3][KB/16][128][16]
    uint8_t *sB = sA + 3 * (size_t)128 * KB;                    // [3][KB/16][NP][16]
    uint16_t *s_res = (uint16_t *)(sB + 3 * (size_t)MB);        // [12][2 K][64]
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int lg_nbt = 32 - __clz(((g.nb + 1) >> 1) - 1), lg_ns = 31 - __clz(g.ns);

    if (warp == 0) tmem_alloc<512>(&s_tmem);
    if (tid == 0) { mbar_init(&bar_mat, 1); mbar_init(&bar_mma, 1); mbar_fence_init(); }
    for (int i = tid; i < 3 * 128 * KB / 4; i += F8_THREADS) ((uint32_t *)sA)[i] = 0;  // padding bytes stay zero
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = s_tmem;
    const uint32_t idesc = make_idesc(CFMT_F32, F8_E4M3, F8_E4M3, 128, NP);
    uint32_t ph_mat = 0, ph_mma = 0;

    for (long long tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        int tb, ts, to;
        tile_coords_pow2(g, tile, lg_nbt, lg_ns, tb, ts, to);
        const uint8_t *mb = mat + (size_t)(g.matsel ? ts : 0) * 12 * 3 * MB;
        if (tid < 64) { s_tmax[tid] = -100000; s_flag[tid] = 0; }
        __syncthreads();
        // ---- a1, a2: load, column exponent
        for (int idx = tid; idx < K * 64; idx += F8_THREADS) {
            const int j = idx >> 6, col = idx & 63, blk = 2 * tb + (col >> 5);
            const bool valid = blk * 32 + (col & 31) < g.ncols;
            const uint4 v = valid ? __ldg(in + ((long long)blk * g.ib + (long long)ts * g.is + (long long)to * g.io + (long long)(col & 31) * g.lane + (long long)j * g.ji))
                                  : make_uint4(0, 0, 0, 0);
            ((uint4 *)s_q)[idx] = v;
            int T, fl = 0, tm = -100000;
            int cls = classify_top(((uint64_t)v.y << 32) | v.x, T);
            if (cls == CLS_FINITE) { fl |= 1; tm = T; }
            if (cls == CLS_NONFINITE) fl |= 2;
            cls = classify_top(((uint64_t)v.w << 32) | v.z, T);
            if (cls == CLS_FINITE) { fl |= 1; tm = max(tm, T); }
            if (cls == CLS_NONFINITE) fl |= 2;
            if (fl & 1) atomicMax(&s_tmax[col], tm);
            if (fl) atomicOr(&s_flag[col], fl);
        }
        __syncthreads();
        // ---- a3 (first half): quantise once
        for (int idx = tid; idx < K * 64; idx += F8_THREADS) {
            const int col = idx & 63;
            const uint4 v = ((uint4 *)s_q)[idx];
            const uint64_t br = ((uint64_t)v.y << 32) | v.x, bi = ((uint64_t)v.w << 32) | v.z;
            const bool ok = s_flag[col] == 1;
            const int64_t ar = ok ? (int64_t)quantise_mag(br, s_tmax[col]) : 0, ai = ok ? (int64_t)quantise_mag(bi, s_tmax[col]) : 0;
            s_q[idx] = make_longlong2((br >> 63) ? -ar : ar, (bi >> 63) ? -ai : ai);
        }
        __syncthreads();
        for (int i = 0; i < 12; i++) {
            if (tid == 0) {  // matrix planes A_R, A_I, A_S of this modulus (the previous modulus' MMAs are complete)
                mbar_expect_tx(&bar_mat, 3 * MB);
                bulk_g2s(sB, mb + (size_t)i * 3 * MB, 3 * MB, &bar_mat);
            }
            // ---- a3 (second half): residues of x_R, x_I and of the Karatsuba operand x_R + x_I; hex digits as E4M3
            const uint32_t m = kc.m[i];
            for (int idx = tid; idx < K * 64; idx += F8_THREADS) {
                const int j = idx >> 6, col = idx & 63;
                const longlong2 q = s_q[idx];
                uint32_t rR = residue53((uint64_t)(q.x < 0 ? -q.x : q.x), i, kc), rI = residue53((uint64_t)(q.y < 0 ? -q.y : q.y), i, kc);
                if (q.x < 0 && rR) rR = m - rR;
                if (q.y < 0 && rI) rI = m - rI;
                uint32_t rS = rR + rI;
                if (rS >= m) rS -= m;
                const uint32_t r3[3] = {rR, rI, rS};
#pragma unroll
                for (int gg = 0; gg < 3; gg++)
#pragma unroll
                    for (int e = 0; e < 3; e++) {
                        const int kap = 3 * j + e;
                        uint8_t *p = sA + (size_t)gg * 128 * KB + (kap >> 4) * 2048 + col * 16 + (kap & 15);
                        const uint8_t b = (uint8_t)e4m3_of_hex((r3[gg] >> (4 * e)) & 15);
                        p[0] = b;
                        p[64 * 16] = b;  // rows 64..127 repeat rows 0..63
                    }
            }
            fence_async_smem();
            tc_fence_before();
            __syncthreads();
            // ---- a4: D, E, F on the tensor core
            if (tid == 0) {
                tc_fence_after();
                mbar_wait(&bar_mat, ph_mat);
                for (int gg = 0; gg < 3; gg++)
                    for (int ks = 0; ks < KB / 32; ks++)
                        mma_f8f6f4_ss(tmem + gg * NP, make_sdesc(smem_u32(sA) + gg * 128 * KB + ks * 2 * 2048, 2048, 128),
                                      make_sdesc(smem_u32(sB) + gg * MB + ks * 2 * NP * 16, NP * 16, 128), idesc, ks > 0);
                tc_commit(&bar_mma);
            }
            ph_mat ^= 1;
            mbar_wait(&bar_mma, ph_mma);
            ph_mma ^= 1;
            tc_fence_after();
            // ---- a5: recombine the hex planes, Karatsuba combine in the residue domain, canonicalise, park
            {
                const int row = (warp & 3) * 32 + lane, col = row & 63, part4 = (row >> 6) * 2 + (warp >> 2);
                const uint32_t ta = tmem + ((uint32_t)((warp & 3) * 32) << 16);
                const uint32_t off = kc.off28[i], mu = kc.mu[i];
                for (int k = part4 * K / 4; k < (part4 + 1) * K / 4; k++) {
                    int v[3];
#pragma unroll
                    for (int gg = 0; gg < 3; gg++) {
                        uint32_t p0, p1, p2;
                        tmem_ld_x1(ta + gg * NP + 3 * k, p0);
                        tmem_ld_x1(ta + gg * NP + 3 * k + 1, p1);
                        tmem_ld_x1(ta + gg * NP + 3 * k + 2, p2);
                        tmem_ld_wait();
                        v[gg] = __float2int_rn(__uint_as_float(p0)) + 16 * __float2int_rn(__uint_as_float(p1)) + 256 * __float2int_rn(__uint_as_float(p2));
                    }
                    const int re = v[0] - v[1], im = v[2] - v[0] - v[1];  // Re = D - E, Im = F - D - E
                    s_res[((size_t)i * 2 * K + k) * 64 + col] = (uint16_t)barrett((uint32_t)(re + (int)off), m, mu);
                    s_res[((size_t)i * 2 * K + K + k) * 64 + col] = (uint16_t)barrett((uint32_t)(im + (int)off), m, mu);
                }
            }
            tc_fence_before();
            __syncthreads();
        }
        // ---- a6-a9, a12: reconstruction on the SIMT pipe, store
        for (int idx = tid; idx < K * 64; idx += F8_THREADS) {
            const int k = idx >> 6, col = idx & 63, blk = 2 * tb + (col >> 5);
            if (blk * 32 + (col & 31) >= g.ncols) continue;
            const int flag = s_flag[col], gexp = 53 + 52 - s_tmax[col];
            uint64_t y[2];
#pragma unroll
            for (int P = 0; P < 2; P++) {
                if (flag & 2) y[P] = 0x7FF8000000000000ull;
                else if (flag == 0) y[P] = 0;
                else {
                    uint32_t v[12], r[4];
#pragma unroll
                    for (int i = 0; i < 12; i++) v[i] = s_res[((size_t)i * 2 * K + P * K + k) * 64 + col];
                    crt_limbs(v, r);
                    y[P] = pack_limbs(r, gexp);
                }
            }
            out[(long long)blk * g.ob + (long long)ts * g.os + (long long)to * g.oo + (long long)(col & 31) * g.olane + (long long)k * g.ko] =
                make_uint4((uint32_t)y[0], (uint32_t)(y[0] >> 32), (uint32_t)y[1], (uint32_t)(y[1] >> 32));
        }
        __syncthreads();
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc<512>(tmem);
}

inline bool stage_f8_prepare() {
    return cudaFuncSetAttribute(stage_f8_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)f8_smem_bytes(32)) == cudaSuccess;
}

inline cudaError_t stage_f8_launch(const StageGeom &g, const void *src, void *dst, const uint8_t *mat, int sms, cudaStream_t st) {
    int nbt = 1;
    while (nbt < (g.nb + 1) / 2) nbt <<= 1;
    if (g.ns & (g.ns - 1)) return cudaErrorInvalidValue;
    const long long nt = (long long)nbt * g.ns * g.no;
    if (nt >= (1ll << 31)) return cudaErrorInvalidValue;
    stage_f8_kernel<<<(unsigned)(nt < sms ? nt : sms), F8_THREADS, f8_smem_bytes(g.K), st>>>(g, (const uint4 *)src, (uint4 *)dst, mat, nt);
    return cudaGetLastError();
}

}  // namespace oz
