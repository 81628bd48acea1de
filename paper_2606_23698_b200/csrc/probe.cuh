// probe.cuh -- test hooks of the library (included by ozfft.cu so that they see the same constant bank):
//  * ozfft_probe_mma:   one chained tcgen05.mma (M=128) on caller-supplied operand bytes; tests/test_gpu_silicon.py
//    checks that integer-valued E4M3 / F16 / S8 / U8 operands accumulate exactly (PAPER.md:338, 890 flags this
//    contract as unmeasured).
//  * ozfft_probe_chain: MMA1 (u8 x u8 -> s32 in TMEM) followed by MMA2 whose A operand IS the TMEM accumulator of
//    MMA1 read as unsigned bytes (the contract the byte-fed stage kernel leans on for Phase A).
//  * ozfft_probe_crt:   the device reconstruction (Phase A MMA + deposits + lift + two-sided centring,
//    PAPER.md:370-373, Alg. 2 lines 9-13) on caller residues.
#pragma once
#include "arith.cuh"
#include "tc.cuh"
#include "ozfft.h"

namespace {

using namespace oz;

// A: [128][kb] bytes row-major (K-major), B: [n][kb] bytes row-major, D: [128][n] raw 32-bit accumulators.
// kind: 0 f8f6f4(E4M3,f32) 1 f16(f16,f32) 2 i8(s8,s32) 3 f16 with A staged through TMEM (tcgen05.st + .ts MMA)
//       4 i8(u8 x u8,s32)
__global__ void __launch_bounds__(128, 1) probe_kernel(int kind, int n, int kb, const uint8_t *A, const uint8_t *B, uint32_t *D) {
    extern __shared__ __align__(128) uint8_t smem[];
    __shared__ uint64_t bar;
    __shared__ uint32_t tmem_base_s;
    uint8_t *sA = smem;                  // [kb/16][128][16]
    uint8_t *sB = smem + 128 * kb;       // [kb/16][n][16]
    const int tid = threadIdx.x, warp = tid >> 5;
    for (int i = tid; i < 128 * (kb / 16); i += 128) {
        int r = i % 128, c = i / 128;
        *(uint4 *)(sA + (c * 128 + r) * 16) = *(const uint4 *)(A + (size_t)r * kb + c * 16);
    }
    for (int i = tid; i < n * (kb / 16); i += 128) {
        int r = i % n, c = i / n;
        *(uint4 *)(sB + (c * n + r) * 16) = *(const uint4 *)(B + (size_t)r * kb + c * 16);
    }
    if (warp == 0) tmem_alloc<512>(&tmem_base_s);
    if (tid == 0) { mbar_init(&bar, 1); mbar_fence_init(); }
    fence_async_smem();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = tmem_base_s;
    const uint32_t lane_addr = tmem + ((uint32_t)(warp * 32) << 16);
    if (kind == 3) {  // stage A (f16, kb bytes = kb/4 columns per lane) at TMEM column 256
        for (int c0 = 0; c0 < kb / 4; c0 += 8) {
            uint32_t v[8];
            for (int i = 0; i < 8; i++) v[i] = *(const uint32_t *)(A + (size_t)tid * kb + (c0 + i) * 4);
            tmem_st_x8(lane_addr + 256 + c0, v);
        }
        tmem_st_wait();
        tc_fence_before();
        __syncthreads();
        tc_fence_after();
    }
    if (tid == 0) {
        const uint32_t cf = (kind == 2 || kind == 4) ? CFMT_S32 : CFMT_F32;
        const uint32_t fmt = kind == 0 ? F8_E4M3 : (kind == 2 ? I8_S8 : (kind == 4 ? I8_U8 : F16_F16));
        const uint32_t idesc = make_idesc(cf, fmt, fmt, 128, n);
        for (int ks = 0; ks < kb / 32; ks++) {
            uint64_t ad = make_sdesc(smem_u32(sA) + ks * 2 * 128 * 16, 128 * 16, 128);
            uint64_t bd = make_sdesc(smem_u32(sB) + ks * 2 * n * 16, n * 16, 128);
            if (kind == 0) mma_f8f6f4_ss(tmem, ad, bd, idesc, ks > 0);
            else if (kind == 1) mma_f16_ss(tmem, ad, bd, idesc, ks > 0);
            else if (kind == 2 || kind == 4) mma_i8_ss(tmem, ad, bd, idesc, ks > 0);
            else mma_f16_ts(tmem, tmem + 256 + ks * 8, bd, idesc, ks > 0);
        }
        tc_commit(&bar);
    }
    mbar_wait(&bar, 0);
    tc_fence_after();
    for (int c = 0; c < n; c++) {
        uint32_t v;
        tmem_ld_x1(lane_addr + c, v);
        tmem_ld_wait();
        D[(size_t)tid * n + c] = v;
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc<512>(tmem);
}

}  // namespace

extern "C" int ozfft_probe_mma(int kind, int n, int kbytes, const void *dA, const void *dB, void *dD, void *stream) {
    if (kind < 0 || kind > 4 || n < 16 || n > 256 || (n % 16) || kbytes < 32 || (kbytes % 32)) return OZFFT_EINVAL;
    size_t sm = (size_t)(128 + n) * kbytes;
    if (sm > 200 * 1024) return OZFFT_EINVAL;
    cudaFuncSetAttribute(probe_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    probe_kernel<<<1, 128, sm, (cudaStream_t)stream>>>(kind, n, kbytes, (const uint8_t *)dA, (const uint8_t *)dB, (uint32_t *)dD);
    return cudaGetLastError() == cudaSuccess ? OZFFT_OK : OZFFT_ECUDA;
}

namespace {

using namespace oz;

// MMA1: D1[128][n1] = A[128][kb] * B1[n1][kb]^T (u8 x u8 -> s32) into TMEM columns [0, n1).
// MMA2: D2[128][n2] = bytes(D1)[128][4 n1] * B2[n2][4 n1]^T with the A operand read from TMEM columns [0, n1):
// K byte 4c + b of row r is byte b (little endian) of the s32 accumulator D1[r][c].  D2 lands at column 256.
__global__ void __launch_bounds__(128, 1) probe_chain_kernel(int n1, int kb, int n2, const uint8_t *A, const uint8_t *B1,
                                                              const uint8_t *B2, uint32_t *D1, uint32_t *D2) {
    extern __shared__ __align__(128) uint8_t smem[];
    __shared__ uint64_t bar;
    __shared__ uint32_t tmem_base_s;
    const int kb2 = 4 * n1;
    uint8_t *sA = smem, *sB1 = sA + 128 * kb, *sB2 = sB1 + n1 * kb;
    const int tid = threadIdx.x, warp = tid >> 5;
    for (int i = tid; i < 128 * (kb / 16); i += 128) {
        int r = i % 128, c = i / 128;
        *(uint4 *)(sA + (c * 128 + r) * 16) = *(const uint4 *)(A + (size_t)r * kb + c * 16);
    }
    for (int i = tid; i < n1 * (kb / 16); i += 128) {
        int r = i % n1, c = i / n1;
        *(uint4 *)(sB1 + (c * n1 + r) * 16) = *(const uint4 *)(B1 + (size_t)r * kb + c * 16);
    }
    for (int i = tid; i < n2 * (kb2 / 16); i += 128) {
        int r = i % n2, c = i / n2;
        *(uint4 *)(sB2 + (c * n2 + r) * 16) = *(const uint4 *)(B2 + (size_t)r * kb2 + c * 16);
    }
    if (warp == 0) tmem_alloc<512>(&tmem_base_s);
    if (tid == 0) { mbar_init(&bar, 1); mbar_fence_init(); }
    fence_async_smem();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = tmem_base_s;
    const uint32_t lane_addr = tmem + ((uint32_t)(warp * 32) << 16);
    if (tid == 0) {
        const uint32_t id1 = make_idesc(CFMT_S32, I8_U8, I8_U8, 128, n1), id2 = make_idesc(CFMT_S32, I8_U8, I8_U8, 128, n2);
        for (int ks = 0; ks < kb / 32; ks++)
            mma_i8_ss(tmem, make_sdesc(smem_u32(sA) + ks * 2 * 128 * 16, 128 * 16, 128),
                      make_sdesc(smem_u32(sB1) + ks * 2 * n1 * 16, n1 * 16, 128), id1, ks > 0);
        // no wait in between: MMAs issued by one thread execute in order, MMA2 reads what MMA1 wrote
        for (int ks = 0; ks < kb2 / 32; ks++)
            mma_i8_ts(tmem + 256, tmem + ks * 8, make_sdesc(smem_u32(sB2) + ks * 2 * n2 * 16, n2 * 16, 128), id2, ks > 0);
        tc_commit(&bar);
    }
    mbar_wait(&bar, 0);
    tc_fence_after();
    for (int c = 0; c < n1; c++) {
        uint32_t v;
        tmem_ld_x1(lane_addr + c, v);
        tmem_ld_wait();
        D1[(size_t)tid * n1 + c] = v;
    }
    for (int c = 0; c < n2; c++) {
        uint32_t v;
        tmem_ld_x1(lane_addr + 256 + c, v);
        tmem_ld_wait();
        D2[(size_t)tid * n2 + c] = v;
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc<512>(tmem);
}

// Device reconstruction on caller residues res[n][12] (u16, any representative below 2^13).
// variant 1: the tensor-core form -- residues as two-limb bytes -> Phase-A MMA against the slice matrix ->
// deposit_slices -> crt_from_E (lift from the top bits of E, two-sided centring); variant 0: crt_centre
// (plain 128-bit sums, fractional-column lift).  out[n][4] = two's-complement limbs of R in [-M/2, M/2).
__global__ void __launch_bounds__(128, 1) probe_crt_kernel(int variant, int n, const uint16_t *res, uint32_t *out,
                                                            const oz::DevConsts *cptr) {
    __shared__ __align__(128) uint8_t sR[4096];
    __shared__ __align__(128) uint8_t sPA[512];
    __shared__ uint64_t bar;
    __shared__ uint32_t tmem_base_s;
    const int tid = threadIdx.x, warp = tid >> 5;
    const long idx = (long)blockIdx.x * 128 + tid;
    uint32_t v[12];
    for (int k = 0; k < 12; k++) v[k] = idx < n ? res[idx * 12 + k] : 0;
    if (variant == 0) {
        const i128 R = crt_centre(v, *cptr);
        if (idx < n)
            for (int l = 0; l < 4; l++) out[idx * 4 + l] = (uint32_t)((u128)R >> (32 * l));
        return;
    }
    for (int i = tid; i < 1024; i += 128) ((uint32_t *)sR)[i] = 0;
    __syncthreads();
    for (int k = 0; k < 12; k++) *(uint16_t *)(sR + (k >> 3) * 2048 + tid * 16 + (k & 7) * 2) = (uint16_t)v[k];
    ((uint32_t *)sPA)[tid] = kc.phaseA[tid];
    if (warp == 0) tmem_alloc<32>(&tmem_base_s);
    if (tid == 0) { mbar_init(&bar, 1); mbar_fence_init(); }
    fence_async_smem();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = tmem_base_s;
    if (tid == 0) {
        mma_i8_ss(tmem, make_sdesc(smem_u32(sR), 128 * 16, 128), make_sdesc(smem_u32(sPA), 16 * 16, 128),
                  make_idesc(CFMT_S32, I8_U8, I8_U8, 128, 16), 0);
        tc_commit(&bar);
    }
    mbar_wait(&bar, 0);
    tc_fence_after();
    uint32_t P[16], R[4];
    tmem_ld_x16(tmem + ((uint32_t)(warp * 32) << 16), P);
    tmem_ld_wait();
    deposit_slices(P, R);
    if (idx < n)
        for (int l = 0; l < 4; l++) out[idx * 4 + l] = R[l];
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc<32>(tmem);
}

}  // namespace

namespace {
// A[128][kb] (row-major bytes) -> shared memory chunks [kb/16][128][16] -> tcgen05.cp into TMEM columns [0, kb/4)
// -> tcgen05.ld -> D[128][kb/4] words; must reproduce A's bytes (little endian) word for word.
__global__ void __launch_bounds__(128, 1) probe_cp_kernel(int kb, const uint8_t *A, uint32_t *D) {
    extern __shared__ __align__(128) uint8_t smem[];
    __shared__ uint64_t bar;
    __shared__ uint32_t tmem_base_s;
    const int tid = threadIdx.x, warp = tid >> 5;
    for (int i = tid; i < 128 * (kb / 16); i += 128) {
        int r = i % 128, c = i / 128;
        *(uint4 *)(smem + (c * 128 + r) * 16) = *(const uint4 *)(A + (size_t)r * kb + c * 16);
    }
    if (warp == 0) tmem_alloc<512>(&tmem_base_s);
    if (tid == 0) { mbar_init(&bar, 1); mbar_fence_init(); }
    fence_async_smem();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = tmem_base_s;
    if (warp == 0) {
        if (elect_one()) {
            for (int c = 0; c < kb / 16; c++) tmem_cp_128x128b(tmem + 4 * c, make_sdesc(smem_u32(smem) + c * 2048, 2048, 128));
            tc_commit(&bar);
        }
        __syncwarp();
    }
    mbar_wait(&bar, 0);
    tc_fence_after();
    for (int c = 0; c < kb / 4; c++) {
        uint32_t v;
        tmem_ld_x1(tmem + ((uint32_t)(warp * 32) << 16) + c, v);
        tmem_ld_wait();
        D[(size_t)tid * (kb / 4) + c] = v;
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc<512>(tmem);
}
}  // namespace

extern "C" int ozfft_probe_cp(int kbytes, const void *dA, void *dD, void *stream) {
    if (kbytes < 16 || kbytes > 1024 || (kbytes % 16)) return OZFFT_EINVAL;
    cudaFuncSetAttribute(probe_cp_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 128 * kbytes);
    probe_cp_kernel<<<1, 128, 128 * kbytes, (cudaStream_t)stream>>>(kbytes, (const uint8_t *)dA, (uint32_t *)dD);
    return cudaGetLastError() == cudaSuccess ? OZFFT_OK : OZFFT_ECUDA;
}

extern "C" int ozfft_probe_chain(int n1, int kbytes, int n2, const void *dA, const void *dB1, const void *dB2, void *dD1,
                                 void *dD2, void *stream) {
    if (n1 < 16 || n1 > 256 || (n1 % 16) || n2 < 16 || n2 > 256 || (n2 % 16) || kbytes < 32 || (kbytes % 32)) return OZFFT_EINVAL;
    const size_t sm = (size_t)(128 + n1) * kbytes + (size_t)n2 * 4 * n1;
    if (sm > 200 * 1024) return OZFFT_EINVAL;
    cudaFuncSetAttribute(probe_chain_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    probe_chain_kernel<<<1, 128, sm, (cudaStream_t)stream>>>(n1, kbytes, n2, (const uint8_t *)dA, (const uint8_t *)dB1,
                                                             (const uint8_t *)dB2, (uint32_t *)dD1, (uint32_t *)dD2);
    return cudaGetLastError() == cudaSuccess ? OZFFT_OK : OZFFT_ECUDA;
}
