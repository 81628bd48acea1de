// probe.cu -- silicon-contract probe: one chained tcgen05.mma (M=128) on caller-supplied operand bytes.
// Used by tests/test_gpu_silicon.py to check that integer-valued E4M3 / F16 / S8 operands accumulate
// exactly (PAPER.md:338, 890 flags this contract as unmeasured).
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
