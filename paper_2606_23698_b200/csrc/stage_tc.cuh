// stage_tc.cuh -- tensor-core stage kernel: one Bailey stage with the residue DFT on tcgen05 kind::i8 MMAs.
//
// Tile: 64 columns.  MMA row r (= TMEM lane r) = (column r/2, part r&1): the re row holds the digits of
// [x_R ; -x_I], the im row those of [x_I ; x_R], so ONE matrix operand [a_R ; a_I] yields both parts
// (direct 4-product complex form).
// Digits (PAPER.md:113 leaves the layout to the builder): every residue is kept as a representative r in
// [0, 2m] (< 2^12) whose two bytes ARE the digits, x = x0 + 256 x1 (u8, u8 <= 15); -x is 2m - r, so all
// digits are unsigned.  Matrix entries a and a' = 256 a mod m split the same way, and
//   a x == (a0 x0 + a'0 x1) + 256 (a1 x0 + a'1 x1) (mod m):
// two s32 accumulators (u8 x u8 products) per output and modulus, contraction over (half, j, digit) = 4 K bytes,
// lo + 256 hi < 2^26.
// Per modulus pair: deconstruct digits -> SMEM operand -> tcgen05.mma kind::i8 into TMEM (double buffered)
// while the SIMT epilogue of the previous pair reduces its accumulators into the residue store; matrix planes
// arrive by TMA bulk copy one pair ahead.  The residue store is the data operand of Phase A (tc-CRT):
// a second kind::i8 MMA against the byte slices of the CRT idempotents; Phase B deposits the slice sums,
// lifts (mod M, two-sided) and packs once to fp64.  CTAs are persistent and prefetch the next tile's inputs.
#pragma once
#include <vector>

#include "arith.cuh"
#include "stage.cuh"
#include "tables.cuh"
#include "tc.cuh"

namespace oz {

// threads per CTA = 128 * Q: Q thread groups share each MMA row and split its contraction elements / outputs
__host__ __device__ constexpr int tc_q(int KP) { return 4; }
// TMEM columns: [0,256) stage accumulators (2 pairs x 2 x 64); the Phase-A sums of batch b reuse [128 b, 128 b + 128)
__host__ __device__ constexpr int tc_tmem_cols(int KP) { return KP >= 32 ? 512 : 256; }

// bytes of one modulus' matrix planes for padded length KP: rows n = 2k + d (d = digit 0/1), 4 KP bytes each,
// stored in the canonical K-major no-swizzle core-matrix order [chunk = byte/16][row n][16 B]
__host__ __device__ constexpr int tc_mat_bytes(int KP) { return 8 * KP * KP; }
__host__ __device__ constexpr int tc_pad(int K) { return K < 8 ? 8 : K; }
__host__ __device__ constexpr size_t tc_smem_bytes(int KP) {
    return 2 * (size_t)128 * 4 * KP + 4 * (size_t)tc_mat_bytes(KP) + (size_t)KP * 4096 + 512;
}

// host: digit planes of matrix set (K, fusedN) for all matrix ids and moduli: [mid][i][tc_mat_bytes]
inline void build_mat_tc(std::vector<uint8_t> &h, int K, int fusedN, int sign, const Twiddles &T) {
    const int KP = tc_pad(K), nmat = fusedN ? 32 : 1, MB = tc_mat_bytes(KP);
    h.assign((size_t)nmat * 12 * MB, 0);
    for (int mid = 0; mid < nmat; mid++)
        for (int i = 0; i < 12; i++) {
            uint8_t *dst = h.data() + ((size_t)mid * 12 + i) * MB;
            const int m = kModuli[i];
            for (int k = 0; k < K; k++)
                for (int j = 0; j < K; j++) {
                    const int t = fusedN ? (int)(((long)(TABLE_N / fusedN) * j * (mid + 32L * k)) % TABLE_N)
                                         : (int)(((long)(TABLE_N / K) * j * k) % TABLE_N);
                    const int a[2] = {residue_of(T.c[t], m), residue_of((int64_t)sign * T.s[t], m)};
                    for (int half = 0; half < 2; half++) {
                        const int av = a[half], ap = (av * 256) % m;  // a and a' = 256 a mod m
                        for (int d = 0; d < 2; d++) {                 // digit plane -> output row 2k + d
                            const int n = 2 * k + d;
                            const int e0 = d ? av >> 8 : av & 255, e1 = d ? ap >> 8 : ap & 255;
                            const int kap = half * 2 * KP + 2 * j;  // byte index in the contraction
                            dst[(kap / 16) * (2 * KP * 16) + n * 16 + kap % 16] = (uint8_t)e0;
                            dst[((kap + 1) / 16) * (2 * KP * 16) + n * 16 + (kap + 1) % 16] = (uint8_t)e1;
                        }
                    }
                }
        }
}

template <int KP>
__global__ void __launch_bounds__(128 * tc_q(KP), KP >= 32 ? 1 : 2) stage_tc_kernel(StageGeom g, const uint64_t *__restrict__ in,
                                                                 ulonglong2 *__restrict__ out,
                                                                 const uint8_t *__restrict__ mat, long long ntiles) {
    constexpr int Q = tc_q(KP);
    constexpr int JC = KP / Q;         // contraction elements (and outputs) per thread
    constexpr int ABYTES = 128 * 4 * KP;
    constexpr int MB = tc_mat_bytes(KP);
    constexpr int EPB = 8 / Q;         // outputs per thread per Phase-A batch: a batch is 8 MMAs of N = 16 (128 columns)
    constexpr int NB = JC / EPB;       // Phase-A batches
    constexpr int NCOL = 2 * KP;       // accumulator columns per modulus
    extern __shared__ __align__(128) uint8_t smem[];
    __shared__ __align__(8) uint64_t bar_full[2], bar_load[2], bar_pa[4];
    __shared__ uint32_t s_tmem;
    __shared__ int s_tmax[2][64], s_flag[2][64];
    uint8_t *sA = smem, *sB = smem + 2 * ABYTES, *sR = smem + 2 * ABYTES + 4 * MB;
    uint8_t *sPA = sR + KP * 4096;  // Phase-A constant matrix (operand order), 512 B
    // sR: residue store = Phase-A data operand: per output k a [2 chunks][128 rows][16 B] tile, residue i of row r at
    // k*4096 + (i/8)*2048 + r*16 + (i%8)*2 (u16 little endian = the two limbs v0, v1 of PAPER.md:759)

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int row = (warp & 3) * 32 + lane, q = warp >> 2;  // q < Q
    const int col = row >> 1, part = row & 1;
    const int K = g.K;
    // tile grid along b rounded up to a power of two (surplus tiles are fully masked); ns is a power of two
    const int lg_nbt = 32 - __clz(((g.nb + 1) >> 1) - 1), lg_ns = 31 - __clz(g.ns);

    if (tid < 64) { s_tmax[0][tid] = s_tmax[1][tid] = -100000; s_flag[0][tid] = s_flag[1][tid] = 0; }
    if (tid < 128) ((uint32_t *)sPA)[tid] = kc.phaseA[tid];
    if (warp == 0) tmem_alloc<tc_tmem_cols(KP)>(&s_tmem);
    if (tid == 0) {
        mbar_init(&bar_full[0], 1); mbar_init(&bar_full[1], 1);
        mbar_init(&bar_load[0], 1); mbar_init(&bar_load[1], 1);
        for (int i = 0; i < 4; i++) mbar_init(&bar_pa[i], 1);
        mbar_fence_init();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = s_tmem;
    const uint32_t idesc = make_idesc(CFMT_S32, I8_U8, I8_U8, 128, NCOL);
    const uint32_t lane_taddr = tmem + ((uint32_t)((warp & 3) * 32) << 16);
    const uint32_t full_addr = smem_u32(&bar_full[0]);

    // per-tile addressing: (valid, input base, output base, matrix base)
    // element offsets fit 32 bits (at most 2^30 elements per array); they widen only when the address is formed
    auto locate = [&](long long t, bool &valid, uint32_t &ib, uint32_t &ob, const uint8_t *&mb) {
        int tb, ts, to;
        tile_coords_pow2(g, t, lg_nbt, lg_ns, tb, ts, to);
        const int blk = 2 * tb + (col >> 5);
        valid = blk * 32 + (col & 31) < g.ncols;
        ib = (uint32_t)blk * (uint32_t)g.ib + (uint32_t)ts * (uint32_t)g.is + (uint32_t)to * (uint32_t)g.io + (uint32_t)(col & 31) * (uint32_t)g.lane;
        ob = (uint32_t)blk * (uint32_t)g.ob + (uint32_t)ts * (uint32_t)g.os + (uint32_t)to * (uint32_t)g.oo + (uint32_t)(col & 31) * (uint32_t)g.olane;
        mb = mat + (size_t)(g.matsel ? ts : 0) * 12 * MB;
    };
    const uint32_t ji32 = (uint32_t)g.ji, ko32 = (uint32_t)g.ko;
    auto load_inputs = [&](bool valid, uint32_t ib, uint64_t *bits) {  // a1: own part of own contraction elements
#pragma unroll
        for (int jj = 0; jj < JC; jj++) {
            const int j = q * JC + jj;
            bits[jj] = (valid && j < K) ? __ldg(in + 2 * (size_t)(ib + (uint32_t)j * ji32) + part) : 0ull;
        }
    };

    long long tile = blockIdx.x;
    if (tile >= ntiles) {  // (never with grid <= ntiles) still release TMEM
        if (warp == 0) tmem_dealloc<tc_tmem_cols(KP)>(tmem);
        return;
    }
    bool colvalid;
    uint32_t ibase, obase;
    const uint8_t *matbase;
    locate(tile, colvalid, ibase, obase, matbase);
    if (tid == 0) {  // matrix planes of modulus pairs 0 and 1 of the first tile
        mbar_expect_tx(&bar_load[0], 2 * MB);
        bulk_g2s(sB, matbase, 2 * MB, &bar_load[0]);
        mbar_expect_tx(&bar_load[1], 2 * MB);
        bulk_g2s(sB + 2 * MB, matbase + 2 * MB, 2 * MB, &bar_load[1]);
    }
    uint64_t bits[JC];
    load_inputs(colvalid, ibase, bits);
    int tpar = 0;
    // a2: column exponent = max of the 11-bit exponent fields (integer compare, no fp); subnormals can only matter
    // when the thread saw no normal number at all.  Scanned one tile ahead (the inputs are prefetched), so the
    // result is published by barriers the pipeline has anyway.
    auto exponent_scan = [&](int par) {
        int tm = -100000, fl = 0;
        uint32_t efmax = 0;
#pragma unroll
        for (int jj = 0; jj < JC; jj++) efmax = max(efmax, ((uint32_t)(bits[jj] >> 32) >> 20) & 0x7FFu);
        if (efmax == 0x7FF) fl = 2;
        else if (efmax) { fl = 1; tm = (int)efmax - 1023; }
        else {
#pragma unroll
            for (int jj = 0; jj < JC; jj++) {
                int T;
                if (classify_top(bits[jj], T) == CLS_FINITE) { fl = 1; tm = max(tm, T); }
            }
        }
        if (fl & 1) atomicMax(&s_tmax[par][col], tm);
        if (fl) atomicOr(&s_flag[par][col], fl);
    };
    exponent_scan(0);
    __syncthreads();
    uint32_t pa_phase = 0;  // parity of the next completion of the Phase-A barriers (one completion per tile each)
    uint32_t full_ph = 0, load_ph = 0;  // same for the MMA-done and matrix-landed barriers (bit = buffer)

#pragma unroll 1
    for (; tile < ntiles; tile += gridDim.x, tpar ^= 1) {
    const int Tmax = s_tmax[tpar][col], flag = s_flag[tpar][col];
    if (tid < 64) { s_tmax[tpar ^ 1][tid] = -100000; s_flag[tpar ^ 1][tid] = 0; }  // for the next tile
    // ---- a3 (first half): quantise to 53-bit magnitudes, keep as 18/18/17-bit limbs (PAPER.md:190 planes)
    uint32_t x0[JC], x1[JC], x2[JC];  // planes of the SIGNED x~ (two unsigned, the top one signed)
#pragma unroll
    for (int jj = 0; jj < JC; jj++) {
        const uint64_t a = (flag == 1) ? quantise_mag_fast(bits[jj], Tmax) : 0ull;
        const uint64_t sg = (uint64_t)((int64_t)bits[jj] >> 63);  // all ones for a negative element
        const uint64_t v = (a ^ sg) - sg;                          // x~ in two's complement
        x0[jj] = (uint32_t)v & 0x3FFFF;                            // unsigned 18 bits
        x1[jj] = (uint32_t)(v >> 18) & 0x3FFFF;                    // unsigned 18 bits
        x2[jj] = (uint32_t)((int32_t)(v >> 32) >> 4);              // signed top: x~ = x0 + 2^18 x1 + 2^36 x2
    }
    // ---- prefetch the next tile's inputs; they are consumed at the top of the next iteration
    const long long ntile = tile + gridDim.x;
    const bool more = ntile < ntiles;
    bool nvalid = false;
    uint32_t nib = 0, nob = 0;
    const uint8_t *nmat = matbase;
    if (more) locate(ntile, nvalid, nib, nob, nmat);
    load_inputs(more && nvalid, nib, bits);

    // Moduli go through the pipeline in pairs (one barrier, one fence and one commit per pair).  While the MMAs
    // of pair p run, the threads reduce the accumulators of pair p-1 AND compute the digits of pair p+1 in one
    // basic block, so two independent instruction streams fill the issue slots.
    uint32_t r0[2 * JC], r1[2 * JC];  // accumulators of a pair as read from TMEM
    uint32_t w[2][JC / 2], o[2][JC / 2];  // digit words of a pair: own row, partner row
    auto acc_load = [&](int p) {  // wait for the MMAs of pair p, start reading their accumulators
        const int buf = p & 1;
        mbar_wait_addr(full_addr + 8 * buf, (full_ph >> buf) & 1);
        full_ph ^= 1u << buf;
        tc_fence_after();
        if (tid == 0 && (p + 2 < 6 || more)) {  // their matrix buffer takes pair p+2 (or the next tile's pair p-4)
            const uint8_t *src = p + 2 < 6 ? matbase + (size_t)(p + 2) * 2 * MB : nmat + (size_t)(p - 4) * 2 * MB;
            mbar_expect_tx(&bar_load[buf], 2 * MB);
            bulk_g2s(sB + buf * 2 * MB, src, 2 * MB, &bar_load[buf]);
        }
        const uint32_t ta = lane_taddr + buf * 128 + 2 * q * JC;
        if constexpr (JC == 8) { tmem_ld_x16(ta, r0); tmem_ld_x16(ta + 64, r1); }
        else if constexpr (JC == 4) { tmem_ld_x8(ta, r0); tmem_ld_x8(ta + 64, r1); }
        else { tmem_ld_x4(ta, r0); tmem_ld_x4(ta + 64, r1); }
    };
    auto acc_reduce = [&](int p) {  // a5: recombine digits, reduce, park the residues of moduli 2p and 2p+1
        tmem_ld_wait();
        const int i0 = 2 * p;
        const uint32_t negm0 = 0u - kc.m[i0], mu0 = kc.mu[i0], negm1 = 0u - kc.m[i0 + 1], mu1 = kc.mu[i0 + 1];
        uint8_t *dst = sR + (q * JC) * 4096 + (i0 >> 3) * 2048 + row * 16 + (i0 & 7) * 2;
#pragma unroll
        for (int kk = 0; kk < JC; kk++) {  // residues left in [0, 2m): any representative serves the CRT
            const uint32_t v0 = add_alu(r0[2 * kk + 1] << 8, r0[2 * kk]), v1 = add_alu(r1[2 * kk + 1] << 8, r1[2 * kk]);  // < 2^26
            *(uint32_t *)(dst + kk * 4096) = pack16(barrett_lazy(v0, mu0, negm0), barrett_lazy(v1, mu1, negm1));
        }
        tc_fence_before();
    };
    auto digits = [&](int p) {  // a3 (second half): residues mod m_i of own elements; the u16 is the digit pair
#pragma unroll
        for (int h2 = 0; h2 < 2; h2++) {
            const int i = 2 * p + h2;
            const uint32_t mu = kc.mu[i], negm = 0u - kc.m[i], m2m2 = kc.m2m2[i], c18 = kc.c18[i], c36 = kc.c36[i], off = kc.off30[i];
#pragma unroll
            for (int jj = 0; jj < JC; jj++) {
                // signed plane sum made positive by a multiple of m: in (0, 2^31)
                const uint32_t rr = barrett_lazy(add_alu(x2[jj] * c36 + (x1[jj] * c18 + off), x0[jj]), mu, negm);  // in [0, 2m)
                if (jj & 1) w[h2][jj >> 1] = pack16(w[h2][jj >> 1], rr);
                else w[h2][jj >> 1] = rr;
            }
            // partner row (row^1) gets the same digits, negated (2m - r per half-word) when this is the im thread:
            // the re row holds [x_R ; -x_I], the im row [x_I ; x_R]
#pragma unroll
            for (int t = 0; t < JC / 2; t++) o[h2][t] = part ? m2m2 - w[h2][t] : w[h2][t];
        }
    };
    auto stage_issue = [&](int p) {  // digits -> data operand; a4: residue DFTs of moduli 2p, 2p+1 on the tensor core
#pragma unroll
        for (int h2 = 0; h2 < 2; h2++) {
            uint8_t *A = sA + h2 * ABYTES;
            const int kap = q * JC * 2;  // first contraction byte of this thread within a half
            uint8_t *d0 = A + (kap >> 4) * (128 * 16) + row * 16 + (kap & 15);
            uint8_t *d1 = A + ((2 * KP + kap) >> 4) * (128 * 16) + (row ^ 1) * 16 + (kap & 15);
            if constexpr (JC == 8) { *(uint4 *)d0 = make_uint4(w[h2][0], w[h2][1], w[h2][2], w[h2][3]); *(uint4 *)d1 = make_uint4(o[h2][0], o[h2][1], o[h2][2], o[h2][3]); }
            else if constexpr (JC == 4) { *(uint2 *)d0 = make_uint2(w[h2][0], w[h2][1]); *(uint2 *)d1 = make_uint2(o[h2][0], o[h2][1]); }
            else { *(uint32_t *)d0 = w[h2][0]; *(uint32_t *)d1 = o[h2][0]; }
        }
        fence_async_smem();
        tc_fence_before();
        __syncthreads();
        if (tid == 0) {
            tc_fence_after();
            mbar_wait(&bar_load[p & 1], (load_ph >> (p & 1)) & 1);
            load_ph ^= 1u << (p & 1);
#pragma unroll
            for (int h2 = 0; h2 < 2; h2++) {
                const uint32_t a0 = smem_u32(sA + h2 * ABYTES), b0 = smem_u32(sB + (p & 1) * 2 * MB + h2 * MB);
#pragma unroll
                for (int ks = 0; ks < KP / 8; ks++) {
                    const uint64_t ad = make_sdesc(a0 + ks * 2 * 128 * 16, 128 * 16, 128);
                    const uint64_t bd = make_sdesc(b0 + ks * 2 * NCOL * 16, NCOL * 16, 128);
                    mma_i8_ss(tmem + (p & 1) * 128 + h2 * 64, ad, bd, idesc, ks > 0);
                }
            }
            tc_commit(&bar_full[p & 1]);
        }
    };
    // the data operand is single-buffered: the MMAs of pair p must be done before pair p+1 overwrites it
    auto operand_free = [&](int p) { mbar_wait_addr(full_addr + 8 * (p & 1), (full_ph >> (p & 1)) & 1); };

    digits(0);
    stage_issue(0);
    digits(1);
    operand_free(0);
    stage_issue(1);
#pragma unroll
    for (int p = 1; p < 5; p++) {  // MMAs of pair p in flight (unrolled: the per-modulus constants become immediates)
        acc_load(p - 1);
        digits(p + 1);
        acc_reduce(p - 1);
        operand_free(p);
        stage_issue(p + 1);
    }
    acc_load(4);
    acc_reduce(4);
    acc_load(5);
    acc_reduce(5);


    exponent_scan(tpar ^ 1);  // the next tile's columns (its inputs arrived long ago); published by the barrier below
    // ---- a6: Phase A on the tensor core (Eq. 20, two-limb form 759-764): for each output k,
    // P[row][s] = sum over the 24 residue-limb bytes of the row x the slice matrix; u8 x u8 -> s32, N = 16.
    // Batch b covers outputs k = q'*JC + 2b + e (q' < 4, e < 2): thread group q' reads its 32 columns at q'*32.
    fence_async_smem();
    tc_fence_before();
    __syncthreads();
    auto issue_pa = [&](int b) {
        const uint32_t idesc_pa = make_idesc(CFMT_S32, I8_U8, I8_U8, 128, 16);
        const uint64_t bd = make_sdesc(smem_u32(sPA), 16 * 16, 128);
        const uint32_t dcol = tmem + b * 128;
#pragma unroll
        for (int qq = 0; qq < Q; qq++)
#pragma unroll
            for (int e = 0; e < EPB; e++) {
                const int k = qq * JC + EPB * b + e;
                mma_i8_ss(dcol + (qq * EPB + e) * 16, make_sdesc(smem_u32(sR) + k * 4096, 128 * 16, 128), bd, idesc_pa, 0);
            }
        tc_commit(&bar_pa[b]);
    };
    if (tid == 0) {
        tc_fence_after();
#pragma unroll
        for (int b = 0; b < NB; b++) issue_pa(b);  // every batch has its own TMEM columns: no barrier between batches
    }
    // ---- a7-a9: Phase B deposits, lift, pack; a12: store (the re thread stores even k, the im thread odd k)
    const int gexp = 53 + 52 - Tmax;
#pragma unroll 1
    for (int b = 0; b < NB; b++) {
        mbar_wait(&bar_pa[b], pa_phase);
        tc_fence_after();
        uint32_t P[16 * EPB];
        if constexpr (EPB == 2) tmem_ld_x32(lane_taddr + b * 128 + q * 32, P);
        else tmem_ld_x16(lane_taddr + b * 128 + q * 16, P);
        tmem_ld_wait();
#pragma unroll
        for (int e = 0; e < EPB; e++) {
            const int k = q * JC + EPB * b + e;
            uint64_t y;
            if (flag & 2) y = 0x7FF8000000000000ull;
            else if (flag == 0) y = 0;
            else {
                uint32_t R[4];
                deposit_slices(P + 16 * e, R);
                y = pack_limbs(R, gexp);
            }
            const uint32_t plo = __shfl_xor_sync(0xFFFFFFFFu, (uint32_t)y, 1), phi = __shfl_xor_sync(0xFFFFFFFFu, (uint32_t)(y >> 32), 1);
            const uint64_t yp = ((uint64_t)phi << 32) | plo;
            if (colvalid && k < K && (k & 1) == part) {
                ulonglong2 o;
                o.x = part ? yp : y;
                o.y = part ? y : yp;
                out[(size_t)(obase + (uint32_t)k * ko32)] = o;
            }
        }
    }
    pa_phase ^= 1;
    tc_fence_before();  // the next tile's MMAs overwrite the columns just read (after its barriers)
    colvalid = nvalid; ibase = nib; obase = nob; matbase = nmat;
    }  // tile loop
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc<tc_tmem_cols(KP)>(tmem);
}

inline bool stage_tc_prepare(const DevConsts &hc) {
    cudaError_t e = cudaMemcpyToSymbol(kc, &hc, sizeof(DevConsts));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(stage_tc_kernel<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tc_smem_bytes(32));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(stage_tc_kernel<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tc_smem_bytes(16));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(stage_tc_kernel<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tc_smem_bytes(8));
    return e == cudaSuccess;
}

// resident CTAs per SM of one instantiation on the current device (persistent grid = SMs x this)
template <int KP> inline int stage_tc_per_sm() {
    cudaFuncAttributes fa;
    int dev = 0, smem_sm = 0, regs_sm = 0, per_sm = 1;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&smem_sm, cudaDevAttrMaxSharedMemoryPerMultiprocessor, dev);
    cudaDeviceGetAttribute(&regs_sm, cudaDevAttrMaxRegistersPerMultiprocessor, dev);
    if (cudaFuncGetAttributes(&fa, stage_tc_kernel<KP>) == cudaSuccess) {
        const int by_smem = smem_sm / (int)(tc_smem_bytes(KP) + fa.sharedSizeBytes + 1024);
        const int by_regs = regs_sm / (((fa.numRegs + 7) & ~7) * 128 * tc_q(KP));
        per_sm = by_smem < by_regs ? by_smem : by_regs;
    }
    if (per_sm < 1) per_sm = 1;
    if (per_sm > 512 / tc_tmem_cols(KP)) per_sm = 512 / tc_tmem_cols(KP);  // TMEM columns
    return per_sm;
}
// per_sm[0..2]: KP = 8, 16, 32 (kept in the plan: per-device state)
inline void stage_tc_occupancy(int *per_sm) {
    per_sm[0] = stage_tc_per_sm<8>();
    per_sm[1] = stage_tc_per_sm<16>();
    per_sm[2] = stage_tc_per_sm<32>();
}

template <int KP>
inline bool stage_tc_launch_kp(const StageGeom &g, const uint64_t *in, ulonglong2 *out, const uint8_t *mat, long long nt, int sms, int per_sm, cudaStream_t st) {
    const long long cap = (long long)sms * per_sm;
    const unsigned grid = (unsigned)(nt < cap ? nt : cap);
    stage_tc_kernel<KP><<<grid, 128 * tc_q(KP), tc_smem_bytes(KP), st>>>(g, in, out, mat, nt);
    return cudaGetLastError() == cudaSuccess;
}

inline bool stage_tc_launch(const StageGeom &g, const void *src, void *dst, const uint8_t *mat, int sms, const int *per_sm, cudaStream_t st) {
    const int KP = tc_pad(g.K);
    int nbt = 1;
    while (nbt < (g.nb + 1) / 2) nbt <<= 1;  // rounded up to a power of two: shifts instead of divisions on the device
    if (g.ns & (g.ns - 1)) return false;
    const long long nt = (long long)nbt * g.ns * g.no;
    if (nt >= (1ll << 31)) return false;
    const uint64_t *in = (const uint64_t *)src;
    ulonglong2 *out = (ulonglong2 *)dst;
    if (KP == 32) return stage_tc_launch_kp<32>(g, in, out, mat, nt, sms, per_sm[2], st);
    if (KP == 16) return stage_tc_launch_kp<16>(g, in, out, mat, nt, sms, per_sm[1], st);
    return stage_tc_launch_kp<8>(g, in, out, mat, nt, sms, per_sm[0], st);
}

}  // namespace oz
