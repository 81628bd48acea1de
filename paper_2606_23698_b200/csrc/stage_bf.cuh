// stage_bf.cuh -- "byte-fed" stage kernel: one Bailey stage whose per-modulus work runs entirely on tcgen05.
//
// Idea (what differs from the paper's sketch, and from stage_tc.cuh): the DATA operand of the
// stage GEMM is not a residue plane but the raw bytes of the quantised 54-bit integers, w = x~ + 2^53 =
// sum_b w_b 256^b (7 unsigned bytes), so it is the SAME for all twelve moduli and is written once per tile.
// The modulus-dependent part moves into the MATRIX operand: for modulus m_i, entry (k, j, h, b) is the
// two-byte split (digit d = 0, 1) of  c_{kjh} 256^b mod m_i,  c = a_R (h = 0) or a_I (h = 1)
// ("sum_k b_k (2^{8k} mod m_i)" folded into the DFT matrix, Eq. 6 for the fused one).
// One u8 x u8 -> s32 MMA therefore yields, per (column, output, modulus), two accumulators lo, hi with
// lo + 256 hi == sum_j c_kj w_j (mod m_i): deconstruction (a3), the residue GEMM (a4) and the recombination (a5)
// are one tensor-core operation, and no per-modulus SIMT instruction exists.
//
// Rows: MMA row r = data column r.  The re part contracts [x_R ; -x_I] and the im part [x_I ; x_R] against the one
// matrix [a_R ; a_I] (direct 4-product complex form): three byte planes XI, XR, NXI (-x_I) per tile serve both.
// Radix-2 in the output index: with H = K/2, a~_{k+H,j} = (-1)^j a~_{k,j} holds EXACTLY in the quantised table
// (T[t+512] = -T[t], reading S5), so the even-j and odd-j partial sums S^E_k, S^O_k (k < H) are accumulated
// separately (half the matrix, half the MMA work) and out_k = S^E + S^O, out_{k+H} = S^E - S^O are formed inside
// Phase A, which is linear: its constant matrix carries u_i for the sum and M - u_i for the difference.
//
// Phase A (tc-CRT, two-limb form 759-764, here a byte-limb form): the s32 stage accumulators
// stay in TMEM and ARE the A operand of a second kind::i8 MMA (a 32-bit TMEM cell = four unsigned K bytes; contract
// measured by tests/test_gpu_silicon.py): P_s = sum_{i,d,b} byte_b(acc_{i,d}) * byte_s(256^{d+b} u_i mod M).
// Phase B (Alg. 2): deposits E = sum_s P_s 256^s, lift, two-sided centring (arith.cuh), minus the
// offset constant C_k = 2^53 sum_j (a_R + a_I)_kj, one RNE pack to fp64.
//
// Capacity: |R + C| <= 2^111.5 + 2^111.5 < M/2 = 2^116.9.  E < 30768 M < 2^134.
#pragma once
#include <utility>
#include <vector>

#include "arith.cuh"
#include "stage.cuh"
#include "tables.cuh"
#include "tc.cuh"

namespace oz {

// ---- geometry of the operands for contraction length K (2..32, power of two)
__host__ __device__ constexpr int bf_H(int K) { return K / 2; }                                 // output pairs (k, k + H)
__host__ __device__ constexpr int bf_PB(int K) { return ((7 * (K / 2) + 15) / 16) * 16; }       // bytes of one (plane, parity) block
__host__ __device__ constexpr int bf_NCK(int K) { return bf_PB(K) / 16; }                       // its 16-byte chunks = K steps of a chain
__host__ __device__ constexpr int bf_NCH(int K) { return (K / 2 + 1) / 2; }                     // matrix chunks (2 pairs each) per tile
constexpr int BF_N = 48;            // stage MMA N: 2 pairs x 12 moduli x 2 digits
constexpr int BF_COLS = 128;        // data columns per tile = MMA M
constexpr int BF_PA_BYTES = 32 * 192;  // Phase-A constant matrix: N = 2 outputs x 16 slices, K = (E|O) x 12 x 2 x 4 bytes
__host__ __device__ constexpr int bf_slot_bytes(int K) { return BF_N * 2 * bf_PB(K); }          // one parity of one chunk
__host__ __device__ constexpr int bf_plane_bytes(int K) { return 2 * bf_NCK(K) * BF_COLS * 16; }  // both parities
__host__ __device__ constexpr int bf_aset_bytes(int K) { return 3 * bf_plane_bytes(K); }        // XI, XR, NXI
__host__ __device__ constexpr size_t bf_mat_bytes(int K) { return (size_t)bf_NCH(K) * 2 * bf_slot_bytes(K); }  // per matrix id

inline int bf_tw_index(int K, int fusedN, int mid, int k, int j) {
    if (!fusedN) return (int)(((long)(TABLE_N / K) * j * k) % TABLE_N);
    return (int)(((long)(TABLE_N / fusedN) * j * (mid + 32L * k)) % TABLE_N);
}

// host: matrix byte planes for all matrix ids: [mid][chunk][parity][kappa/16][n = g*24 + i*2 + d][16 B], kappa =
// h*PB + jj*7 + b for element j = 2 jj + parity, half h, byte b; and the offset constants C[mid][k] (two's complement,
// four 32-bit limbs) = 2^53 * sum_j (a_R + a_I)_{kj}.
inline void build_mat_bf(std::vector<uint8_t> &B, std::vector<uint32_t> &Cc, int K, int fusedN, int sign, const Twiddles &T) {
    const int H = bf_H(K), PB = bf_PB(K), NCH = bf_NCH(K), nmat = fusedN ? 32 : 1, SB = bf_slot_bytes(K);
    B.assign((size_t)nmat * bf_mat_bytes(K), 0);
    Cc.assign((size_t)nmat * K * 4, 0);
    int p256[R_MOD][7];
    for (int i = 0; i < R_MOD; i++) {
        p256[i][0] = 1 % kModuli[i];
        for (int b = 1; b < 7; b++) p256[i][b] = (p256[i][b - 1] * 256) % kModuli[i];
    }
    for (int mid = 0; mid < nmat; mid++) {
        for (int k = 0; k < K; k++) {
            __int128 s = 0;
            for (int j = 0; j < K; j++) {
                const int t = bf_tw_index(K, fusedN, mid, k, j);
                s += (__int128)T.c[t] + (__int128)sign * T.s[t];
            }
            const unsigned __int128 c = (unsigned __int128)(s * ((__int128)1 << 53));
            for (int l = 0; l < 4; l++) Cc[((size_t)mid * K + k) * 4 + l] = (uint32_t)(c >> (32 * l));
        }
        for (int ch = 0; ch < NCH; ch++)
            for (int par = 0; par < 2; par++) {
                uint8_t *dst = B.data() + (size_t)mid * bf_mat_bytes(K) + ((size_t)ch * 2 + par) * SB;
                for (int g = 0; g < 2; g++) {
                    const int kp = 2 * ch + g;
                    if (kp >= H) continue;  // padding pair (K = 2): zero rows
                    for (int jj = 0; jj < H; jj++) {
                        const int j = 2 * jj + par, t = bf_tw_index(K, fusedN, mid, kp, j);
                        const int64_t cf[2] = {T.c[t], (int64_t)sign * T.s[t]};
                        for (int h = 0; h < 2; h++)
                            for (int i = 0; i < R_MOD; i++) {
                                const int a = residue_of(cf[h], kModuli[i]);
                                for (int b = 0; b < 7; b++) {
                                    const int v = (a * p256[i][b]) % kModuli[i], kap = h * PB + jj * 7 + b;
                                    for (int d = 0; d < 2; d++) {
                                        const int n = g * 24 + i * 2 + d;
                                        dst[(kap / 16) * (BF_N * 16) + n * 16 + kap % 16] = (uint8_t)(d ? v >> 8 : v & 255);
                                    }
                                }
                            }
                    }
                }
            }
    }
}

// host: Phase-A constant matrix [kappa/16][n = o*16 + s][16 B], kappa = part*96 + (i*2 + d)*4 + b (part 0 = even-j
// sum, 1 = odd-j sum): byte s of U = 256^(d+b) u_i mod M, or of M - U for (part 1, o = 1): out_{k+H} = S^E - S^O.
inline void build_pa_bf(uint8_t *pa, const CrtConsts &C) {
    for (int i = 0; i < BF_PA_BYTES; i++) pa[i] = 0;
    for (int i = 0; i < R_MOD; i++) {
        u128 U = C.u[i] % C.M;
        for (int e = 0; e < 5; e++) {  // e = d + b
            for (int d = 0; d < 2; d++) {
                const int b = e - d;
                if (b < 0 || b > 3) continue;
                for (int part = 0; part < 2; part++)
                    for (int o = 0; o < 2; o++) {
                        const u128 X = (part && o) ? (C.M - U) % C.M : U;
                        const int kap = part * 96 + (i * 2 + d) * 4 + b;
                        for (int s = 0; s < 16; s++)
                            pa[(kap / 16) * (32 * 16) + (o * 16 + s) * 16 + kap % 16] = (uint8_t)(X >> (8 * s));
                    }
            }
            U = (U << 8) % C.M;
        }
    }
}


// ---------------------------------------------------------------------------------------------------- kernel
// Warp roles (768 threads): warp 0 = matrix producer (TMA bulk copies into a ring), warp 1 = the one tensor-core issuer
// (tcgen05.cp, stage MMAs, Phase-A MMAs: program order is execution order), warps 2-3 idle, warps 4-11 = deconstruction
// (a1-a3: load, column exponent, quantise, byte planes), warps 12-23 = epilogue (a7-a9, a12: deposits, lift, pack, store;
// three groups of four warps, one TMEM lane quarter each).  All hand-offs are mbarriers; there is no block-wide barrier
// inside the tile loop.  One CTA per SM: 488 of the 512 TMEM columns, 178 KB of shared memory, 80 registers per thread.
constexpr int BF_NG = 3;            // epilogue groups of four warps (units go round-robin over them)
constexpr int BF_THREADS = 128 * (3 + BF_NG);
constexpr int BF_NSLOT = 8;         // matrix ring: half-slots of one parity of one chunk; a ring entry is one chunk (two of them)
constexpr int BF_NCS = BF_NSLOT / 2;
// TMEM columns: [0,168) data operand (per parity 84: XI | XR | NXI, 4 columns per 16-byte chunk), [168,360) stage
// accumulators of one chunk ([re rows: E 48 | O 48][im rows: E 48 | O 48]), [360,488) Phase-A results (2 slots x 64)
constexpr int BF_TA = 0, BF_TD = 168, BF_DPA = 360;
template <int K> __host__ __device__ constexpr size_t bf_smem_bytes() {
    return (size_t)bf_aset_bytes(K) + (size_t)BF_NSLOT * bf_slot_bytes(K) + BF_PA_BYTES;
}

#ifdef OZFFT_PIPE_TIMERS
__device__ unsigned long long g_bf_dbg[160][12];  // per CTA: see ozfft_debug_timers (include/ozfft.h)
#define OZ_T0() const long long t0_ = clock64()
#define OZ_T1(i) dbg_[i] += clock64() - t0_
#else
#define OZ_T0()
#define OZ_T1(i)
#endif
// [ledger: sync: mbarrier waits]
// bounded wait: a pipeline bug must not hang the GPU (traps after 2^26 failed polls).  Measured and left alone: dropping the
// poll counter (a tighter loop) costs 9 % at 1024^3, a nanosleep or a short arithmetic delay between polls 0.5-1.5 %, back-off
// only on the waits with slack nothing -- the loop below is the best of the forms tried.
template <int UNUSED> __device__ __forceinline__ void bf_wait_t(uint64_t *bar, uint32_t parity) {
    const uint32_t a = smem_u32(bar);
    uint32_t done, spins = 0;
    do {
        // the suspend-time hint lets the hardware park the warp instead of re-issuing the poll
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done) : "r"(a), "r"(parity), "r"(1000000u) : "memory");
        if (!done && ++spins > (1u << 26)) __trap();
    } while (!done);
}
__device__ __forceinline__ void bf_wait(uint64_t *bar, uint32_t parity) { bf_wait_t<0>(bar, parity); }
__device__ __forceinline__ void bf_wait_pa(uint64_t *bar, uint32_t parity) { bf_wait_t<0>(bar, parity); }
__device__ __forceinline__ void bf_wait_slack(uint64_t *bar, uint32_t parity) { bf_wait_t<0>(bar, parity); }

// [ledger: a3 deconstruction: quantise, offset, byte planes]
// tile of iteration `it` of this CTA: CTAs take PAIRS of consecutive tiles.  In the second stage of the contiguous axis
// consecutive tiles are k2, k2+1 over the same pencils, whose 16-byte outputs are the two halves of the same 32-byte
// sectors: written by one SM back to back they merge in L2 instead of reaching DRAM as partial (read-modify-write) sectors.
__device__ __forceinline__ long long bf_tile(long long it) { return ((it >> 1) * gridDim.x + blockIdx.x) * 2 + (it & 1); }

// append the 7 bytes of w = (hi:lo) (hi < 2^24) at byte position 7 e of a little-endian word array; e is a
// compile-time constant after unrolling, so every index and shift folds
__device__ __forceinline__ void bf_append7(uint32_t *wd, int e, uint32_t lo, uint32_t hi) {
    const int t = (7 * e) / 4, s = ((7 * e) % 4) * 8;
    if (s == 0) { wd[t] = lo; wd[t + 1] = hi; }
    else {
        wd[t] |= lo << s;
        wd[t + 1] = __funnelshift_l(lo, hi, s);
        if (s >= 16) wd[t + 2] = hi >> (32 - s);
    }
}

// ---------------------------------------------------------------------------------------------------- fused axis
// Both stages of one axis of length 1024 in ONE launch (beta -> 1; Alg. 1 lines 7-8).
// The paper keeps Y' of one transform on chip; a tcgen05 tile here is 128 columns that share one matrix, so the unit of
// fusion is a GROUP of 128 pencils: 32 first-stage tiles (4 pencils x 32 j1 each, or one j1 of 128 lanes) followed by 32
// second-stage tiles (one k2 each), with Y' of the group (2 MB) in a ring of R slots that stays in the 126 MB L2 -- it is
// written once, read once and overwritten before it is evicted, so it never reaches HBM.  The persistent CTAs walk one
// tile sequence in which a group's second stage comes `Lg` groups after its first stage; a second-stage tile waits (global
// counter, acquire) until all first-stage tiles of its group have stored, a first-stage tile until the ring slot it will
// overwrite has been read.  Every wait is on tiles earlier in the sequence, and all CTAs are resident: no deadlock.
struct BfFuse {
    StageGeom g2;                  // second stage: input side = ring (compact), output side = the axis output
    const uint8_t *mat2;           // its 32 twiddle-fused matrices (Eq. 6)
    const uint4 *ctab2;
    uint4 *ring;                   // R slots x 131072 elements
    unsigned int *wr_done, *rd_done;  // per group: first-stage (warp, unit) stores done; second-stage warps done reading
    int G, Lg, R;                  // groups, lag, ring slots (R > Lg, a power of two)
    int lg_nbt;                    // group = (go << lg_nbt) | gb
    int s1_mulb, s1_tlb, s1_tls;   // first-stage input tile: tb = gb * s1_mulb + tl * s1_tlb, ts = tl * s1_tls, to = go
    int r1_tlb, r1_tls;            // first-stage output (ring) tile: tb = tl * r1_tlb, ts = tl * r1_tls
};
constexpr int BF_GROUP_ELEMS = 32 * 4096;          // Y' of one group
constexpr unsigned BF_WR_TARGET = 32 * 16 * 4;     // first-stage tiles x units x warps per unit
constexpr unsigned BF_RD_TARGET = 32 * 8;          // second-stage tiles x deconstruction warps

struct BfLoc { int st, grp, tl, tbi, tsi, toi, tbo, tso, too; };

// block q (32 tiles) of the fused tile sequence -> (stage, group): the first-stage blocks of the first Lg groups, then
// alternately the first stage of group Lg + i and the second stage of group i, then the second-stage blocks of the last Lg
// groups.  tests/test_fuse_sequence_cpu.py checks on the host that this is a bijection and that every wait of the ring
// hand-shake points at earlier blocks.
__host__ __device__ inline void bf_sequence(int q, int Lg, int G, int &st, int &grp) {
    if (q < Lg) { st = 0; grp = q; return; }
    const int r = q - Lg;
    if (r < 2 * (G - Lg)) { st = r & 1; grp = st ? (r >> 1) : Lg + (r >> 1); }
    else { st = 1; grp = G - Lg + (r - 2 * (G - Lg)); }
}

template <bool FUSED>
__device__ __forceinline__ BfLoc bf_locate(const StageGeom &g, const BfFuse &f, long long tile, int lg_nbt, int lg_ns) {
    BfLoc L;
    if (!FUSED) {
        int tb, ts, to;
        tile_coords_pow2(g, tile, lg_nbt, lg_ns, tb, ts, to);
        L.st = 0; L.grp = 0; L.tl = 0;
        L.tbi = L.tbo = tb; L.tsi = L.tso = ts; L.toi = L.too = to;
        return L;
    }
    L.tl = (int)tile & 31;
    bf_sequence((int)(tile >> 5), f.Lg, f.G, L.st, L.grp);
    const int gb = L.grp & ((1 << f.lg_nbt) - 1), go = L.grp >> f.lg_nbt;
    if (L.st == 0) { L.tbi = gb * f.s1_mulb + L.tl * f.s1_tlb; L.tsi = L.tl * f.s1_tls; L.toi = go; L.tbo = L.tl * f.r1_tlb; L.tso = L.tl * f.r1_tls; L.too = 0; }
    else { L.tbi = 0; L.tsi = L.tl; L.toi = 0; L.tbo = gb; L.tso = L.tl; L.too = go; }
    return L;
}

// loads of the stage input: read-only path, or L2-coherent (the ring is written by other SMs during the launch)
template <bool FUSED> __device__ __forceinline__ uint4 bf_ld(const uint4 *p) {
    if (!FUSED) return __ldg(p);
    uint4 v;
    asm volatile("ld.global.cg.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
    return v;
}
// [ledger: sync: fused-axis ring counters (global acquire polls)]
// wait until a global counter reaches `target` (acquire; bounded: a protocol bug must trap, not hang)
__device__ __forceinline__ void bf_wait_global(const unsigned int *ctr, unsigned int target) {
    unsigned int v, spins = 0;
    for (;;) {
        asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(ctr) : "memory");
        if (v >= target) break;
        if (++spins > (1u << 24)) __trap();
        __nanosleep(200);
    }
}

// [ledger: setup, tile decode, loop control]
template <int K, bool FUSED>
__global__ void __launch_bounds__(BF_THREADS, 1) stage_bf_kernel(StageGeom g, const uint4 *__restrict__ in, uint4 *__restrict__ out,
                                                                 const uint8_t *__restrict__ mat, const uint4 *__restrict__ ctab,
                                                                 const uint4 *__restrict__ pa_g, long long ntiles, BfFuse f) {
    constexpr int H = bf_H(K), PB = bf_PB(K), NCK = bf_NCK(K), NCH = bf_NCH(K);
    constexpr int SB = bf_slot_bytes(K), PLANE = bf_plane_bytes(K), ASET = bf_aset_bytes(K), PARB = NCK * BF_COLS * 16;
    constexpr int NW = PB / 4;
    extern __shared__ __align__(128) uint8_t smem[];
    __shared__ __align__(8) uint64_t a_full[1], a_empty[1], e_start[1], b_full[BF_NCS], b_empty[BF_NCS], pa_full[BF_NG], pa_empty[1];
    __shared__ uint32_t s_tmem;
    __shared__ int s_T[2][BF_COLS], s_flag[2][BF_COLS];
    uint8_t *sA = smem, *sB = smem + ASET, *sPA = sB + BF_NSLOT * SB;

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int lg_nbt = 32 - __clz(((g.nb + 3) >> 2) - 1), lg_ns = 31 - __clz(g.ns);

    for (int i = tid; i < BF_PA_BYTES / 16; i += BF_THREADS) ((uint4 *)sPA)[i] = __ldg(pa_g + i);
    if (warp == 0) tmem_alloc<512>(&s_tmem);
    if (tid == 0) {
        // pa_full is per epilogue group; pa_empty counts the eight warps that drain the two units of one chunk (the two D_PA
        // slots hold exactly one chunk; a waiter must see every phase of its barrier in turn:
        // try_wait on parity p passes at once while the barrier is still in the phase before p)
        mbar_init(&a_full[0], 8); mbar_init(&a_empty[0], 1); mbar_init(&e_start[0], 4 * BF_NG);
        for (int i = 0; i < BF_NG; i++) mbar_init(&pa_full[i], 1);
        mbar_init(&pa_empty[0], 8);
        for (int i = 0; i < BF_NCS; i++) { mbar_init(&b_full[i], 1); mbar_init(&b_empty[i], 1); }
        mbar_fence_init();
    }
    fence_async_smem();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = s_tmem;
    if (tmem != 0) __trap();  // the CTA owns all 512 columns of its SM: the allocation starts at lane 0, column 0

    // uses of a matrix ring entry per tile: the chunk loops below are unrolled once around the ring, so every ring index is a
    // compile-time constant
    constexpr int UPT = (NCH + BF_NCS - 1) / BF_NCS;
    static_assert(NCH <= BF_NCS || NCH % BF_NCS == 0, "matrix ring: chunks per tile must tile the ring");
    if (warp == 0) {
        // [ledger: a11 matrix stream (TMA bulk copies)]
        // ------------------------------------------------ matrix producer (whole warp walks the loop, one lane issues)
        for (uint32_t pit = 0; bf_tile(pit) < ntiles; pit++) {
            const BfLoc L = bf_locate<FUSED>(g, f, bf_tile(pit), lg_nbt, lg_ns);
            const uint8_t *mb = (FUSED && L.st) ? f.mat2 + (size_t)L.tso * bf_mat_bytes(K) : mat + (size_t)((!FUSED && g.matsel) ? L.tso : 0) * bf_mat_bytes(K);
#pragma unroll
            for (int ch = 0; ch < NCH; ch++) {  // one copy per chunk: its two parity blocks are adjacent in the table
                const int cs = ch % BF_NCS;
                const uint32_t use = UPT * pit + ch / BF_NCS;  // how often this ring entry has been filled before
                if (use) bf_wait_slack(&b_empty[cs], (use - 1) & 1);
                if (elect_one()) {
                    mbar_expect_tx(&b_full[cs], 2 * SB);
                    bulk_g2s(sB + cs * 2 * SB, mb + (size_t)ch * 2 * SB, 2 * SB, &b_full[cs]);
                }
                __syncwarp();
            }
        }
    } else if (warp == 1) {
        // [ledger: a4 + a6 tensor-core issue (copies, stage MMAs, Phase-A MMAs)]
        // ------------------------------------------------ tensor-core issuer (one elected lane; program order = execution order)
        // per tile: tcgen05.cp of the data operand shared memory -> TMEM (then the shared copy is free for the next
        // tile); per chunk: a4 stage MMAs with A from TMEM (a3 and a5 folded into the operands), then a6 Phase A with
        // A = the stage accumulators.  This warp's instruction stream paces the tensor pipe (ncu: the pipe idles while the
        // issuer works through waits and address set-up), so the stream is kept short: the chunk loop is unrolled (ring
        // slots and barrier parities are constants), and one elected region per chunk issues Phase A of the PREVIOUS chunk
        // followed by the stage MMAs of this one -- the same program order as chunk-by-chunk issue, a quarter of the
        // wait / elect / reconverge sequences.
        const uint32_t idesc_st = make_idesc(CFMT_S32, I8_U8, I8_U8, 128, BF_N), idesc_pa = make_idesc(CFMT_S32, I8_U8, I8_U8, 128, 32);
        const uint64_t bdesc0 = make_sdesc(smem_u32(sB), BF_N * 16, 128), pdesc0 = make_sdesc(smem_u32(sPA), 32 * 16, 128);
        const uint64_t adesc0 = make_sdesc(smem_u32(sA), BF_COLS * 16, 128);
        constexpr int ACOLS = 3 * NCK * 4;  // TMEM columns of one parity of the data operand
        // the TMEM base (0) as a value of the uniform datapath that the compiler cannot fold or hoist: every TMEM address
        // below is then one uniform add next to its use, not a constant built in a vector register and moved across
        const uint32_t tz0 = (uint32_t)g.K >> 16;
        auto tzero = [&]() { uint32_t z; asm volatile("mov.u32 %0, %1;" : "=r"(z) : "r"(tz0)); return z; };
        auto opaque64 = [](uint64_t v) { uint64_t z; asm volatile("mov.b64 %0, %1;" : "=l"(z) : "l"(v)); return z; };  // same for descriptors
        uint32_t it = 0;
        uint32_t gc = 0;  // Phase-A unit -> epilogue group (round robin)
        bool pend = false;                           // Phase A of the last issued chunk is still to be issued
#ifdef OZFFT_PIPE_TIMERS
        long long dbg_[8] = {0, 0, 0, 0, 0, 0, 0, 0};
        const long long tstart_ = clock64();
#endif
        // Phase A of chunk number j (counted over the launch) needs the two D_PA slots back from chunk j - 1: one barrier,
        // eight arrivals (two units x four warps)
        uint32_t npa = 0;  // chunks whose Phase A has been issued
        auto wait_pa = [&]() {
            if (npa) { OZ_T0(); bf_wait(&pa_empty[0], (npa - 1) & 1); OZ_T1(2); }
            npa++;
        };
        auto issue_pa = [&](uint32_t g0, uint32_t g1) {  // elected lane only
            const uint32_t tz = tzero();
            const uint64_t pdz = opaque64(pdesc0);
#pragma unroll
            for (int gg = 0; gg < 2; gg++) {
#pragma unroll
                for (int P = 0; P < 2; P++)
#pragma unroll
                    for (int s = 0; s < 6; s++)
                        mma_i8_ts(tz + (BF_DPA + gg * 64 + P * 32), tz + (BF_TD + P * 96 + (s >= 3 ? 48 : 0) + gg * 24 + (s % 3) * 8),
                                  pdz + (uint64_t)((s * 2 * 32 * 16) >> 4), idesc_pa, s > 0);
                tc_commit(&pa_full[gg ? g1 : g0]);
            }
        };
        constexpr int UNR = NCH < BF_NCS ? NCH : BF_NCS;  // unrolled once around the matrix ring (code size: the instruction cache)
        for (; bf_tile(it) < ntiles; it++) {
#pragma unroll 1
            for (int c4 = 0; c4 < NCH; c4 += UNR)
#pragma unroll
            for (int u = 0; u < UNR; u++) {
                const int ch = c4 + u;
                const uint32_t g0 = gc, g1 = gc + 1 == BF_NG ? 0 : gc + 1;
                if (pend) wait_pa();
                if (ch == 0) {  // tile boundary: Phase A of the previous tile's last chunk goes out before the wait for the new operand
                    if (pend) {
                        tc_fence_after();
                        if (elect_one()) issue_pa(g0, g1);
                        __syncwarp();
                    }
                    { OZ_T0(); bf_wait(&a_full[0], it & 1); OZ_T1(0); }
                }
                { OZ_T0(); bf_wait(&b_full[u], (UPT * it + ch / BF_NCS) & 1); OZ_T1(1); }
                tc_fence_after();
                if (elect_one()) {
                    const uint32_t tz = tzero();
                    const uint64_t bdz = opaque64(bdesc0), adz = opaque64(adesc0);
                    if (ch == 0) {
#pragma unroll
                        for (int par = 0; par < 2; par++)
#pragma unroll
                            for (int pl = 0; pl < 3; pl++)
#pragma unroll
                                for (int t = 0; t < NCK; t++)
                                    tmem_cp_128x128b(tz + (BF_TA + par * ACOLS + (pl * NCK + t) * 4),
                                                     adz + (uint64_t)((pl * PLANE + par * PARB + t * (BF_COLS * 16)) >> 4));
                        tc_commit(&a_empty[0]);
                    } else if (pend) {
                        issue_pa(g0, g1);
                    }
#pragma unroll
                    for (int par = 0; par < 2; par++) {
                        const uint64_t bd = bdz + (uint64_t)(((u * 2 + par) * SB) >> 4);
#pragma unroll
                        for (int P = 0; P < 2; P++)  // P = 0: re rows [XR ; NXI] (planes 1, 2), P = 1: im rows [XI ; XR] (planes 0, 1)
#pragma unroll
                            for (int s = 0; s < NCK; s++)  // K step s = chunks 2s, 2s+1 of the two adjacent planes
                                mma_i8_ts(tz + (BF_TD + P * 96 + par * 48), tz + (BF_TA + par * ACOLS + ((1 - P) * NCK + 2 * s) * 4),
                                          bd + (uint64_t)((s * 2 * BF_N * 16) >> 4), idesc_st, s > 0);
                    }
                    tc_commit(&b_empty[u]);
                }
                __syncwarp();
                if (pend) gc = g1 + 1 == BF_NG ? 0 : g1 + 1;
                pend = true;
            }
        }
        if (pend) {  // Phase A of the very last chunk
            const uint32_t g0 = gc, g1 = gc + 1 == BF_NG ? 0 : gc + 1;
            wait_pa();
            tc_fence_after();
            if (elect_one()) issue_pa(g0, g1);
            __syncwarp();
        }
#ifdef OZFFT_PIPE_TIMERS
        if (lane == 0) { dbg_[3] = clock64() - tstart_; dbg_[4] = it; for (int i = 0; i < 5; i++) g_bf_dbg[blockIdx.x][i] = dbg_[i]; }
#endif
    } else if (warp >= 4 && warp < 12) {
        // [ledger: a1 load + addressing]
        // ------------------------------------------------ deconstruction: thread = (column, parity of j)
        const int dw = warp - 4, par = lane >> 4, c = dw * 16 + (lane & 15);
        constexpr int BS = H < 8 ? H : 8;  // elements loaded together (memory-level parallelism)
        // this thread's column offsets (either stage), kept across tiles as 32-bit values (they are below 2^22 for every plan):
        // every per-tile, per-thread instruction counts at this utilisation (-13 % at 512^3, -3 % at 1024^3 fused)
        const int cin1 = (int)col_part(g.ci, c), cin2 = FUSED ? (int)col_part(f.g2.ci, c) : 0;
        uint32_t it = 0;
#ifdef OZFFT_PIPE_TIMERS
        long long dbg_[12] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
        const long long tstart_ = clock64();
#endif
        for (long long tile; (tile = bf_tile(it)) < ntiles; it++) {
            const uint32_t buf = it & 1;
            const BfLoc L = bf_locate<FUSED>(g, f, tile, lg_nbt, lg_ns);
            const bool second = FUSED && L.st;  // second-stage tile of a fused axis: reads the ring
            const bool valid = FUSED || L.tbi * BF_COLS + c < g.ncols;
            const long long ji = second ? f.g2.ji : g.ji;
            const uint4 *src = second
                ? f.ring + ((long long)(L.grp & (f.R - 1)) * BF_GROUP_ELEMS + tile_part(f.g2.ci, L.tbi) + cin2 + (long long)L.tsi * f.g2.is + (long long)par * ji)
                : in + (tile_part(g.ci, L.tbi) + cin1 + (long long)L.tsi * g.is + (long long)L.toi * g.io + (long long)par * ji);
            const long long jstep = 2 * ji;
            if (FUSED) {  // the ring hand-shake (see BfFuse): data of this group written / the slot to be overwritten read
                OZ_T0();
                if (second) bf_wait_global(f.wr_done + L.grp, BF_WR_TARGET);
                else if (L.grp >= f.R) bf_wait_global(f.rd_done + (L.grp - f.R), BF_RD_TARGET);
                OZ_T1(8);
                __syncwarp();
            }
            // [ledger: a2 column exponent]
            // a2: column exponent = max of the 11-bit exponent fields (integer compare on the high words)
            uint32_t hmax = 0;
#pragma unroll
            for (int jj = 0; jj < H; jj++) {
                const uint4 v = valid ? bf_ld<FUSED>(src + jj * jstep) : make_uint4(0, 0, 0, 0);
                hmax = max(hmax, max(v.y & 0x7FFFFFFFu, v.w & 0x7FFFFFFFu));
            }
            hmax = max(hmax, __shfl_xor_sync(0xFFFFFFFFu, hmax, 16));
            int Tmax = 0, flag = 0;
            const uint32_t ef = hmax >> 20;
            if (ef == 0x7FF) flag = 2;
            else if (ef) { flag = 1; Tmax = (int)ef - 1023; }
            if (__any_sync(0xFFFFFFFFu, ef == 0)) {  // some column holds only zeros and subnormals: true leading bits
                int tm = -100000;                   // (warp-uniform branch: the exchange below needs every lane)
                for (int jj = 0; jj < H; jj++) {
                    const uint4 v = valid ? bf_ld<FUSED>(src + jj * jstep) : make_uint4(0, 0, 0, 0);
                    int T;
                    if (classify_top(((uint64_t)v.y << 32) | v.x, T) == CLS_FINITE) tm = max(tm, T);
                    if (classify_top(((uint64_t)v.w << 32) | v.z, T) == CLS_FINITE) tm = max(tm, T);
                }
                tm = max(tm, __shfl_xor_sync(0xFFFFFFFFu, tm, 16));
                if (ef == 0 && tm > -100000) { flag = 1; Tmax = tm; }
            }
            // [ledger: a3 deconstruction: quantise, offset, byte planes]
            // the previous tile's operand must have been copied to TMEM before the shared copy is overwritten
            if (it >= 1) { OZ_T0(); bf_wait_slack(&a_empty[0], (it - 1) & 1); OZ_T1(9); }
            if (par == 0) { s_T[buf][c] = Tmax; s_flag[buf][c] = flag; }
            // a3: quantise, offset by 2^53, split into bytes; planes XI (0), XR (1), NXI (2)
            uint32_t wr[NW + 2], wi[NW + 2], wn[NW + 2];
#pragma unroll
            for (int t = 0; t < NW + 2; t++) wr[t] = wi[t] = wn[t] = 0;
            uint8_t *dst = sA + par * PARB + c * 16;
#pragma unroll
            for (int e0 = 0; e0 < H; e0 += BS) {
                uint4 vv[BS];
#pragma unroll
                for (int x = 0; x < BS; x++) vv[x] = valid ? bf_ld<FUSED>(src + (e0 + x) * jstep) : make_uint4(0, 0, 0, 0);
#pragma unroll
                for (int x = 0; x < BS; x++) {
                    const int e = e0 + x;
                    const uint4 v = vv[x];
                    const uint64_t br = ((uint64_t)v.y << 32) | v.x, bi = ((uint64_t)v.w << 32) | v.z;
                    const uint64_t ar = flag == 1 ? quantise_mag_fast(br, Tmax) : 0ull, ai = flag == 1 ? quantise_mag_fast(bi, Tmax) : 0ull;
                    const uint64_t sr = (uint64_t)((int64_t)br >> 63), si = (uint64_t)((int64_t)bi >> 63);
                    const uint64_t off = 1ull << 53;
                    const uint64_t qr = ((ar ^ sr) - sr) + off, qi = ((ai ^ si) - si) + off, qn = 2 * off - qi;
                    bf_append7(wr, e, (uint32_t)qr, (uint32_t)(qr >> 32));
                    bf_append7(wi, e, (uint32_t)qi, (uint32_t)(qi >> 32));
                    bf_append7(wn, e, (uint32_t)qn, (uint32_t)(qn >> 32));
#pragma unroll
                    for (int t = 0; t < NCK; t++)
                        if (16 * (t + 1) <= 7 * (e + 1) && 16 * (t + 1) > 7 * e) {  // chunk t just completed
                            *(uint4 *)(dst + t * (BF_COLS * 16)) = make_uint4(wi[4 * t], wi[4 * t + 1], wi[4 * t + 2], wi[4 * t + 3]);
                            *(uint4 *)(dst + PLANE + t * (BF_COLS * 16)) = make_uint4(wr[4 * t], wr[4 * t + 1], wr[4 * t + 2], wr[4 * t + 3]);
                            *(uint4 *)(dst + 2 * PLANE + t * (BF_COLS * 16)) = make_uint4(wn[4 * t], wn[4 * t + 1], wn[4 * t + 2], wn[4 * t + 3]);
                        }
                }
            }
#pragma unroll
            for (int t = 0; t < NCK; t++)
                if (16 * (t + 1) > 7 * H) {  // trailing chunk(s) that the last element did not complete (zero padded)
                    *(uint4 *)(dst + t * (BF_COLS * 16)) = make_uint4(wi[4 * t], wi[4 * t + 1], wi[4 * t + 2], wi[4 * t + 3]);
                    *(uint4 *)(dst + PLANE + t * (BF_COLS * 16)) = make_uint4(wr[4 * t], wr[4 * t + 1], wr[4 * t + 2], wr[4 * t + 3]);
                    *(uint4 *)(dst + 2 * PLANE + t * (BF_COLS * 16)) = make_uint4(wn[4 * t], wn[4 * t + 1], wn[4 * t + 2], wn[4 * t + 3]);
                }
            // every epilogue warp must have observed the a_full phase of tile it-1 (and read its exponents) before
            // this tile's phase may complete: a waiter that falls two phases behind would wait forever
            if (it >= 1) { OZ_T0(); bf_wait_slack(&e_start[0], (it - 1) & 1); OZ_T1(9); }
            fence_async_smem();
            __syncwarp();
            if (second) {
                // this warp's share of the ring slot (16 columns x 32 elements = 8 KB) has been consumed: drop the lines from L2
                // without a write-back (Y' is dead until the slot is written again), 256 bytes per lane, then report the read
                const int col = dw * 16 + (ji == 1 ? (lane >> 1) : 0), j0 = ji == 1 ? (lane & 1) * 16 : lane;
                const uint4 *dl = f.ring + ((long long)(L.grp & (f.R - 1)) * BF_GROUP_ELEMS + col_off(f.g2.ci, L.tbi, col) + (long long)L.tsi * f.g2.is + (long long)j0 * ji);
                asm volatile("discard.global.L2 [%0], 128;" ::"l"(dl) : "memory");
                asm volatile("discard.global.L2 [%0], 128;" ::"l"(dl + 8) : "memory");
                __syncwarp();
            }
            if (lane == 0) {
                mbar_arrive(&a_full[0]);
                if (second) atomicAdd(f.rd_done + L.grp, 1u);
            }
        }
#ifdef OZFFT_PIPE_TIMERS
        if (warp == 4 && lane == 0) { g_bf_dbg[blockIdx.x][8] = dbg_[8]; g_bf_dbg[blockIdx.x][9] = dbg_[9]; g_bf_dbg[blockIdx.x][10] = clock64() - tstart_; }
#endif
    } else if (warp >= 12) {
        // [ledger: a12 store + addressing]
        // ------------------------------------------------ epilogue: thread = data column (TMEM lane), both parts
        const int qd = (warp - 12) >> 2, row = (warp & 3) * 32 + lane;
        const uint32_t lane_taddr = tmem + ((uint32_t)((warp & 3) * 32) << 16);
        uint32_t it = 0, nu = 0;  // tiles seen, units this group has consumed
#ifdef OZFFT_PIPE_TIMERS
        long long dbg_[8] = {0, 0, 0, 0, 0, 0, 0, 0};
        const long long tstart_ = clock64();
#endif
        int turn = qd;            // units to skip until the next one of this group (units go round-robin over the groups)
        const int cout1 = (int)col_part(g.co, row), cout2 = FUSED ? (int)col_part(f.g2.co, row) : 0;
        unsigned int wr_cnt = 0;  // fused axis: units of a first-stage tile this warp has stored and not yet counted
        int wr_grp = 0;
        for (long long tile; (tile = bf_tile(it)) < ntiles; it++) {
            const uint32_t buf = it & 1;
            if (FUSED && wr_cnt) {  // first-stage stores of the previous tile: visible, then counted (before any wait of this tile)
                __threadfence();
                __syncwarp();
                if (lane == 0) atomicAdd(f.wr_done + wr_grp, wr_cnt);
                wr_cnt = 0;
            }
            const BfLoc L = bf_locate<FUSED>(g, f, tile, lg_nbt, lg_ns);
            const bool second = FUSED && L.st;
            const bool valid = FUSED || L.tbo * BF_COLS + row < g.ncols;
            const long long ko = second ? f.g2.ko : g.ko;
            uint4 *dstp = second ? out + (tile_part(f.g2.co, L.tbo) + cout2 + (long long)L.tso * f.g2.os + (long long)L.too * f.g2.oo)
                          : (FUSED ? f.ring + (long long)(L.grp & (f.R - 1)) * BF_GROUP_ELEMS : out) + (tile_part(g.co, L.tbo) + cout1 + (long long)L.tso * g.os + (long long)L.too * g.oo);
            const uint4 *ct = second ? f.ctab2 + (size_t)L.tso * K : ctab + (size_t)((!FUSED && g.matsel) ? L.tso : 0) * K;
            { OZ_T0(); bf_wait_slack(&a_full[0], it & 1); OZ_T1(6); }  // the column exponents of this tile are published (s_T is double buffered: the
            const int Tmax = s_T[buf][row], flag = s_flag[buf][row];  // deconstruction runs at most one tile ahead)
            __syncwarp();
            if (lane == 0) mbar_arrive(&e_start[0]);
            const int gexp = 53 + 52 - Tmax;
            const long long hko = (long long)H * ko;  // output k + H sits this far from output k
#pragma unroll 1
            for (int ch = 0; ch < NCH; ch++)
#pragma unroll 1
                for (int gg = 0; gg < 2; gg++) {
                    if (turn) { turn--; continue; }
                    turn = BF_NG - 1;
                    const int kp = 2 * ch + gg;
                    uint4 cc[2];
                    cc[0] = __ldg(ct + (kp < H ? kp : 0));
                    cc[1] = __ldg(ct + (kp < H ? kp + H : 0));
                    // [ledger: a7 Phase B deposits (TMEM loads, slice sums -> E)]
                    { OZ_T0(); bf_wait_pa(&pa_full[qd], nu & 1); OZ_T1(5); }
                    tc_fence_after();
                    uint32_t E[4][5];  // [part*2 + o]
#pragma unroll
                    for (int x = 0; x < 4; x++) {
                        uint32_t P[16];
                        tmem_ld_x16(lane_taddr + BF_DPA + gg * 64 + x * 16, P);
                        tmem_ld_wait();
                        slices_to_E(P, E[x]);
                    }
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&pa_empty[0]);
                    nu++;
                    if (kp >= H || !valid) continue;
                    // [ledger: a12 store + addressing]
                    uint4 *dk = dstp + (long long)kp * ko;
                    if (flag == 1) {  // the usual column: finite, not all zero
                        // a8 lift + a9 pack of the four outputs as one straight-line block (finish_fast); the rare outputs that
                        // need the two-sided correction, are tiny against the column scale or leave the normal range are redone
                        uint64_t y[4];
#pragma unroll
                        for (int x = 0; x < 4; x++) {
                            uint32_t r[4], r2[4];
                            crt_from_E(E[x][0], E[x][1], E[x][2], E[x][3], E[x][4], r);
                            sub128(r2, r[0], r[1], r[2], r[3], cc[x & 1].x, cc[x & 1].y, cc[x & 1].z, cc[x & 1].w);
                            y[x] = pack_limbs(r2, gexp);
                        }
                        dk[0] = make_uint4((uint32_t)y[0], (uint32_t)(y[0] >> 32), (uint32_t)y[2], (uint32_t)(y[2] >> 32));    // a12: out k
                        dk[hko] = make_uint4((uint32_t)y[1], (uint32_t)(y[1] >> 32), (uint32_t)y[3], (uint32_t)(y[3] >> 32));  //      out k + H
                    } else {  // all-zero column -> +0, non-finite column -> NaN (reading S18)
                        const uint32_t hi = (flag & 2) ? 0x7FF80000u : 0u;
                        dk[0] = make_uint4(0, hi, 0, hi);
                        dk[hko] = make_uint4(0, hi, 0, hi);
                    }
                    if (FUSED && !second) { wr_cnt++; wr_grp = L.grp; }
                }
        }
        if (FUSED && wr_cnt) {
            __threadfence();
            __syncwarp();
            if (lane == 0) atomicAdd(f.wr_done + wr_grp, wr_cnt);
        }
#ifdef OZFFT_PIPE_TIMERS
        if (warp == 12 && lane == 0) { g_bf_dbg[blockIdx.x][5] = dbg_[5]; g_bf_dbg[blockIdx.x][6] = dbg_[6]; g_bf_dbg[blockIdx.x][7] = clock64() - tstart_; }
#endif
    }
    // [ledger: setup, tile decode, loop control]
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc<512>(tmem);
}

template <int K>
inline bool stage_bf_launch_k(const StageGeom &g, const void *in, void *out, const uint8_t *mat, const void *ctab, const void *pa,
                              long long nt, int sms, cudaStream_t st) {
    const long long pairs = (nt + 1) / 2;  // CTAs walk pairs of consecutive tiles (bf_tile)
    const unsigned grid = (unsigned)(pairs < sms ? pairs : sms);
    stage_bf_kernel<K, false><<<grid, BF_THREADS, bf_smem_bytes<K>(), st>>>(g, (const uint4 *)in, (uint4 *)out, mat, (const uint4 *)ctab, (const uint4 *)pa, nt, BfFuse{});
    return cudaGetLastError() == cudaSuccess;
}

inline bool stage_bf_prepare() {
    cudaError_t e = cudaFuncSetAttribute(stage_bf_kernel<32, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bf_smem_bytes<32>());
    if (e == cudaSuccess) e = cudaFuncSetAttribute(stage_bf_kernel<32, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bf_smem_bytes<32>());
    if (e == cudaSuccess) e = cudaFuncSetAttribute(stage_bf_kernel<16, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bf_smem_bytes<16>());
    if (e == cudaSuccess) e = cudaFuncSetAttribute(stage_bf_kernel<8, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bf_smem_bytes<8>());
    if (e == cudaSuccess) e = cudaFuncSetAttribute(stage_bf_kernel<4, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bf_smem_bytes<4>());
    if (e == cudaSuccess) e = cudaFuncSetAttribute(stage_bf_kernel<2, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bf_smem_bytes<2>());
    return e == cudaSuccess;
}

// tiles of 128 columns = 4 blocks of 32; the block grid along b is rounded up to a power of two (masked surplus)
inline bool stage_bf_launch(const StageGeom &g, const void *src, void *dst, const uint8_t *mat, const void *ctab, const void *pa, int sms,
                            cudaStream_t st) {
    int nbt = 1;
    while (nbt < (g.nb + 3) / 4) nbt <<= 1;
    if (g.ns & (g.ns - 1)) return false;
    const long long nt = (long long)nbt * g.ns * g.no;
    if (nt >= (1ll << 31)) return false;
    switch (g.K) {
        case 32: return stage_bf_launch_k<32>(g, src, dst, mat, ctab, pa, nt, sms, st);
        case 16: return stage_bf_launch_k<16>(g, src, dst, mat, ctab, pa, nt, sms, st);
        case 8: return stage_bf_launch_k<8>(g, src, dst, mat, ctab, pa, nt, sms, st);
        case 4: return stage_bf_launch_k<4>(g, src, dst, mat, ctab, pa, nt, sms, st);
        case 2: return stage_bf_launch_k<2>(g, src, dst, mat, ctab, pa, nt, sms, st);
    }
    return false;
}

// both stages of one axis of length 1024 in one launch (BfFuse): g1 = first stage (output side = ring), f.g2 = second stage
// (input side = ring).  The group counters are zeroed on the stream first.
inline bool stage_bf_launch_fused(const StageGeom &g1, const BfFuse &f, const void *src, void *dst, const uint8_t *mat1, const void *ctab1,
                                  const void *pa, int sms, cudaStream_t st) {
    if (g1.K != 32 || f.g2.K != 32 || f.R <= f.Lg || (f.R & (f.R - 1)) || f.Lg > f.G) return false;
    if (cudaMemsetAsync(f.wr_done, 0, (size_t)f.G * 4, st) != cudaSuccess || cudaMemsetAsync(f.rd_done, 0, (size_t)f.G * 4, st) != cudaSuccess) return false;
    const long long nt = 2LL * f.G * 32;
    const long long pairs = nt / 2;
    const unsigned grid = (unsigned)(pairs < sms ? pairs : sms);
    stage_bf_kernel<32, true><<<grid, BF_THREADS, bf_smem_bytes<32>(), st>>>(g1, (const uint4 *)src, (uint4 *)dst, mat1, (const uint4 *)ctab1, (const uint4 *)pa, nt, f);
    return cudaGetLastError() == cudaSuccess;
}

}  // namespace oz
