/* ozfft.h -- C ABI of the emulated-fp64 FFT (arxiv/paper_2606_23698, "FP8 is All You Need, Part 2").
 *
 * The library computes the unnormalised complex DFT  Y_k = sum_j X_j w_N^{jk}, per axis of a
 * 3-D array, as a Bailey six-step transform whose kernels contain no fp64
 * arithmetic: Ozaki-II residue GEMMs on tcgen05 tensor cores (Alg. 1 at 216-241), tc-CRT
 * reconstruction and Kulisch integer accumulation with a two-sided lift and one correctly
 * rounded pack per stage output (Alg. 2).
 *
 * Conventions (readings S1..S8): sign = -1 forward (w_N = exp(-2 pi i/N)), +1 inverse, never
 * normalised.  Sizes are powers of two, 2 <= n <= 1024 per axis (every such shape is accepted; a batched 1-D plan takes
 * any batch >= 1 with n * batch <= 2^30).  Arrays are row-major, z fastest:
 * element (x,y,z) at index (x*ny + y)*nz + z; one element = {re, im} as two IEEE-754 binary64 (16 bytes).
 * `in` and `out` are DEVICE pointers, 16-byte aligned, must not overlap; `in` is read only, `out` is fully
 * overwritten.  Inputs must be finite; a column holding a non-finite value produces NaN in the outputs of
 * that 1-D transform stage.  All plan memory (tables, workspace) is owned by the plan; the caller owns in/out.
 * ozfft_exec is asynchronous and ordered on `stream` (a cudaStream_t passed as void*); it never synchronises.
 * A plan must not execute concurrently on two streams (it owns workspace); different plans may be created and
 * executed from different host threads.  A destroyed or unknown handle is refused with OZFFT_EINVAL (the library
 * keeps a registry of live plans; it never dereferences a stale pointer).  Kernel selection: environment variable
 * OZFFT_VARIANT = bf (default: byte-fed tensor-core kernel), tc (residue-digit tensor-core kernel), simt, fp8 (kind::f8f6f4
 * rung), garner / fp64sum (ablations), read at plan creation.  OZFFT_SCHEDULE = unfused makes the byte-fed kernel run
 * every axis as two launches; by default an axis of length 1024 runs both stages in one launch with the intermediate
 * array in an L2-resident ring.  Results are bit-identical for every variant but fp64sum and for
 * both schedules.  No CPU fallback exists.
 */
#ifndef OZFFT_H
#define OZFFT_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

#define OZFFT_OK 0
#define OZFFT_EINVAL 1 /* null / misaligned pointer, bad size or sign, destroyed plan */
#define OZFFT_ECUDA 2  /* CUDA allocation or launch failure; text in ozfft_last_error() */

typedef struct ozfft_plan_s *ozfft_plan; /* opaque, library-owned */

/* 3-D plan (three axis passes z, y, x).  NULL on failure. */
ozfft_plan ozfft_plan_create(int nx, int ny, int nz, int sign);
/* batched contiguous 1-D plan: `batch` pencils of length n, pencil b at element offset b*n (BASELINE.json
 * config 3; one Bailey transform).  NULL on failure. */
ozfft_plan ozfft_plan_create_1d(int n, int batch, int sign);
/* out = DFT(in).  Device pointers to nx*ny*nz (or n*batch) complex128.  Returns OZFFT_*. */
int ozfft_exec(ozfft_plan plan, const void *in, void *out, void *stream);
/* Same through HOST buffers: copies in to the device, runs, copies back, synchronises `stream`. */
int ozfft_exec_host(ozfft_plan plan, const void *host_in, void *host_out, void *stream);
void ozfft_plan_destroy(ozfft_plan plan); /* NULL is a no-op */
const char *ozfft_last_error(void);       /* thread-local text of the last failure */

/* ---- entry point that allocates nothing ----
 * For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it) and so
 * cannot create a plan: out = DFT_1024 of each of `batch` contiguous pencils (pencil b at element offset 1024 b; the same
 * transform, bit for bit, as ozfft_plan_create_1d(1024, batch, sign) + ozfft_exec), computed by the fused-axis launch of the
 * byte-fed kernel with its scratch -- an 8-slot ring for the intermediate array and the
 * group counters -- in a file-scope `static __device__` array of OZFFT_STATIC_SCRATCH_BYTES (16 MiB + 4 KiB) and its constant
 * operand tables in a second one (11.4 MB): every GPU that loads the library holds both until the process exits.  `in` / `out`
 * as for ozfft_exec (device pointers, 16-byte aligned, distinct); asynchronous on `stream`.  Limits: batch a multiple of 128
 * with 128 <= batch <= OZFFT_STATIC_MAX_BATCH, anything else is refused with OZFFT_EINVAL and a message.  The call itself
 * issues two memsets of the counters and one kernel launch and never calls cudaMalloc / cudaFree or an allocating library
 * routine.  ozfft_static_setup() (once per device, with that device current; the first ozfft_fft1d_1024_static call on a device
 * does it implicitly) takes the arrays' addresses with cudaGetSymbolAddress and fills the tables with synchronous copies -- no
 * allocation either, but call it before starting a graph capture.  ALL calls on a device share the one scratch array, which
 * keeps the last call's contents: calls that overlap on the GPU (two streams, two host threads) race and give wrong results;
 * calls ordered on one stream are safe (the counters are re-zeroed on the stream, every ring slot is written before it is read). */
#define OZFFT_STATIC_MAX_BATCH 65536
#define OZFFT_STATIC_SCRATCH_BYTES (2 * 512 * 4 + 8 * 131072 * 16)
int ozfft_static_setup(void);
int ozfft_fft1d_1024_static(int batch, int sign, const void *in, void *out, void *stream);

/* ---- introspection / test hooks (not needed by users) ---- */
/* FNV-1a over the plan's 1024-entry table of (RN(2^53 cos), RN(2^53 sin)) of 2 pi t/1024 (reading S5);
 * must equal the oracle's independent generator. */
uint64_t ozfft_twiddle_checksum(void);
/* Kernel launches one ozfft_exec of this plan issues. */
int ozfft_plan_num_launches(ozfft_plan plan);
/* Device bytes the plan owns (tables + workspace). */
size_t ozfft_plan_device_bytes(ozfft_plan plan);
/* Run only axis pass `axis` (0 = z, 1 = y, 2 = x; a 1-D plan has axis 0 only) of a 3-D plan: out = pass(in).
 * Used by the sampled-pencil parity check at sizes the oracle cannot hold in full. */
int ozfft_exec_axis(ozfft_plan plan, int axis, const void *in, void *out, void *stream);
/* Silicon-contract probe: D[128][n] (raw 32-bit accumulators) = A[128][kbytes] * B[n][kbytes]^T as chained
 * M=128 tcgen05.mma of K = 32 bytes each.  kind 0: f8f6f4 E4M3 -> f32; 1: f16 -> f32; 2: i8 (s8) -> s32;
 * 3: f16 with A fed from TMEM; 4: i8 (u8 x u8) -> s32.  All pointers device.  n multiple of 16 in [16,256], kbytes multiple of 32. */
int ozfft_probe_mma(int kind, int n, int kbytes, const void *dA, const void *dB, void *dD, void *stream);
/* Host-only table export of the byte-fed stage kernel (no GPU needed; tests/test_bf_tables_cpu.py emulates the
 * kernel's integer dataflow on these tables and compares with the oracle's stage).  K = contraction length,
 * fusedN = 0 (plain DFT_K) or 32*K (twiddle-fused second stage, Eq. 6).  HOST pointers, any may be
 * NULL: h_B receives the matrix byte planes (return value = their size in bytes, 0 on a bad argument), h_C the
 * offset constants (nmat*K*16 bytes), h_PA the Phase-A constant matrix (6144 bytes).  Layouts: csrc/stage_bf.cuh. */
size_t ozfft_debug_bf_tables(int K, int fusedN, int sign, void *h_B, void *h_C, void *h_PA);
/* Chained probe: D1[128][n1] = A[128][kbytes] * B1[n1][kbytes]^T (u8 x u8 -> s32, kept in TMEM), then
 * D2[128][n2] = bytes(D1)[128][4 n1] * B2[n2][4 n1]^T with the second MMA reading its A operand straight from the
 * TMEM accumulator of the first (K byte 4c+b = little-endian byte b of D1[.][c]).  The byte-fed stage kernel uses
 * exactly this to run Phase A on the stage accumulators without a SIMT pass.  Device pointers. */
int ozfft_probe_chain(int n1, int kbytes, int n2, const void *dA, const void *dB1, const void *dB2, void *dD1, void *dD2,
                      void *stream);
/* tcgen05.cp probe: A[128][kbytes] -> shared-memory operand chunks -> TMEM -> D[128][kbytes/4] 32-bit words; D must
 * hold A's bytes unchanged (row r in lane r, 16 bytes = 4 columns).  The byte-fed kernel moves its data operand into
 * TMEM this way once per tile.  kbytes multiple of 16, <= 1024.  Device pointers. */
int ozfft_probe_cp(int kbytes, const void *dA, void *dD, void *stream);
/* Device CRT probe (PAPER.md:316-329 direct CRT, 370-373 two-sided lift, Alg. 2 lines 9-13 at 408-413):
 * d_residues = n x 12 uint16 (any representative of each residue below 2^13), d_out = n x 4 uint32 = two's-complement
 * limbs of the centred result in [-M/2, M/2).  variant 1: the tensor-core form the stage kernels use (Phase-A MMA,
 * deposits, quotient from the top of E, two-sided centring); variant 0: the SIMT kernel's 128-bit form.
 * Synchronises `stream`.  Device pointers. */
int ozfft_probe_crt(int n, const void *d_residues, void *d_out, int variant, void *stream);

/* Host-only: block `block` (32 tiles) of the fused-axis tile sequence for `groups` groups and lag `lag` (csrc/stage_bf.cuh
 * bf_sequence, the function the kernel uses) -> *stage (0 first, 1 second), *group.  The plan uses lag = min(8, groups) and a
 * ring of 16 slots.  Returns OZFFT_OK or OZFFT_EINVAL. */
int ozfft_debug_fuse_sequence(int block, int lag, int groups, int *stage, int *group);
/* Pipeline timers of the byte-fed stage kernel (measuring build only: paper_2606_23698_b200/build.py --timers compiles with
 * -DOZFFT_PIPE_TIMERS; the product build returns 0 and writes nothing).  h receives 160 x 12 uint64 (HOST pointer), one row per
 * CTA of the LAST launch, in SM clock cycles summed over the CTA's tiles: [0] issuer waiting for the data operand (a_full),
 * [1] for matrix planes (b_full), [2] for the Phase-A result slots (pa_empty), [3] issuer loop total, [4] tiles of the CTA,
 * [5] epilogue warp 12 waiting for Phase-A results, [6] for the column exponents, [7] its loop total, [8] deconstruction
 * warp 4 waiting on the fused-axis ring counters, [9] on a_empty / e_start, [10] its loop total.  Returns the row count. */
int ozfft_debug_timers(unsigned long long *h);

#ifdef __cplusplus
}
#endif
#endif
