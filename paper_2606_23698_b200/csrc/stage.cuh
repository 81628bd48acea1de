// stage.cuh -- launch geometry shared by every stage kernel.
//
// One "stage" is one residue DFT-by-matrix over columns of length K (PAPER.md:115-124 Bailey six-step; Alg. 1
// lines 1-7 for the first stage, 8-14 for the twiddle-fused second stage).  Columns come in
// blocks of 32 (adjacent in memory where the axis allows).  A block has coordinates (b, s, o): b enumerates
// blocks that share one matrix, s the matrix / sub-column index (j1 in stage 1, k2 in stage 2), o the outer
// index.  All offsets are in complex elements (16 bytes).
#pragma once
#include <cstdint>

namespace oz {

struct StageGeom {
    int K;               // contraction length = number of outputs per column (2..32)
    int nb, ns, no;      // block grid
    int ncols;           // columns along the b coordinate: column 32 b + lane exists iff it is < ncols (masked tail block)
    long long ib, is, io;  // input base strides per block coordinate
    long long ob, os, oo;  // output base strides
    long long lane;      // stride between the 32 columns of a block in the input
    long long olane;     // the same in the output
    long long ji;        // input stride between contraction elements j
    long long ko;        // output stride between output rows k
    int matsel;          // matrix index of a block: 0 -> 0, 1 -> s
    int order;           // enumeration order of a launch: 0 -> b fastest, 1 -> s fastest (then b), o slowest
    // Column addressing of the byte-fed kernel (stage_bf.cuh): column c (0..127) of tile tb along the b coordinate sits at
    //   (tb >> t_sh) * t_hi + (tb & t_mask) * t_lo + (c & c_mask) * c_lo + (c >> c_sh) * c_hi        (input: ci, output: co)
    // Natural order: four blocks of 32 lanes (t_sh 0, t_mask 0, t_hi 4 ib, c_mask 31, c_lo lane, c_sh 5, c_hi ib).
    // Patch order: the pass over the contiguous axis leaves its output with the inner index permuted, z' = k1 + p k2
    // instead of z = k2 + 32 k1 (each second-stage column then writes one contiguous run instead of 16-byte pieces 512
    // bytes apart, which reached DRAM as partial sectors); the first stage of the next axis, whose lanes run along z, takes
    // the permutation out: its 128 tile columns are an 8 (k1) x 16 (k2) patch read in 128-byte runs and written in
    // 256-byte runs (input: t_sh 1, t_mask 1, t_hi 8, t_lo 16 p, c_mask 7, c_lo 1, c_sh 3, c_hi p; output: t_hi 256,
    // t_lo 16, c_lo 32, c_hi 1).
    struct ColMap { int t_sh, t_mask, c_mask, c_sh; long long t_hi, t_lo, c_lo, c_hi; } ci, co;
};

// the column part does not change from tile to tile (a thread keeps it), the tile part is the same for a whole warp
__device__ __forceinline__ long long col_part(const StageGeom::ColMap &m, int c) {
    return (long long)(c & m.c_mask) * m.c_lo + (long long)(c >> m.c_sh) * m.c_hi;
}
__device__ __forceinline__ long long tile_part(const StageGeom::ColMap &m, int tb) {
    return (long long)(tb >> m.t_sh) * m.t_hi + (long long)(tb & m.t_mask) * m.t_lo;
}
__device__ __forceinline__ long long col_off(const StageGeom::ColMap &m, int tb, int c) { return tile_part(m, tb) + col_part(m, c); }

// the same with nbt = 2^lg_nbt and ns = 2^lg_ns (every supported size is a power of two): shifts, no division
__device__ __forceinline__ void tile_coords_pow2(const StageGeom &g, long long t, int lg_nbt, int lg_ns, int &b, int &s, int &o) {
    const uint32_t u = (uint32_t)t;
    if (g.order == 0) { b = u & ((1u << lg_nbt) - 1); s = (u >> lg_nbt) & ((1u << lg_ns) - 1); o = u >> (lg_nbt + lg_ns); }
    else { s = u & ((1u << lg_ns) - 1); b = (u >> lg_ns) & ((1u << lg_nbt) - 1); o = u >> (lg_nbt + lg_ns); }
}

// linear tile index -> (b, s, o) with nbt tiles along b
__host__ __device__ inline void tile_coords(const StageGeom &g, long long t, int nbt, int &b, int &s, int &o) {
    if (g.order == 0) { b = (int)(t % nbt); t /= nbt; s = (int)(t % g.ns); o = (int)(t / g.ns); }
    else { s = (int)(t % g.ns); t /= g.ns; b = (int)(t % nbt); o = (int)(t / nbt); }
}

}  // namespace oz
