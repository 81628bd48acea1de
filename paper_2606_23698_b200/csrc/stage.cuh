// stage.cuh -- launch geometry shared by every stage kernel.
//
// One "stage" is one residue DFT-by-matrix over columns of length K (PAPER.md:115-124 Bailey six-step; Alg. 1
// lines 1-7 for the first stage, 8-14 for the twiddle-fused second stage).  A tile is 32
// columns that share one matrix.  Tile t decomposes as t = (t2*n1 + t1)*n0 + t0; all offsets are in complex
// elements (16 bytes).
#pragma once
#include <cstdint>

namespace oz {

struct StageGeom {
    int K;               // contraction length = number of outputs per column (2..32)
    int n0, n1, n2;      // tile grid
    long long i0, i1, i2;  // input base strides per tile coordinate
    long long o0, o1, o2;  // output base strides
    long long lane;      // stride between the 32 columns of a tile (same for input and output)
    long long ji;        // input stride between contraction elements j
    long long ko;        // output stride between output rows k
    int matsel;          // matrix index of a tile: 0 -> 0, 1 -> t0, 2 -> t1
    int nmat;
};

__host__ __device__ inline long long tile_count(const StageGeom &g) { return (long long)g.n0 * g.n1 * g.n2; }

}  // namespace oz
