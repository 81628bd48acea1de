// stage_tc.cuh -- tensor-core stage kernel (placeholder until the tcgen05 path lands).
#pragma once
#include <vector>
#include "arith.cuh"
#include "stage.cuh"
#include "tables.cuh"
namespace oz {
inline void build_mat_tc(std::vector<uint8_t> &h, int, int, int, const Twiddles &) { h.assign(16, 0); }
inline bool stage_tc_prepare() { return false; }
inline bool stage_tc_launch(const StageGeom &, const void *, void *, const uint8_t *, const DevConsts *, cudaStream_t) { return false; }
}  // namespace oz
