// ss_warp_kernel.cuh -- one warp per (object, frequency) eval for n <= SS_WARP_MAX_N.
// (placeholder until the register/shuffle kernel lands: objects of this class are served by the
// BLOCK path)
#pragma once
#include "ss_common.cuh"
#include "../../include/ss_periodogram.h"

namespace ss {
constexpr bool WARP_IMPLEMENTED = false;
constexpr int WARPS_PER_CTA = 8;
inline int warp_variant_for_n(int n) { return (n + 31) / 32; }
inline ss_status_t launch_warp_kernel(const EvalParams&, int, int64_t, cudaStream_t) { return SS_ERR_UNSUPPORTED; }
}  // namespace ss
