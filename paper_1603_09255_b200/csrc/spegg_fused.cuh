// spegg_fused.cuh -- fused single-pass kernels of the hot configurations (sm_100a).
#pragma once
#include "spegg_internal.h"

namespace spegg {

__host__ inline bool fused_bit_supported(const SpK &) { return false; }
inline void launch_fused_bit(const SpK &, uint32_t, cudaStream_t) {}

}  // namespace spegg
