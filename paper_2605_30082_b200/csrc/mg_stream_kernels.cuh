// mg_stream_kernels.cuh -- fused 2.5-D streaming kernels (placeholder until implemented)
#pragma once
#include "mg_common.cuh"
namespace mg {
inline bool stream_sweep_supported(int, int, int) { return false; }
inline int launch_stream_sweep(Lv, bool, const double *, double *, int, cudaStream_t) { return -1; }
inline int launch_stream_residual_norm2(Lv, bool, const double *, const double *, double *, int *, int, int, cudaStream_t) { return -1; }
} // namespace mg
