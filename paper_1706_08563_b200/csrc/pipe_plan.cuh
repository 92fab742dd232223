// pipe_plan.cuh -- transform plans of the pipelined slice-step kernels (slice_pipe_row.cu, slice_pipe_col.cu):
// every thread holds E = 32 points, so lines up to 1024 points need one shared-memory exchange.
#pragma once
#include "fft_core.cuh"

namespace prism {

template <int N> struct PipePlan;
template <> struct PipePlan<256>  { using type = Plan<256, 32, 16, 16, 1>; };
template <> struct PipePlan<512>  { using type = Plan<512, 32, 32, 16, 1>; };
template <> struct PipePlan<1024> { using type = Plan<1024, 32, 32, 32, 1>; };
template <> struct PipePlan<2048> { using type = Plan<2048, 32, 32, 16, 4>; };

}  // namespace prism
