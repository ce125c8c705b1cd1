// CTA output tile of the fused GEMM-pair kernel; shared by the planner (segmentation, executed
// flop count) and the kernels.
#pragma once
namespace su2 {
constexpr int TILE_M = 64;   // rows of F per CTA
constexpr int TILE_P = 64;   // columns of F per CTA
}  // namespace su2
