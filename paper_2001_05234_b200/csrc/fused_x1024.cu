// fused_x1024.cu -- fused pass-A / pass-C kernels (fused_pass.cuh) for nx = 1024 and every fused ny.
#include "fused_kernels.cuh"

namespace cans {
CANS_FUSED_DEFINE(1024)
}  // namespace cans
