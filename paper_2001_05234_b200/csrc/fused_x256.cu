// fused_x256.cu -- fused pass-A / pass-C kernels (fused_pass.cuh) for nx = 256 and every fused ny.
#include "fused_kernels.cuh"

namespace cans {
CANS_FUSED_DEFINE(256)
}  // namespace cans
