// fused_x384.cu -- fused pass-A / pass-C kernels (fused_pass.cuh) for nx = 384 and every fused ny.
#include "fused_kernels.cuh"

namespace cans {
CANS_FUSED_DEFINE(384)
}  // namespace cans
