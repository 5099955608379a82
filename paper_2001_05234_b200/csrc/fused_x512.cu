// fused_x512.cu -- fused pass-A / pass-C kernels (fused_pass.cuh) for nx = 512 and every fused ny.
#include "fused_kernels.cuh"

namespace cans {
CANS_FUSED_DEFINE(512)
}  // namespace cans
