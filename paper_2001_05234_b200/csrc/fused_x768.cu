// fused_x768.cu -- fused pass-A / pass-C kernels (fused_pass.cuh) for nx = 768 and every fused ny.
#include "fused_kernels.cuh"

namespace cans {
CANS_FUSED_DEFINE(768)
}  // namespace cans
