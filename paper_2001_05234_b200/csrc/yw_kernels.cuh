// yw_kernels.cuh -- host-callable launcher of the warp-per-column y transforms (defined in yw_kernels.cu).
#pragma once
#include <cuda_runtime.h>
#include "yw_pass.cuh"
#include "xy_kernels.cuh"

namespace cans {

// op: OP_Y_FWD, OP_Y_INV, or OP_CONFIGURE at plan time (xy_kernels.cuh); tw = W_N^(p k1) table [R1][32] of the plan.
// Returns false if length n has no warp-per-column kernel.
bool yw_launch(int n, int op, const XYArgs& a, const cplx* tw, cudaStream_t st, cudaError_t* err);

}  // namespace cans
