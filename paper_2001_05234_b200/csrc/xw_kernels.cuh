// xw_kernels.cuh -- host-callable launcher of the warp-per-line x transforms (defined in xw_kernels.cu).
#pragma once
#include <cuda_runtime.h>
#include "xw_pass.cuh"
#include "xy_kernels.cuh"

namespace cans {

// op: OP_X_FWD, OP_X_FWD_DIV, OP_X_INV, or OP_CONFIGURE at plan time (xy_kernels.cuh); tw = W_N^(p k1) table [R1][32] of the plan.
// Returns false if length n has no warp-per-line kernel.
bool xw_launch(int n, int op, const XYArgs& a, const cplx* tw, cudaStream_t st, cudaError_t* err);

}  // namespace cans
