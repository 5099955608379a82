// yt_kernels.cuh -- host-callable launcher of the TMA-fed y transforms (defined in yt_kernels.cu).
#pragma once
#include <cuda_runtime.h>
#include "yt_pass.cuh"
#include "xy_kernels.cuh"

namespace cans {

// op: OP_Y_FWD or OP_Y_INV; tw = W_N^(p k1) table [R1][32] of the plan; a.p must be 16-byte aligned and
// a.nx / 2 a multiple of YT_COLS.  Returns false if length n has no TMA-fed kernel.
bool yt_launch(int n, int op, const XYArgs& a, const cplx* tw, int num_sms, cudaStream_t st, cudaError_t* err);

}  // namespace cans
